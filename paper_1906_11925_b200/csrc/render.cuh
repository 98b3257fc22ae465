// render.cuh -- launchers of the volume renderer (render.cu).
#pragma once
#include <cuda_runtime.h>

namespace hlb {

struct RenderSetup {
  int nx = 0, ny = 0, nz = 0, width = 0, height = 0;
  float rot[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
  float zoom = 1, step = 1, tf_scale = 1, tf_offset = 0, opacity = 1;
};

// Copies the viewing parameters and the 256 x RGBA look-up table (host) into constant memory.
cudaError_t render_upload(const RenderSetup& r, const float* lut_host, cudaStream_t s);
// image [height][width][4] floats (device), vol [nz][ny][nx] floats (device); occ: macro-cell
// emptiness bytes from launch_occupancy, or NULL (no empty-space skipping; same image)
void launch_raymarch(const RenderSetup& r, const float* vol, const unsigned char* occ, float* image,
                     cudaStream_t s);
// occ [occupancy_cells()] bytes: != 0 where every voxel a sample of the 8^3 macro-cell can touch
// is +0 (2: all macro-cells of the enclosing 64^3 super-cell are)
long long occupancy_cells(int nx, int ny, int nz);
void launch_occupancy(const float* vol, int nx, int ny, int nz, unsigned char* occ, cudaStream_t s);
// vol[voxel[c]] = |u| (field 0) or rho - 1 (field 1) of canonical site c
void launch_scatter_field(const double* rho, const double* u, const long long* voxel, long long N,
                          int field, float* vol, cudaStream_t s);

}  // namespace hlb
