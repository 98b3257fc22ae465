// render.cuh -- launchers of the volume renderer (render.cu).
#pragma once
#include <cuda_runtime.h>

namespace hlb {

struct RenderSetup {
  int nx = 0, ny = 0, nz = 0, width = 0, height = 0;
  float rot[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
  float zoom = 1, step = 1, tf_scale = 1, tf_offset = 0, opacity = 1;
};

// image [height][width][4] floats (device), vol [nz][ny][nx] floats (device); the viewing
// parameters and the 256 x RGBA look-up table (host) travel as a by-value kernel argument (the
// launch's own constant bank). tex: 0, or a point-sampled texture object over a 3-D array
// holding the same values as vol (then the samples are fetched through it). occ: macro-cell
// emptiness bytes from launch_occupancy, or NULL (no empty-space skipping; same image)
void launch_raymarch(const RenderSetup& r, const float* lut_host, const float* vol, cudaTextureObject_t tex,
                     const unsigned char* occ, float* image, cudaStream_t s);
// occ [occupancy_cells()] bytes: != 0 where every voxel a sample of the 8^3 macro-cell can touch
// is +0 (2: all macro-cells of the enclosing 64^3 super-cell are)
long long occupancy_cells(int nx, int ny, int nz);
void launch_occupancy(const float* vol, int nx, int ny, int nz, unsigned char* occ, cudaStream_t s);
// vol[voxel[c]] = |u| (field 0) or rho - 1 (field 1) of canonical site c
// surf: 0, or a surface object over the 3-D array of the texture path, written as well
void launch_scatter_field(const double* rho, const double* u, const long long* voxel, long long N,
                          int field, float* vol, cudaSurfaceObject_t surf, int nx, int ny, cudaStream_t s);

}  // namespace hlb
