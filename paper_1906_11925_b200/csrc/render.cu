// render.cu -- direct volume rendering by ray marching to a headless device buffer
// (SURVEY.md §8(f) NEXT-4). This is the one GPU kernel the paper itself describes: "The CUDA
// cores in the rendering layer perform the volume rendering kernel based on the ray marching
// algorithm", with "the viewing parameters and the look-up table" in "GPU
// constant memory buffers" and steering by "zooming, model rotation and adjustment of scaling
// and offset of the transfer functions" (lines 97-99). The OpenGL / Qt display tiers are
// unavailable on this box; the image stays in a device buffer (or is copied to the host).
//
// Definition of the image: DESIGN.md reading R-render (orthographic camera, trilinear
// sampling, 256-entry RGBA look-up table, front-to-back compositing, early ray termination at
// A >= 0.995). Arithmetic: binary32, one explicit round-to-nearest intrinsic per operation,
// in the order the definition states, so that the result does not depend on compiler
// contraction. The paper keeps the volume in a 3-D texture; here it is a plain float array
// read through the read-only cache with the interpolation done in the kernel: the texture
// unit filters with 8-bit weights, which would make the image a property of the hardware
// filter rather than of the definition (and break exact comparison with the oracle).
#include <cuda_runtime.h>

#include <cstdint>

#include "render.cuh"

namespace hlb {
namespace {

struct ViewParams {
  int nx, ny, nz, width, height;
  float rot[9];
  float zoom, step, tf_scale, tf_offset, opacity;
};

// "GPU constant memory buffers" for the look-up table and the viewing parameters: both
// travel as ONE by-value kernel argument, which the hardware serves from the constant bank of
// that launch -- not from module-global __constant__ arrays, which two geometries (or two host
// threads) rendering on different streams would overwrite under each other's running kernels.
struct RenderParams {
  ViewParams v;
  float lut[256 * 4];
};

__device__ __forceinline__ float clamp01(float x) { return x < 0.0f ? 0.0f : (x > 1.0f ? 1.0f : x); }

__device__ __forceinline__ float lerp_rn(float f, float a, float b) {  // a + f (b - a)
  return __fmaf_rn(f, __fsub_rn(b, a), a);
}

// The volume: a plain float array read through the read-only cache (TEX = false), or a 3-D
// CUDA array behind a POINT-sampled texture object (TEX = true; the paper keeps its volume "in
// a 3D texture unit"). Either way the eight corner values are fetched exactly and the
// interpolation below is the same arithmetic, so the two give bit-identical images; the
// texture's own (8-bit-weight) filtering is not used.
template <bool TEX>
__device__ __forceinline__ float voxel_at(const float* __restrict__ vol, cudaTextureObject_t tex,
                                          int nx, int ny, int x, int y, int z) {
  if (TEX) return tex3D<float>(tex, (float)x + 0.5f, (float)y + 0.5f, (float)z + 0.5f);
  return __ldg(vol + ((long long)z * ny + y) * nx + x);
}
template <bool TEX>
__device__ __forceinline__ float trilinear(const float* __restrict__ vol, cudaTextureObject_t tex,
                                           int nx, int ny, int nz, float px, float py, float pz) {
  int ix = (int)floorf(px), iy = (int)floorf(py), iz = (int)floorf(pz);
  ix = min(ix, nx - 2); iy = min(iy, ny - 2); iz = min(iz, nz - 2);
  ix = max(ix, 0); iy = max(iy, 0); iz = max(iz, 0);
  const float fx = __fsub_rn(px, (float)ix), fy = __fsub_rn(py, (float)iy), fz = __fsub_rn(pz, (float)iz);
  const int x1 = ix + 1 < nx ? ix + 1 : ix, y1 = iy + 1 < ny ? iy + 1 : iy, z1 = iz + 1 < nz ? iz + 1 : iz;
  const float c00 = lerp_rn(fx, voxel_at<TEX>(vol, tex, nx, ny, ix, iy, iz), voxel_at<TEX>(vol, tex, nx, ny, x1, iy, iz));
  const float c10 = lerp_rn(fx, voxel_at<TEX>(vol, tex, nx, ny, ix, y1, iz), voxel_at<TEX>(vol, tex, nx, ny, x1, y1, iz));
  const float c01 = lerp_rn(fx, voxel_at<TEX>(vol, tex, nx, ny, ix, iy, z1), voxel_at<TEX>(vol, tex, nx, ny, x1, iy, z1));
  const float c11 = lerp_rn(fx, voxel_at<TEX>(vol, tex, nx, ny, ix, y1, z1), voxel_at<TEX>(vol, tex, nx, ny, x1, y1, z1));
  return lerp_rn(fz, lerp_rn(fy, c00, c10), lerp_rn(fy, c01, c11));
}

constexpr int TILE = 16;

// occ (may be NULL): one byte per 8 x 8 x 8 macro-cell, != 0 = every voxel a sample of the cell
// can touch ([8c, 8c + 8] per axis) is exactly +0 (2 = the same holds for all macro-cells of
// the 64^3 super-cell around it, so the jump may span the super-cell). Such a sample has the value +0 exactly; if
// the transfer function gives value 0 no opacity, it contributes exactly nothing and may be
// skipped, together with the following samples that provably stay in the same cell. The
// image is therefore bit-identical with and without occ.
template <bool TEX>
__global__ void __launch_bounds__(TILE * TILE)
k_raymarch(const __grid_constant__ RenderParams par, const float* __restrict__ vol, cudaTextureObject_t tex,
           const unsigned char* __restrict__ occ, float* __restrict__ image) {
  const int px = blockIdx.x * TILE + threadIdx.x, py = blockIdx.y * TILE + threadIdx.y;
  const ViewParams& v = par.v;
  const float* c_lut = par.lut;
  if (px >= v.width || py >= v.height) return;
  const float fnx = (float)v.nx, fny = (float)v.ny, fnz = (float)v.nz;
  const float cx = __fmul_rn(0.5f, (float)(v.nx - 1)), cy = __fmul_rn(0.5f, (float)(v.ny - 1)),
              cz = __fmul_rn(0.5f, (float)(v.nz - 1));
  const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(fnx, fnx), __fmul_rn(fny, fny)), __fmul_rn(fnz, fnz));
  const float T = __fmul_rn(0.5f, __fsqrt_rn(d2));
  const int K = (int)floorf(__fdiv_rn(__fmul_rn(2.0f, T), v.step)) + 1;
  const float hx = (float)(v.nx - 1), hy = (float)(v.ny - 1), hz = (float)(v.nz - 1);
  const float X = __fdiv_rn(__fsub_rn(__fadd_rn((float)px, 0.5f), __fmul_rn(0.5f, (float)v.width)), v.zoom);
  const float Y = __fdiv_rn(__fsub_rn(__fadd_rn((float)py, 0.5f), __fmul_rn(0.5f, (float)v.height)), v.zoom);
  // the part of the position that does not depend on the sample index
  const float bx = __fmaf_rn(v.rot[1], Y, __fmaf_rn(v.rot[0], X, cx));
  const float by = __fmaf_rn(v.rot[4], Y, __fmaf_rn(v.rot[3], X, cy));
  const float bz = __fmaf_rn(v.rot[7], Y, __fmaf_rn(v.rot[6], X, cz));
  // Samples outside the box are skipped by definition, so only the samples of a CONSERVATIVE
  // ray / box interval need visiting (slab test in plain float arithmetic, widened by 0.05
  // voxel and two samples; the exact per-sample test below still decides). Most rays of a
  // sparse vascular box cross a small part of the 2T march or miss it altogether.
  int k0 = 0, k1 = K - 1;
  {
    float z0 = -T, z1 = T;
    const float b[3] = {bx, by, bz}, h[3] = {hx, hy, hz}, r[3] = {v.rot[2], v.rot[5], v.rot[8]};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (fabsf(r[a]) > 1e-6f) {
        const float ta = (-0.05f - b[a]) / r[a], tb = (h[a] + 0.05f - b[a]) / r[a];
        z0 = fmaxf(z0, fminf(ta, tb));
        z1 = fminf(z1, fmaxf(ta, tb));
      } else if (b[a] < -0.05f || b[a] > h[a] + 0.05f) {
        z1 = z0 - 1.0f;  // parallel to the slab and outside it: misses
      }
    }
    if (z1 < z0) {
      k1 = -1;
    } else {
      k0 = max(0, (int)floorf((z0 + T) / v.step) - 2);
      k1 = min(K - 1, (int)ceilf((z1 + T) / v.step) + 2);
    }
  }
  // does the value 0 have zero opacity? (same operations as for a sample of value 0)
  bool skip_empty = false;
  if (occ) {
    const float t0 = clamp01(__fmaf_rn(0.0f, v.tf_scale, v.tf_offset));
    const int i0 = (int)__fmaf_rn(t0, 255.0f, 0.5f);
    skip_empty = clamp01(__fmul_rn(c_lut[4 * i0 + 3], v.opacity)) == 0.0f;
  }
  const int mx = (v.nx + 7) >> 3, my = (v.ny + 7) >> 3;
  const float r2[3] = {v.rot[2], v.rot[5], v.rot[8]};
  // per ray: 1 / (direction component) and 1 / step for the jump lengths (their rounding is
  // far inside the margin below)
  float inv[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) inv[a] = fabsf(r2[a]) > 1e-6f ? 1.0f / fabsf(r2[a]) : 0.0f;
  const float inv_step = 1.0f / v.step;
  float Cr = 0.0f, Cg = 0.0f, Cb = 0.0f, A = 0.0f;
  for (int k = k0; k <= k1; ++k) {
    const float Z = __fmaf_rn((float)k, v.step, -T);
    const float qx = __fmaf_rn(v.rot[2], Z, bx), qy = __fmaf_rn(v.rot[5], Z, by), qz = __fmaf_rn(v.rot[8], Z, bz);
    if (qx < 0.0f || qx > hx || qy < 0.0f || qy > hy || qz < 0.0f || qz > hz) continue;
    if (skip_empty) {
      // the cell of the sample's lower corner voxel, as trilinear() clamps it
      const int ix = max(min((int)floorf(qx), v.nx - 2), 0), iy = max(min((int)floorf(qy), v.ny - 2), 0),
                iz = max(min((int)floorf(qz), v.nz - 2), 0);
      const int cxm = ix >> 3, cym = iy >> 3, czm = iz >> 3;
      const int level = __ldg(occ + ((long long)czm * my + cym) * mx + cxm);
      if (level) {
        // level 2: the whole 64^3 super-cell around the macro-cell is empty
        const int sh = level == 2 ? 6 : 3;
        // conservative count of further samples whose lower corner stays in this cell: keep a
        // margin (>= 0.01 voxel, far above the rounding of the sample positions) clear of the
        // cell faces; an axis the ray hardly moves along must already be clear of them
        const float q[3] = {qx, qy, qz};
        const int c8[3] = {(ix >> sh) << sh, (iy >> sh) << sh, (iz >> sh) << sh};
        float room = 1e30f;  // distance in Z the ray may still travel
#pragma unroll
        for (int a = 0; a < 3; ++a) {
          const float margin = 0.01f * (1.0f + fabsf(r2[a]));
          const float hi = (float)(c8[a] + (1 << sh)) - margin - q[a], lo = q[a] - (float)c8[a] - margin;
          if (r2[a] > 1e-6f) room = fminf(room, hi * inv[a]);
          else if (r2[a] < -1e-6f) room = fminf(room, lo * inv[a]);
          else if (hi < 0.0f || lo < 0.0f) room = 0.0f;
        }
        // samples k+1 .. k+jump lie within `room` of this one: inside the cell, margin to spare
        const int jump = room > 0.0f ? (int)fminf(floorf(room * inv_step), 1.0e6f) : 0;
        if (jump > 0) k += jump;
        continue;
      }
    }
    const float val = trilinear<TEX>(vol, tex, v.nx, v.ny, v.nz, qx, qy, qz);
    const float t = clamp01(__fmaf_rn(val, v.tf_scale, v.tf_offset));
    const int i = (int)__fmaf_rn(t, 255.0f, 0.5f);
    const float* e = c_lut + 4 * i;
    const float a = clamp01(__fmul_rn(e[3], v.opacity));
    const float wgt = __fmul_rn(__fsub_rn(1.0f, A), a);
    Cr = __fmaf_rn(wgt, e[0], Cr);
    Cg = __fmaf_rn(wgt, e[1], Cg);
    Cb = __fmaf_rn(wgt, e[2], Cb);
    A = __fadd_rn(A, wgt);
    if (A >= 0.995f) break;
  }
  reinterpret_cast<float4*>(image)[(long long)py * v.width + px] = make_float4(Cr, Cg, Cb, A);
}

// volume[voxel of site c] = scalar field of site c (canonical order); the rest stays 0
__global__ void __launch_bounds__(256)
k_scatter_field(const double* __restrict__ rho, const double* __restrict__ u,
                const long long* __restrict__ voxel, long long N, int field, float* __restrict__ vol,
                cudaSurfaceObject_t surf, int nx, int ny) {
  const long long c = (long long)blockIdx.x * 256 + threadIdx.x;
  if (c >= N) return;
  double s;
  if (field == 2) {
    s = 1.0;  // marks the fluid voxels (occupancy of the geometry)
  } else if (field == 1) {
    s = rho[c] - 1.0;
  } else {
    const double ux = u[3 * c], uy = u[3 * c + 1], uz = u[3 * c + 2];
    s = sqrt(ux * ux + uy * uy + uz * uz);
  }
  const long long v = voxel[c];
  vol[v] = (float)s;
  if (surf) {  // the same value into the 3-D array behind the texture object
    const long long row = v / nx;
    surf3Dwrite((float)s, surf, (int)(v - row * nx) * (int)sizeof(float), (int)(row % ny), (int)(row / ny));
  }
}

}  // namespace

void launch_raymarch(const RenderSetup& r, const float* lut_host, const float* vol, cudaTextureObject_t tex,
                     const unsigned char* occ, float* image, cudaStream_t s) {
  RenderParams par;
  ViewParams& v = par.v;
  v.nx = r.nx; v.ny = r.ny; v.nz = r.nz; v.width = r.width; v.height = r.height;
  for (int k = 0; k < 9; ++k) v.rot[k] = r.rot[k];
  v.zoom = r.zoom; v.step = r.step; v.tf_scale = r.tf_scale; v.tf_offset = r.tf_offset; v.opacity = r.opacity;
  for (int k = 0; k < 1024; ++k) par.lut[k] = lut_host[k];
  const dim3 grid((unsigned)((r.width + TILE - 1) / TILE), (unsigned)((r.height + TILE - 1) / TILE));
  if (tex) k_raymarch<true><<<grid, dim3(TILE, TILE), 0, s>>>(par, vol, tex, occ, image);
  else k_raymarch<false><<<grid, dim3(TILE, TILE), 0, s>>>(par, vol, tex, occ, image);
}

namespace {
// one warp per macro-cell: 1 if all voxels of [8c, 8c + 8] (clipped to the box) are +0.0f bits
__global__ void __launch_bounds__(256)
k_occupancy(const float* __restrict__ vol, int nx, int ny, int nz, unsigned char* __restrict__ occ) {
  const int mx = (nx + 7) >> 3, my = (ny + 7) >> 3, mz = (nz + 7) >> 3;
  const long long cell = ((long long)blockIdx.x * 256 + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (cell >= (long long)mx * my * mz) return;
  const int cx = (int)(cell % mx), cy = (int)((cell / mx) % my), cz = (int)(cell / ((long long)mx * my));
  unsigned any = 0u;
  for (int t = lane; t < 9 * 9 * 9; t += 32) {
    const int x = (cx << 3) + t % 9, y = (cy << 3) + (t / 9) % 9, z = (cz << 3) + t / 81;
    if (x < nx && y < ny && z < nz) any |= __float_as_uint(__ldg(vol + ((long long)z * ny + y) * nx + x));
  }
  any = __reduce_or_sync(0xffffffffu, any);
  if (lane == 0) occ[cell] = any == 0u ? 1 : 0;
}
}  // namespace

namespace {
// one warp per 64^3 super-cell: if all of its macro-cells are empty, mark them 2
__global__ void __launch_bounds__(256)
k_occupancy_super(int mx, int my, int mz, unsigned char* __restrict__ occ) {
  const int sx = (mx + 7) >> 3, sy = (my + 7) >> 3, sz = (mz + 7) >> 3;
  const long long sc = ((long long)blockIdx.x * 256 + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (sc >= (long long)sx * sy * sz) return;
  const int bx = (int)(sc % sx) << 3, by = (int)((sc / sx) % sy) << 3, bz = (int)(sc / ((long long)sx * sy)) << 3;
  bool all = true;
  for (int t = lane; t < 512; t += 32) {
    const int x = bx + (t & 7), y = by + ((t >> 3) & 7), z = bz + (t >> 6);
    if (x < mx && y < my && z < mz && occ[((long long)z * my + y) * mx + x] == 0) all = false;
  }
  if (!__all_sync(0xffffffffu, all)) return;
  for (int t = lane; t < 512; t += 32) {
    const int x = bx + (t & 7), y = by + ((t >> 3) & 7), z = bz + (t >> 6);
    if (x < mx && y < my && z < mz) occ[((long long)z * my + y) * mx + x] = 2;
  }
}
}  // namespace

long long occupancy_cells(int nx, int ny, int nz) {
  return (long long)((nx + 7) >> 3) * ((ny + 7) >> 3) * ((nz + 7) >> 3);
}
void launch_occupancy(const float* vol, int nx, int ny, int nz, unsigned char* occ, cudaStream_t s) {
  const long long threads = occupancy_cells(nx, ny, nz) * 32;
  k_occupancy<<<(unsigned)((threads + 255) / 256), 256, 0, s>>>(vol, nx, ny, nz, occ);
  const int mx = (nx + 7) >> 3, my = (ny + 7) >> 3, mz = (nz + 7) >> 3;
  const long long sthreads = (long long)((mx + 7) >> 3) * ((my + 7) >> 3) * ((mz + 7) >> 3) * 32;
  k_occupancy_super<<<(unsigned)((sthreads + 255) / 256), 256, 0, s>>>(mx, my, mz, occ);
}

void launch_scatter_field(const double* rho, const double* u, const long long* voxel, long long N,
                          int field, float* vol, cudaSurfaceObject_t surf, int nx, int ny, cudaStream_t s) {
  k_scatter_field<<<(unsigned)((N + 255) / 256), 256, 0, s>>>(rho, u, voxel, N, field, vol, surf, nx, ny);
}

}  // namespace hlb
