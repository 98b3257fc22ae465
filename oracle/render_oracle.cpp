// render_oracle.cpp -- the ORACLE for the ray-marching volume renderer.
//
// TEST INFRASTRUCTURE ONLY (same rule as hlb_oracle.cpp): nothing in the product path may
// include, link or call this file; it shares no code with the CUDA renderer.
//
// What the paper says (all of it): "all the voxels for direct volume rendering are stored in
// the rendering layer ... The CUDA cores in the rendering layer perform the volume rendering
// kernel based on the ray marching algorithm [19]"; "the visualization volume is
// stored in a 3D texture unit to enable the fast sampling of voxel values ... to store the
// viewing parameters and the look-up table, the GPU constant memory buffers are used";
// "steerable parameters ... include zooming, model rotation and adjustment of scaling and
// offset of the transfer functions". No formula is given; what follows is textbook
// direct volume rendering by front-to-back compositing, with every choice the paper leaves
// open listed in DESIGN.md (reading R-render). Arithmetic is IEEE binary32 throughout (the
// renderer's precision), one operation per statement, fused only where fmaf() is written
// (the file is compiled with -ffp-contract=off), so that a faithful implementation agrees
// bit for bit.
//
// Geometry. Volume v[z][y][x], nx*ny*nz floats; voxel centres at integer coordinates. View:
// an orthographic camera looking along the view-space +z axis; `rot` (row-major 3x3) maps view
// space to volume space, v_vol = centre + rot * v_view, centre = ((nx-1)/2, (ny-1)/2,
// (nz-1)/2). Pixel (px, py) of a width x height image has view coordinates
//   X = (px + 0.5 - width/2) / zoom,  Y = (py + 0.5 - height/2) / zoom       (zoom: pixels per voxel)
// Its ray starts at view z = -T, T = 0.5 * sqrt(nx^2 + ny^2 + nz^2) (half the box diagonal,
// so every rotation keeps the whole box in range), and takes samples k = 0 .. K-1,
// K = floor(2T / step) + 1, at view z = -T + k * step.
// Sample: position p in volume space; if p is outside [0, nx-1] x [0, ny-1] x [0, nz-1] the
// sample is skipped; else the value is the trilinear interpolation of the 8 surrounding
// voxels (cell index clamped so that the upper corner exists).
// Transfer function: t = clamp(value * tf_scale + tf_offset, 0, 1); entry i = (int)(t * 255
// + 0.5) of the 256-entry RGBA look-up table; sample opacity a = clamp(lut.a * opacity, 0, 1).
// Compositing, front to back: C += (1 - A) * a * lut.rgb ; A += (1 - A) * a ; the ray stops
// once A >= 0.995. Output pixel: (C.r, C.g, C.b, A).

#include <cmath>
#include <cstdint>

namespace {

inline float clamp01(float x) { return x < 0.0f ? 0.0f : (x > 1.0f ? 1.0f : x); }

inline float trilinear(const float* vol, int nx, int ny, int nz, float px, float py, float pz) {
  int ix = (int)std::floor(px), iy = (int)std::floor(py), iz = (int)std::floor(pz);
  if (ix > nx - 2) ix = nx - 2;
  if (iy > ny - 2) iy = ny - 2;
  if (iz > nz - 2) iz = nz - 2;
  if (ix < 0) ix = 0;  // only when the axis has a single voxel
  if (iy < 0) iy = 0;
  if (iz < 0) iz = 0;
  const float fx = px - (float)ix, fy = py - (float)iy, fz = pz - (float)iz;
  const int x1 = ix + 1 < nx ? ix + 1 : ix, y1 = iy + 1 < ny ? iy + 1 : iy, z1 = iz + 1 < nz ? iz + 1 : iz;
  auto at = [&](int x, int y, int z) { return vol[((int64_t)z * ny + y) * nx + x]; };
  // interpolate along x, then y, then z: a + f * (b - a) written as fmaf(f, b - a, a)
  const float c00 = fmaf(fx, at(x1, iy, iz) - at(ix, iy, iz), at(ix, iy, iz));
  const float c10 = fmaf(fx, at(x1, y1, iz) - at(ix, y1, iz), at(ix, y1, iz));
  const float c01 = fmaf(fx, at(x1, iy, z1) - at(ix, iy, z1), at(ix, iy, z1));
  const float c11 = fmaf(fx, at(x1, y1, z1) - at(ix, y1, z1), at(ix, y1, z1));
  const float c0 = fmaf(fy, c10 - c00, c00);
  const float c1 = fmaf(fy, c11 - c01, c01);
  return fmaf(fz, c1 - c0, c0);
}

}  // namespace

extern "C" {

// One trilinear sample (exposed so that the interpolation can be pinned on its own).
float rendo_sample(const float* vol, int nx, int ny, int nz, float px, float py, float pz) {
  return trilinear(vol, nx, ny, nz, px, py, pz);
}

// image: [height][width][4] floats. rot: 9 floats row-major. lut: [256][4] floats.
// Returns the total number of samples taken inside the box (for the closed-form pins), or -1.
int64_t rendo_render(const float* vol, int nx, int ny, int nz, int width, int height,
                     const float* rot, float zoom, float step, float tf_scale, float tf_offset,
                     float opacity, const float* lut, float* image) {
  if (!vol || !rot || !lut || !image || nx <= 0 || ny <= 0 || nz <= 0 || width <= 0 || height <= 0 ||
      !(zoom > 0.0f) || !(step > 0.0f))
    return -1;
  const float cx = 0.5f * (float)(nx - 1), cy = 0.5f * (float)(ny - 1), cz = 0.5f * (float)(nz - 1);
  const float T = 0.5f * std::sqrt((float)nx * (float)nx + (float)ny * (float)ny + (float)nz * (float)nz);
  const int K = (int)std::floor(2.0f * T / step) + 1;
  const float hx = (float)(nx - 1), hy = (float)(ny - 1), hz = (float)(nz - 1);
  int64_t inside = 0;
  for (int py = 0; py < height; ++py)
    for (int px = 0; px < width; ++px) {
      const float X = ((float)px + 0.5f - 0.5f * (float)width) / zoom;
      const float Y = ((float)py + 0.5f - 0.5f * (float)height) / zoom;
      float Cr = 0.0f, Cg = 0.0f, Cb = 0.0f, A = 0.0f;
      for (int k = 0; k < K; ++k) {
        const float Z = fmaf((float)k, step, -T);
        // p = centre + rot * (X, Y, Z), accumulated left to right with fmaf
        const float qx = fmaf(rot[2], Z, fmaf(rot[1], Y, fmaf(rot[0], X, cx)));
        const float qy = fmaf(rot[5], Z, fmaf(rot[4], Y, fmaf(rot[3], X, cy)));
        const float qz = fmaf(rot[8], Z, fmaf(rot[7], Y, fmaf(rot[6], X, cz)));
        if (qx < 0.0f || qx > hx || qy < 0.0f || qy > hy || qz < 0.0f || qz > hz) continue;
        ++inside;
        const float v = trilinear(vol, nx, ny, nz, qx, qy, qz);
        const float t = clamp01(fmaf(v, tf_scale, tf_offset));
        const int i = (int)(fmaf(t, 255.0f, 0.5f));
        const float* e = lut + 4 * i;
        const float a = clamp01(e[3] * opacity);
        const float wgt = (1.0f - A) * a;
        Cr = fmaf(wgt, e[0], Cr);
        Cg = fmaf(wgt, e[1], Cg);
        Cb = fmaf(wgt, e[2], Cb);
        A = A + wgt;
        if (A >= 0.995f) break;
      }
      float* o = image + 4 * ((int64_t)py * width + px);
      o[0] = Cr; o[1] = Cg; o[2] = Cb; o[3] = A;
    }
  return inside;
}

}  // extern "C"
