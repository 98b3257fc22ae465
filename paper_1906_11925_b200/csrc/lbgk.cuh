// lbgk.cuh -- per-site D3Q15 LBGK arithmetic (device), shared by every kernel variant so
// that the two-lattice and A-A schemes, fp64 and fp32 storage, are bitwise identical in
// their arithmetic (SURVEY.md §8(c) pin P14).
//
// Rest-state-shifted form (reading R-shift): registers hold h_q = f_q - w_q.
//   drho = sum_q h_q, rho = 1 + drho, j = sum_q c_q h_q, u = j / rho
//   heq_q = w_q [ drho + rho (3 c_q.u + 4.5 (c_q.u)^2 - 1.5 u.u) ]
//   h*_q  = h_q + omega (heq_q - h_q),  omega = 1 / tau                      (LBGK)
// ("collision"; LBGK and the equilibrium: BASELINE.json north_star and
// the paper gives no formula).
#pragma once
#include "d3q15.h"

namespace hlb {

struct Moments {
  double drho, rho, ux, uy, uz;
};

// Opposite pairs (2k-1, 2k), k = 1..7, first member has c = (1,0,0) (0,1,0) (0,0,1)
// (1,1,1) (1,1,-1) (1,-1,1) (1,-1,-1): sums and differences of pairs give all moments.
__device__ __forceinline__ Moments moments_of(const double (&h)[Q]) {
  const double d1 = h[1] - h[2], d2 = h[3] - h[4], d3 = h[5] - h[6];
  const double d4 = h[7] - h[8], d5 = h[9] - h[10], d6 = h[11] - h[12], d7 = h[13] - h[14];
  const double s_axis = ((h[1] + h[2]) + (h[3] + h[4])) + (h[5] + h[6]);
  const double s_diag = ((h[7] + h[8]) + (h[9] + h[10])) + ((h[11] + h[12]) + (h[13] + h[14]));
  Moments m;
  m.drho = h[0] + (s_axis + s_diag);
  m.rho = 1.0 + m.drho;
  const double jx = d1 + ((d4 + d5) + (d6 + d7));
  const double jy = d2 + ((d4 + d5) - (d6 + d7));
  const double jz = d3 + ((d4 - d5) + (d6 - d7));
  const double inv = 1.0 / m.rho;
  m.ux = jx * inv;
  m.uy = jy * inv;
  m.uz = jz * inv;
  return m;
}

// Shifted equilibrium of direction q (compile-time q after unrolling) for density
// 1 + drho and velocity (ux, uy, uz).
__device__ __forceinline__ double heq_of(int q, double drho, double rho, double ux, double uy,
                                         double uz) {
  const double cu = (double)cx(q) * ux + (double)cy(q) * uy + (double)cz(q) * uz;
  const double uu = ux * ux + uy * uy + uz * uz;
  return weight(q) * (drho + rho * (3.0 * cu + 4.5 * cu * cu - 1.5 * uu));
}

// hs_q = h_q + omega (heq_q(m) - h_q)
__device__ __forceinline__ void collide(const double (&h)[Q], const Moments& m, double omega,
                                        double (&hs)[Q]) {
  const double uu15 = 1.5 * (m.ux * m.ux + m.uy * m.uy + m.uz * m.uz);
#pragma unroll
  for (int q = 0; q < Q; ++q) {
    const double cu = (double)cx(q) * m.ux + (double)cy(q) * m.uy + (double)cz(q) * m.uz;
    const double heq = weight(q) * (m.drho + m.rho * ((3.0 * cu + 4.5 * cu * cu) - uu15));
    hs[q] = h[q] + omega * (heq - h[q]);
  }
}

// storage <-> arithmetic conversions (HLB_STORE_F64 / HLB_STORE_F32; include/hlb.h)
__device__ __forceinline__ double to_real(double v) { return v; }
__device__ __forceinline__ double to_real(float v) { return (double)v; }
template <typename ST> __device__ __forceinline__ ST to_store(double v);
template <> __device__ __forceinline__ double to_store<double>(double v) { return v; }
template <> __device__ __forceinline__ float to_store<float>(double v) { return __double2float_rn(v); }

}  // namespace hlb
