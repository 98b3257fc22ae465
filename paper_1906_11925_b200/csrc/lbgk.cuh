// lbgk.cuh -- per-site LBGK arithmetic (device), for either lattice of lattice.h, shared by
// every kernel variant so that the two-lattice and A-A schemes, fp64 and fp32 storage, are
// bitwise identical in their arithmetic (SURVEY.md §8(c) pin P14).
//
// Rest-state-shifted form (reading R-shift): registers hold h_q = f_q - w_q.
//   drho = sum_q h_q, rho = 1 + drho, j = sum_q c_q h_q, u = j / rho
//   heq_q = w_q [ drho + rho (3 c_q.u + 4.5 (c_q.u)^2 - 1.5 u.u) ]
//   h*_q  = h_q + omega (heq_q - h_q),  omega = 1 / tau                      (LBGK)
// ("collision"; LBGK and the equilibrium: BASELINE.json north_star and
// the paper gives no formula).
#pragma once
#include "lattice.h"

namespace hlb {

struct Moments {
  double drho, rho, ux, uy, uz;
};

// Every floating-point operation below is an explicit round-to-nearest intrinsic
// (__dadd_rn / __dmul_rn / __fma_rn): the compiler may neither contract nor split them, so
// all kernel instantiations (two-lattice, A-A even / odd, table or records, fp64 or fp32
// storage) evaluate bit-identical arithmetic whatever their register allocation or inlining
// context (SURVEY.md §8(c) pin P14).
__device__ __forceinline__ double add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double sub(double a, double b) { return __dadd_rn(a, -b); }
__device__ __forceinline__ double mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return __fma_rn(a, b, c); }

// c_q . u with the +-1 / 0 components folded at compile time (exact: only additions)
template <typename L>
__device__ __forceinline__ double c_dot_u(int q, double ux, double uy, double uz) {
  double r = 0.0;
  bool first = true;
  const int c[3] = {L::cx(q), L::cy(q), L::cz(q)};
  const double u[3] = {ux, uy, uz};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (c[a] == 0) continue;
    const double t = c[a] > 0 ? u[a] : -u[a];
    r = first ? t : add(r, t);
    first = false;
  }
  return r;
}

// Moments from the opposite pairs (a, b) = (2k-1, 2k), c_b = -c_a: with s_k = h_a + h_b and
// d_k = h_a - h_b,  drho = h_0 + sum_k s_k  and  j = sum_k c_a d_k.
template <typename L>
__device__ __forceinline__ Moments moments_of(const double (&h)[L::Q]) {
  constexpr int P = (L::Q - 1) / 2;
  double s[P], d[P];
#pragma unroll
  for (int k = 0; k < P; ++k) {
    s[k] = add(h[2 * k + 1], h[2 * k + 2]);
    d[k] = sub(h[2 * k + 1], h[2 * k + 2]);
  }
  // axis pairs first, then the diagonals, each summed pairwise
  double s_axis = add(add(s[0], s[1]), s[2]);
  double s_diag = add(s[3], s[4]);
#pragma unroll
  for (int k = 5; k + 1 < P; k += 2) s_diag = add(s_diag, add(s[k], s[k + 1]));
  if ((P - 5) % 2) s_diag = add(s_diag, s[P - 1]);
  Moments m;
  m.drho = add(h[0], add(s_axis, s_diag));
  m.rho = add(1.0, m.drho);
  double j[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double acc = 0.0;
    bool first = true;
#pragma unroll
    for (int k = 0; k < P; ++k) {
      const int q = 2 * k + 1;
      const int c = a == 0 ? L::cx(q) : (a == 1 ? L::cy(q) : L::cz(q));
      if (c == 0) continue;
      const double t = c > 0 ? d[k] : -d[k];
      acc = first ? t : add(acc, t);
      first = false;
    }
    j[a] = acc;
  }
  const double inv = __drcp_rn(m.rho);
  m.ux = mul(j[0], inv);
  m.uy = mul(j[1], inv);
  m.uz = mul(j[2], inv);
  return m;
}

__device__ __forceinline__ double u_dot_u(double ux, double uy, double uz) {
  return fma_(ux, ux, fma_(uy, uy, mul(uz, uz)));
}

// Shifted equilibrium of direction q (compile-time q after unrolling) for density
// 1 + drho and velocity (ux, uy, uz): w_q [drho + rho (3 c.u + 4.5 (c.u)^2 - 1.5 u.u)].
template <typename L>
__device__ __forceinline__ double heq_of(int q, double drho, double rho, double ux, double uy,
                                         double uz) {
  const double cu = c_dot_u<L>(q, ux, uy, uz);
  const double uu15 = mul(1.5, u_dot_u(ux, uy, uz));
  const double poly = add(mul(3.0, cu), fma_(mul(4.5, cu), cu, -uu15));
  return mul(L::weight(q), fma_(rho, poly, drho));
}

// hs_q = h_q + omega (heq_q(m) - h_q), evaluated per opposite pair (a, b = opp(a)), c = c_a:
//   heq_a = S + A, heq_b = S - A,  S = w (drho + rho (4.5 (c.u)^2 - 1.5 u.u)),  A = 3 w rho (c.u)
// -- the same equilibrium as heq_of(), with the part even in c computed once per pair (a
// third fewer fp64 operations; the kernels run into the 1 kW power cap otherwise).
//
// Two forms of the relaxation, chosen by the storage type (profiles/r02_tuning.md):
//   FOLDED = false (fp64 storage): applied to the DIFFERENCE, h + omega ((S +- A) - h). heq - h
//     is small and nearly exact, so this is the accurate form: E_u ~ 4e-15 on configs[2] after
//     2000 steps against the oracle.
//   FOLDED = true (fp32 storage): (1 - omega) h + (omega S +- omega A) with omega folded into
//     the weights on the host -- one operation and one dependent step less per direction,
//     1-4 % faster on the fp32-storage kernels (which are latency-, not HBM-bound), and 30x
//     less accurate in fp64 terms (E_u 1.2e-13), which is six orders below the rounding of the
//     stored binary32 values themselves (E_u ~ 1e-7, bar 1e-5).
// emit(q, hs_q) is called as soon as a post-collision value is known, so that a kernel can
// store it at once and free its registers (and those of its address): with all stores after
// the whole collision the A-A odd kernel kept 7 of its 14 offsets in local memory.
// emit0(hs_0) and emit2(a, hs_a, hs_b) for each opposite pair (a, b = a + 1): the form the kernels
// with interpolated walls use -- both BFL rules mix the two members of one pair only.
template <typename L, bool FOLDED, typename F0, typename F2>
__device__ __forceinline__ void collide_emit_pairs(const double (&h)[L::Q], const Moments& m, const Relax& rx,
                                                   F0&& emit0, F2&& emit2) {
  const double uu15 = mul(1.5, u_dot_u(m.ux, m.uy, m.uz));
  if (FOLDED) {
    emit0(fma_(rx.omc, h[0], mul(rx.w0, fma_(-m.rho, uu15, m.drho))));
    const double r3_axis = mul(rx.a3, m.rho), r3_diag = mul(rx.d3, m.rho);
#pragma unroll
    for (int a = 1; a < L::Q; a += 2) {
      const int b = a + 1;  // opp(a)
      const double cu = c_dot_u<L>(a, m.ux, m.uy, m.uz);
      const double S = mul(a <= 6 ? rx.wa : rx.wd, fma_(m.rho, fma_(mul(4.5, cu), cu, -uu15), m.drho));
      const double A = mul(a <= 6 ? r3_axis : r3_diag, cu);
      emit2(a, fma_(rx.omc, h[a], add(S, A)), fma_(rx.omc, h[b], sub(S, A)));
    }
  } else {
    const double omega = rx.omega;
    const double heq0 = mul(L::weight(0), fma_(-m.rho, uu15, m.drho));
    emit0(fma_(omega, sub(heq0, h[0]), h[0]));
    // two weight classes: axis (q = 1..6) and diagonal (q >= 7)
    const double r3_axis = mul(3.0 * L::weight(1), m.rho), r3_diag = mul(3.0 * L::weight(7), m.rho);
#pragma unroll
    for (int a = 1; a < L::Q; a += 2) {
      const int b = a + 1;  // opp(a)
      const double cu = c_dot_u<L>(a, m.ux, m.uy, m.uz);
      const double S = mul(L::weight(a), fma_(m.rho, fma_(mul(4.5, cu), cu, -uu15), m.drho));
      const double A = mul(a <= 6 ? r3_axis : r3_diag, cu);
      const double ha = h[a], hb = h[b];
      emit2(a, fma_(omega, sub(add(S, A), ha), ha), fma_(omega, sub(sub(S, A), hb), hb));
    }
  }
}
template <typename L, bool FOLDED, typename F>
__device__ __forceinline__ void collide_emit(const double (&h)[L::Q], const Moments& m, const Relax& rx,
                                             F&& emit) {
  collide_emit_pairs<L, FOLDED>(h, m, rx, [&](double v) { emit(0, v); },
                                [&](int a, double va, double vb) { emit(a, va); emit(a + 1, vb); });
}
template <typename L, bool FOLDED>
__device__ __forceinline__ void collide(const double (&h)[L::Q], const Moments& m, const Relax& rx,
                                        double (&hs)[L::Q]) {
  collide_emit<L, FOLDED>(h, m, rx, [&](int q, double v) { hs[q] = v; });
}

// storage <-> arithmetic conversions (HLB_STORE_F64 / HLB_STORE_F32; include/hlb.h)
__device__ __forceinline__ double to_real(double v) { return v; }
__device__ __forceinline__ double to_real(float v) { return (double)v; }
template <typename ST> __device__ __forceinline__ ST to_store(double v);
template <> __device__ __forceinline__ double to_store<double>(double v) { return v; }
template <> __device__ __forceinline__ float to_store<float>(double v) { return __double2float_rn(v); }

}  // namespace hlb
