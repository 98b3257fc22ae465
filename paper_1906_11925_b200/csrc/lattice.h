// lattice.h -- the library's velocity sets (host + device): D3Q15 and D3Q19.
//
// Ordering: q = 0 rest; 1..6 = +x -x +y -y +z -z; then the
// diagonals; opposite directions are adjacent, opp(q) = ((q - 1) ^ 1) + 1 for q >= 1, in both
// lattices. The paper names D3Q19 (Fig. 1, 103); BASELINE.json fixes
// D3Q15 for the headline metric, D3Q19 is SURVEY.md §8(f) NEXT-1.
//   D3Q15: weights 2/9, 1/9 (axis), 1/72 (cube diagonals)
//   D3Q19: weights 1/3, 1/18 (axis), 1/36 (face diagonals)
// c_s^2 = 1/3 in both. These tables are the product's own; the oracle builds its sets
// independently (by loops, in another order).
#pragma once
#include <cstdint>

namespace hlb {

#if defined(__CUDACC__)
#define HLB_HD __host__ __device__ __forceinline__
#else
#define HLB_HD inline
#endif

constexpr int MAXQ = 19;

HLB_HD constexpr int opp(int q) { return q == 0 ? 0 : (((q - 1) ^ 1) + 1); }

struct D3Q15 {
  static constexpr int Q = 15;
  //                                           q: 0  1   2  3   4  5   6  7   8  9  10 11  12 13  14
  static HLB_HD constexpr int cx(int q) { constexpr int t[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1}; return t[q]; }
  static HLB_HD constexpr int cy(int q) { constexpr int t[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, 1, -1, -1, 1, -1, 1}; return t[q]; }
  static HLB_HD constexpr int cz(int q) { constexpr int t[Q] = {0, 0, 0, 0, 0, 1, -1, 1, -1, -1, 1, 1, -1, -1, 1}; return t[q]; }
  static HLB_HD constexpr double weight(int q) { return q == 0 ? 2.0 / 9.0 : (q <= 6 ? 1.0 / 9.0 : 1.0 / 72.0); }
};

struct D3Q19 {
  static constexpr int Q = 19;
  //                                           q: 0  1   2  3   4  5   6  7   8  9  10 11  12 13  14 15  16 17  18
  static HLB_HD constexpr int cx(int q) { constexpr int t[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0}; return t[q]; }
  static HLB_HD constexpr int cy(int q) { constexpr int t[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, -1, 1, 0, 0, 0, 0, 1, -1, 1, -1}; return t[q]; }
  static HLB_HD constexpr int cz(int q) { constexpr int t[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, -1, 1, 1, -1, -1, 1}; return t[q]; }
  static HLB_HD constexpr double weight(int q) { return q == 0 ? 1.0 / 3.0 : (q <= 6 ? 1.0 / 18.0 : 1.0 / 36.0); }
};

// Run-time description of a lattice for host code (preprocessor, API).
struct LatticeDesc {
  int Q;
  int c[MAXQ][3];
  double w[MAXQ];
};
template <typename L>
inline LatticeDesc make_desc() {
  LatticeDesc d{};
  d.Q = L::Q;
  for (int q = 0; q < L::Q; ++q) {
    d.c[q][0] = L::cx(q); d.c[q][1] = L::cy(q); d.c[q][2] = L::cz(q);
    d.w[q] = L::weight(q);
  }
  return d;
}
inline const LatticeDesc& lattice_desc(bool d3q19) {
  static const LatticeDesc a = make_desc<D3Q15>(), b = make_desc<D3Q19>();
  return d3q19 ? b : a;
}

// The relaxation constants of one geometry as the step kernels take them (by value), computed
// on the host (IEEE double products, bit-identical to __dmul_rn): omega = 1 / tau for the
// difference form of the relaxation; omc = 1 - omega and the rest / axis / diagonal weights
// times omega (w0, wa, wd) and times 3 omega (a3, d3) for the folded form (lbgk.cuh).
struct Relax {
  double omega, omc, w0, wa, wd, a3, d3;
};
template <typename L>
inline Relax make_relax(double omega) {
  Relax r;
  r.omega = omega;
  r.omc = 1.0 - omega;
  r.w0 = L::weight(0) * omega;
  r.wa = L::weight(1) * omega;
  r.wd = L::weight(7) * omega;
  r.a3 = 3.0 * L::weight(1) * omega;
  r.d3 = 3.0 * L::weight(7) * omega;
  return r;
}

// neighbour-table entry encoding (include/hlb.h, hlb_preprocess_tables)
constexpr uint32_t NBR_WALL_BIT = 0x80000000u;

}  // namespace hlb
