// d3q15.h -- the library's D3Q15 velocity set (host + device).
//
// Ordering: q = 0 rest; opposite directions are adjacent,
// opp(q) = ((q - 1) ^ 1) + 1 for q >= 1. The paper names D3Q19;
// BASELINE.json fixes D3Q15. Weights 2/9, 1/9 (axis), 1/72 (diagonal),
// c_s^2 = 1/3. This table is the product's own; the oracle builds its set independently.
#pragma once
#include <cstdint>

namespace hlb {

constexpr int Q = 15;

#if defined(__CUDACC__)
#define HLB_HD __host__ __device__ __forceinline__
#else
#define HLB_HD inline
#endif

//                                   q: 0  1   2  3   4  5   6  7   8  9  10 11  12 13  14
HLB_HD constexpr int cx(int q) { constexpr int t[Q] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1}; return t[q]; }
HLB_HD constexpr int cy(int q) { constexpr int t[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, 1, -1, -1, 1, -1, 1}; return t[q]; }
HLB_HD constexpr int cz(int q) { constexpr int t[Q] = {0, 0, 0, 0, 0, 1, -1, 1, -1, -1, 1, 1, -1, -1, 1}; return t[q]; }
HLB_HD constexpr int opp(int q) { return q == 0 ? 0 : (((q - 1) ^ 1) + 1); }
HLB_HD constexpr double weight(int q) { return q == 0 ? 2.0 / 9.0 : (q <= 6 ? 1.0 / 9.0 : 1.0 / 72.0); }

// neighbour-table entry encoding (include/hlb.h, hlb_preprocess_tables)
constexpr uint32_t NBR_WALL_BIT = 0x80000000u;
HLB_HD constexpr bool nbr_is_wall(int32_t e) { return e < 0; }                 // solid or iolet
HLB_HD constexpr int nbr_iolet(int32_t e) { return (int)(e & 0x7fffffff) - 1; }  // -1: plain wall

}  // namespace hlb
