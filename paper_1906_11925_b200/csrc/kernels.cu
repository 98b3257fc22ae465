// kernels.cu -- fused LBGK collide-and-stream kernels for sm_100a (D3Q15 and D3Q19).
//
// One thread per fluid site, 128 threads per block, one-shot grids of Ns / 128 blocks.
// Populations are structure-of-arrays buf[slot][site] with plane stride Ns (a multiple of
// 128, planes 1 KiB aligned), so the own-site loads and all stores of a warp are single fully
// coalesced requests; the Q - 1 gathers follow the pull links.
// ~0.7 flop/byte: HBM-bound, no tensor cores, no staging of populations in shared memory (every
// population is read exactly once per step: there is no intra-block reuse to stage; cp.async /
// TMA staging was measured slower, profiles/r01_tuning.md).
//
// What the kernels are shaped by (evidence in profiles/):
//   * links come as 16-byte run-length records per (warp, link) -- up to three runs of consecutive
//     sources -- instead of 32 table entries, decoded with five integer operations per link; the
//     int32 table is the fallback for the rest;
//   * 32-bit flat offsets, explicit round-to-nearest fp64 intrinsics, pair-symmetric BGK:
//     few instructions, because long runs sit at the 1 kW power cap;
//   * 70-80 registers so that 6-7 blocks are resident per SM (more blocks HURT the fp64 kernels):
//     all link loads are issued first, then all population loads, then the arithmetic, and
//     every value is stored the moment it is known;
//   * threads L2-prefetch what the sites 0.68 MB per plane ahead (3/4 of a wave in fp64) will load;
//   * iolets (constant density, Ladd velocity) are a rare path behind one {bits, rank} word per
//     group of 32 sites, loaded with the first loads, and one row of link -> iolet bytes per cap site;
//   * BFL interpolated walls are a third instantiation (V = 2) that applies both rules to
//     registers; the lean (V = 0) and full (V = 1) instantiations carry none of its code.
//
// Sites i in [N, Ns) are padding: their links are all "wall", their populations are 0 (rest
// state in shifted form) and stay exactly 0, so no step kernel needs a bounds branch.
#include "kernels.cuh"

#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <tuple>

#include "lbgk.cuh"

namespace hlb {
namespace {

constexpr int BLOCK = 256;   // read-out / init kernels

#ifndef HLB_STEP_BLOCK
#define HLB_STEP_BLOCK 128   // Ns is a multiple of 128: the step kernels need no bounds test
#endif
// Resident blocks per SM each step kernel's register budget is tuned for (measured on
// B200, profiles/r01_tuning.md): 7 x 128 threads at <= 72 registers for the pull kernel,
// 6 x 128 at <= 80 for the two A-A kernels. Fewer registers spill the 15 populations,
// more cut the loads in flight. The table-reading variants (REC = false) hold 14 more
// live values and get one block less.
#ifndef HLB_PULL_MINB
#define HLB_PULL_MINB 7
#endif
#ifndef HLB_AA_EVEN_MINB
#define HLB_AA_EVEN_MINB 6
#endif
#ifndef HLB_AA_ODD_MINB
#define HLB_AA_ODD_MINB 6
#endif
constexpr int SBLOCK = HLB_STEP_BLOCK;
// D3Q19 keeps 4 more populations (8 registers) and 4 more offsets alive: two blocks less
// (measured: 20.8k vs 20.5k MSUPS A-A, 20.1k vs 19.5k pull on configs[4]).
#ifndef HLB_Q19_MINB_DROP
#define HLB_Q19_MINB_DROP 2
#endif
template <typename L, bool REC> constexpr int pull_minb() {
  return HLB_PULL_MINB - (REC ? 0 : 1) - (L::Q > 15 ? HLB_Q19_MINB_DROP : 0);
}
template <typename L, bool REC> constexpr int aa_odd_minb() {
  return HLB_AA_ODD_MINB - (REC ? 0 : 1) - (L::Q > 15 ? HLB_Q19_MINB_DROP : 0);
}
// The even kernel keeps no offsets: with 4-byte populations it fits 72 registers without
// spills, and the seventh block is worth 2.5 % there (0.704 vs 0.723 ms on configs[4]; nothing
// in fp64, where it sits at the copy rate already).
// k_pull with 8-byte storage and link records gets 80 registers (6 blocks): with the three-run
// decode on its general path ptxas' tighter 72-register allocation cost it 2.7 % on configs[4]
// (1.478 -> 1.515 ms; at 6 blocks 1.491, configs[3] 0.199 either way); 4-byte storage stays at 7
// (0.870 vs 0.890 ms). profiles/r02_tuning.md section 14.
#ifndef HLB_PULL_F64_DROP
#define HLB_PULL_F64_DROP 1
#endif
template <typename L, typename ST, bool REC> constexpr int pull_f64_drop() {
  return sizeof(ST) == 8 && REC && L::Q == 15 ? HLB_PULL_F64_DROP : 0;
}
// (see link_offsets: shared-memory records in the 4-byte-storage A-A odd kernel)
template <typename ST, bool REC> constexpr bool odd_rec_smem() { return sizeof(ST) == 4 && REC; }
// Interpolated walls (V = 2) with 8-byte storage: the gather kernels take one block MORE (7, 72
// registers, 8-20 offsets and coefficients in local memory) -- their flagged warps wait for a
// coefficient row on top of everything else, and more warps hide that better than registers
// do: k_aa_odd 0.233 -> 0.226 ms, k_pull 0.212 -> 0.2095 on configs[3] with every wall link
// interpolated; 5 blocks 0.245, 8 blocks 0.255 / 0.225; the even kernel 0.194 either way. With
// 4-byte storage the odd kernel keeps its seventh block with V = 2 as well (0.185 -> 0.179 ms).
// D3Q19: k_aa_odd 4 -> 5 blocks 0.3145 -> 0.2944 ms (6: 0.3276); k_pull stays at 5 (6: 0.272 -> 0.283).
// (profiles/r02_tuning.md section 15)
#ifndef HLB_BFL_GATHER_ADD
#define HLB_BFL_GATHER_ADD 1
#endif
// D3Q19 with 4-byte storage (V != 2, 32-bit offsets): the populations wait in 19 registers, not
// 38, and these kernels are latency-bound like their D3Q15 twins, so the A-A kernels take two
// blocks more than with 8-byte storage (6; ms per launch on configs[4] / configs[3], same call:
// even 4 blocks 1.016 / 0.139, 5: 0.918 / 0.128, 6: 0.906 / 0.128, 7: 0.919 / 0.126; odd 4: 1.280 /
// 0.203, 5: 1.234 / 0.191, 6: 1.225 / 0.187, 7: 1.259 / 0.190). k_pull stays at 5 (6: 1.190 ->
// 1.233, 7: 1.401). profiles/r02_tuning.md section 21.
#ifndef HLB_Q19F_EVEN_ADD
#define HLB_Q19F_EVEN_ADD 2
#endif
#ifndef HLB_Q19F_ODD_ADD
#define HLB_Q19F_ODD_ADD 2
#endif
#ifndef HLB_Q19F_PULL_ADD
#define HLB_Q19F_PULL_ADD 0
#endif
// 64-bit offsets (above 286 M sites, or HLB_INDEX64): 14 offsets are 28 registers; at 80 the odd
// kernel kept them in local memory (120 B of stack). One block less (96 registers): configs[4]
// forced onto the 64-bit kernels 1.553 -> 1.442 ms per A-A step in fp64, 0.923 -> 0.862 with 4-byte
// storage; two blocks less 1.449 / 0.909 (profiles/r02_tuning.md section 22).
#ifndef HLB_IDX64_ODD_DROP
#define HLB_IDX64_ODD_DROP 1
#endif
template <typename L, typename ST, bool REC, typename IT, int V> constexpr int odd_smem_minb_add() {
  if (V != 2 && sizeof(IT) == 8 && L::Q == 15) return -HLB_IDX64_ODD_DROP;
  if (V == 2 && sizeof(ST) == 8) return sizeof(IT) == 4 ? HLB_BFL_GATHER_ADD : 0;
  if (V != 2 && sizeof(ST) == 4 && L::Q == 19 && sizeof(IT) == 4 && REC) return HLB_Q19F_ODD_ADD;
  return odd_rec_smem<ST, REC>() && L::Q == 15 && sizeof(IT) == 4 ? 1 : 0;  // (64-bit offsets: spills)
}
template <typename L, typename ST> constexpr int aa_even_minb() {
  return HLB_AA_EVEN_MINB + (sizeof(ST) == 4 && L::Q == 15 ? 1 : 0) - (L::Q > 15 ? HLB_Q19_MINB_DROP : 0) +
         (sizeof(ST) == 4 && L::Q == 19 ? HLB_Q19F_EVEN_ADD : 0);
}
template <typename L, typename ST, typename IT, int V> constexpr int bfl_pull_add() {
  if (V != 2 && sizeof(ST) == 4 && L::Q == 19 && sizeof(IT) == 4) return HLB_Q19F_PULL_ADD;
  return V == 2 && sizeof(ST) == 8 && L::Q == 15 && sizeof(IT) == 4 ? HLB_BFL_GATHER_ADD : 0;
}

template <typename L>
__device__ __forceinline__ void load_entries(const int32_t* __restrict__ nbr, long long Ns,
                                             long long i, int32_t (&e)[L::Q - 1]) {
#pragma unroll
  for (int q = 1; q < L::Q; ++q) e[q - 1] = __ldg(nbr + (long long)(q - 1) * Ns + i);
}

// Flat element offsets (slot * Ns + site) of the 14 link populations of site i, for the step
// kernels. IT is the offset type: uint32_t when 15 * Ns < 2^32 (one IMAD.WIDE per access
// instead of 64-bit index arithmetic -- the integer work matters: these kernels run at the
// chip's power cap), long long otherwise.
//   MODE GATHER_PULL  : fluid source e -> q * Ns + e       ; wall -> opp(q) * Ns + i
//   MODE GATHER_AA_ODD: fluid source e -> opp(q) * Ns + e  ; wall -> q * Ns + i
// With REC the warp reads one 16-byte record per link instead of 32 table entries
// (include/hlb.h, hlb_preprocess_records): source = own index + the delta of the lane's run; a
// sentinel record (warp-uniform) sends the warp to the table for that link. The iolet id is
// NOT decoded here; the rare iolet path has its own row of link -> iolet bytes.
// -DHLB_BOUNDS_CHECK (debug builds only; compute-sanitizer is not available on every box):
// every flat offset a step kernel is about to gather from / scatter to must lie inside the
// Q * Ns elements of a population array, else the kernel traps and the next CUDA call fails.
// (-DHLB_BOUNDS_SELFTEST=1 shrinks the limit by one plane so that legitimate accesses trap:
// the negative control that shows the check is live.)
#ifndef HLB_BOUNDS_SELFTEST
#define HLB_BOUNDS_SELFTEST 0
#endif
template <typename L, typename IT>
__device__ __forceinline__ void check_offsets(const IT (&off)[L::Q - 1], long long Ns) {
#ifdef HLB_BOUNDS_CHECK
#pragma unroll
  for (int q = 1; q < L::Q; ++q)
    if ((unsigned long long)off[q - 1] >= (unsigned long long)(L::Q - HLB_BOUNDS_SELFTEST) * (unsigned long long)Ns) __trap();
#else
  (void)off; (void)Ns;
#endif
}

// q * Ns for q = 0 .. Q-1 as 32-bit values in the kernel's parameter space (constant bank):
// the decode adds them as an instruction operand instead of computing q * Ns per thread.
// Meaningful when Q * Ns < 2^32 (the 32-bit offset instantiations); the others ignore it.
struct Planes {
  uint32_t p[MAXQ];
};
// SMEM (with REC): the Q - 1 records of a warp are the same for its 32 lanes; held in registers
// by every lane they are the register peak of a gather kernel (14 x 4 = 56). With SMEM lane
// l < Q - 1 loads record l (ONE load instruction per warp), the warp's slice of shared memory
// holds them, and each link reads its record back by broadcast right before it is decoded.
// Used where the freed registers buy a resident block that pays: the A-A odd kernel with 4-byte
// storage (0.942 -> 0.902 ms on configs[4] at 7 blocks per SM). The fp64 kernels and the
// two-lattice kernel lose 1-5 % with it, with or without the extra block
// (profiles/r02_tuning.md section 13).
template <typename L, int MODE, bool REC, typename IT, bool SMEM = false>
__device__ __forceinline__ void link_offsets(const int32_t* __restrict__ nbr,
                                             const uint4* __restrict__ rec, long long Ns,
                                             long long i, const Planes& pl, IT (&off)[L::Q - 1]) {
  const IT n = (IT)Ns, self = (IT)i;
  if (!REC) {
    int32_t e[L::Q - 1];
#pragma unroll
    for (int q = 1; q < L::Q; ++q) e[q - 1] = __ldg(nbr + (long long)(q - 1) * Ns + i);
#pragma unroll
    for (int q = 1; q < L::Q; ++q) {
      const int qf = MODE == GATHER_PULL ? q : opp(q), qw = MODE == GATHER_PULL ? opp(q) : q;
      off[q - 1] = e[q - 1] < 0 ? (IT)qw * n + self : (IT)qf * n + (IT)e[q - 1];
    }
    check_offsets<L, IT>(off, Ns);
    return;
  }
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t lane_bit = 1u << lane;
  const uint4* r = rec + (i >> 5) * (L::Q - 1);
  // second <= 32 in a real record, 0xffffffff in a sentinel: one warp-uniform test decides
  // whether this warp needs the table at all, so the common path carries no sentinel code
  __shared__ uint4 s_rec[SMEM ? SBLOCK / 32 : 1][SMEM ? L::Q - 1 : 1];
  uint4 v_reg[SMEM ? 1 : L::Q - 1];
  uint4* v = SMEM ? s_rec[threadIdx.x >> 5] : v_reg;
  // word y of a record: second (<= 32) alone when the link has one or two runs; bit 6 set with a
  // third run (include/hlb.h); 0xffffffff = sentinel. "simple" = all Q - 1 records of the warp
  // have at most two runs: the path nearly every warp takes.
  bool simple;
  if (SMEM) {
    bool plain_here = true;
    if (lane < L::Q - 1) {
      const uint4 mine = __ldg(r + lane);
      v[lane] = mine;
      plain_here = (mine.y & 0x80000040u) == 0u;
    }
    simple = __all_sync(0xffffffffu, plain_here);
    __syncwarp();
  } else {
#pragma unroll
    for (int q = 1; q < L::Q; ++q) v[q - 1] = __ldg(r + (q - 1));
    uint32_t any = 0u;
#pragma unroll
    for (int q = 1; q < L::Q; ++q) any |= v[q - 1].y;
    simple = (any & 0x80000040u) == 0u;
  }
  if (simple) {
    // offset = own index + delta + plane: delta is the run's (source - own index), or, at a
    // wall lane, the step from plane qf to plane qw at the site itself -- five integer
    // instructions per link (compare, select, mask test, select, 3-input add)
#pragma unroll
    for (int q = 1; q < L::Q; ++q) {
      const int qf = MODE == GATHER_PULL ? q : opp(q), qw = MODE == GATHER_PULL ? opp(q) : q;
      const uint4 t = v[q - 1];
      uint32_t d = lane >= t.y ? t.w : t.z;
      if (sizeof(IT) == 4) {
        d = (t.x & lane_bit) ? (uint32_t)(qw - qf) * (uint32_t)n : d;
        off[q - 1] = (IT)((uint32_t)self + d + pl.p[qf]);
      } else {
        const long long dd = (t.x & lane_bit) ? (long long)(qw - qf) * (long long)n : (long long)(int32_t)d;
        off[q - 1] = (IT)((long long)self + dd + (long long)qf * (long long)n);
      }
    }
  } else {
#pragma unroll
    for (int q = 1; q < L::Q; ++q) {
      const int qf = MODE == GATHER_PULL ? q : opp(q), qw = MODE == GATHER_PULL ? opp(q) : q;
      const uint4 t = v[q - 1];
      int32_t e;
      bool wall;
      if (t.y == 0xffffffffu) {  // sentinel: more than three runs (or a third delta out of range)
        e = __ldg(nbr + (long long)(q - 1) * Ns + i);
        wall = e < 0;
      } else {  // one, two or three runs, all from the record: no dependent load
        uint32_t d = lane >= (t.y & 63u) ? t.w : t.z;
        if ((t.y & 0x40u) && lane >= ((t.y >> 7) & 31u)) d = t.w + (uint32_t)((int32_t)t.y >> 12);
        e = (int32_t)(d + (uint32_t)i);
        wall = (t.x & lane_bit) != 0u;
      }
      off[q - 1] = wall ? (IT)qw * n + self : (IT)qf * n + (IT)e;
    }
  }
  check_offsets<L, IT>(off, Ns);
}

// Make the compiler forget how a value was computed: the A-A odd kernel scatters to the
// offsets it gathered from, and without this ptxas keeps the 14 64-bit ADDRESSES alive across
// the collision (28 registers, spills) instead of the 14 32-bit offsets (one IMAD.WIDE each to
// rebuild).
__device__ __forceinline__ void opaque(uint32_t& v) { asm volatile("" : "+r"(v)); }
__device__ __forceinline__ void opaque(long long& v) { asm volatile("" : "+l"(v)); }
// The same for a pointer: loads through it are not merged with earlier loads of the same
// address (the rare paths of the step kernels read their populations AGAIN on purpose).
template <typename T>
__device__ __forceinline__ T* relaunder(T* p) {
  asm volatile("" : "+l"(p));
  return p;
}

// Address (element offset) where the pre-collision f_q(x) of link q lives.
template <int MODE>
__device__ __forceinline__ long long slot_of(int q, int32_t e, long long Ns, long long i) {
  if (MODE == GATHER_OWN) return (long long)q * Ns + i;
#ifdef HLB_BOUNDS_CHECK
  if (e >= Ns) __trap();
#endif
  const bool wall = e < 0;
  if (MODE == GATHER_PULL)  // post-collision buffer: wall -> own opposite slot
    return wall ? (long long)opp(q) * Ns + i : (long long)q * Ns + e;
  // GATHER_AA_ODD: slot opp(q) of the source site, slot q of the site itself at walls
  return wall ? (long long)q * Ns + i : (long long)opp(q) * Ns + e;
}

// The iolet index of a group of 32 sites (preprocess.h): {bits, rank}. Loaded at the very top
// of every step kernel -- ncu showed 12-24 % of a warp's lifetime spent waiting for this word
// when it was loaded where it is used, after the collision (profiles/r02_tuning.md section 1).
struct IoletIndex {
  const uint2* idx = nullptr;    // [Ns/32] {bits, rank}
  const uint4* links = nullptr;  // [iolet sites][iolet_row<L>() uint4]: byte p - 1 = k + 1 or 0
};
__device__ __forceinline__ uint2 load_iolet_word(const IoletIndex& io, long long i) {
  return __ldg(io.idx + (i >> 5));
}
__device__ __forceinline__ bool has_iolet_link(uint2 w) { return (w.x >> (threadIdx.x & 31)) & 1u; }
// row of this site in IoletIndex::links, -1 if it has no iolet link (one register instead of two)
__device__ __forceinline__ int iolet_row_of(uint2 w) {
  const unsigned lane = threadIdx.x & 31;
  return ((w.x >> lane) & 1u) ? (int)(w.y + __popc(w.x & ((1u << lane) - 1u))) : -1;
}
template <typename L>
__host__ __device__ constexpr int iolet_row() { return (L::Q - 1 + 15) / 16; }
// iolet id of link p (compile-time p after unrolling) in a row of link bytes; -1: not an iolet link
template <typename L>
__device__ __forceinline__ int iolet_of_link(const uint4 (&row)[iolet_row<L>()], int p) {
  const int b = p - 1;
  const uint4 v = row[b / 16];
  const int wi = (b % 16) / 4;
  const uint32_t word = wi == 0 ? v.x : (wi == 1 ? v.y : (wi == 2 ? v.z : v.w));
  return (int)((word >> (8 * (b % 4))) & 0xffu) - 1;
}

// Rare path (sites on an inlet/outlet cap): for every iolet link p of site i replace
// out[p] -- the value that will be read back as f_p(x, t+1), on entry the bounced h*_opp(p) --
//   constant-density iolet k: by the equilibrium f_eq_p(rho_k, u(x, t))           (reading A6)
//                             (u replaced by (u.n_k) n_k when a normal n_k is given)
//   velocity iolet k (Ladd):  by h*_opp(p) + 6 w_p rho(x, t) c_p.u_k             (reading R-ladd)
//                             (u_k scaled by the site's weight omega(x) when iolet_w is given,
//                              reading R-weights)
// Which links are iolet links comes from ONE row of link bytes per flagged site (one or two
// 128-bit loads), not from the neighbour table: the table version issued Q - 1 dependent loads
// one after the other and cost 6-9 % of all warp time although 3 % of the warps take it.
// Fully unrolled so that out[] stays in registers (no call, no stack).
// FULL = false is the lean instantiation for geometries whose iolets are all plain
// constant-density ones (every BASELINE config): inlined, the Ladd and normal branches make
// the compiler park values in local memory on the COMMON path (profiles/r01_tuning.md).
template <typename L, bool FULL>
__device__ __forceinline__ void iolet_substitute(const IoletIndex& io, int irow, long long i,
                                                 const Moments& m,
                                                 const double* __restrict__ iolet_par,
                                                 const double* __restrict__ iolet_w,
                                                 double (&out)[L::Q]) {
  uint4 row[iolet_row<L>()];
#pragma unroll
  for (int k = 0; k < iolet_row<L>(); ++k) row[k] = __ldg(io.links + (long long)irow * iolet_row<L>() + k);
#pragma unroll
  for (int p = 1; p < L::Q; ++p) {
    const int k = iolet_of_link<L>(row, p);
    if (k >= 0) {
      const double* par = iolet_par + 4 * k;
      const double rk = __ldg(par);
      if (!FULL) {
        out[p] = heq_of<L>(p, rk - 1.0, rk, m.ux, m.uy, m.uz);
      } else if (rk > 0.0) {
        // par[1..3]: unit normal of the iolet, (0,0,0) = none; with a normal the ghost only
        // carries the normal part (u.n) n of the site's velocity
        const double n0 = __ldg(par + 1), n1 = __ldg(par + 2), n2 = __ldg(par + 3);
        if (n0 != 0.0 || n1 != 0.0 || n2 != 0.0) {
          const double un = add(add(mul(m.ux, n0), mul(m.uy, n1)), mul(m.uz, n2));
          out[p] = heq_of<L>(p, rk - 1.0, rk, mul(un, n0), mul(un, n1), mul(un, n2));
        } else {
          out[p] = heq_of<L>(p, rk - 1.0, rk, m.ux, m.uy, m.uz);
        }
      } else {
        double cu = c_dot_u<L>(p, __ldg(par + 1), __ldg(par + 2), __ldg(par + 3));
        if (iolet_w) cu = mul(__ldg(iolet_w + i), cu);  // velocity profile across the cap
        out[p] = fma_(mul(6.0 * L::weight(p), m.rho), cu, out[p]);
      }
    }
  }
}

// Programmatic dependent launch (sm_90+): a step kernel lets the next step's grid start as
// soon as all of its own blocks have started (launch_dependents), and the next grid waits for
// the full completion and memory flush of this one (wait) only right before it touches
// populations. What precedes the wait -- thread setup and the link-record loads, which no
// step kernel writes -- overlaps the tail of the previous step. Without the launch attribute
// (HLB_NO_PDL, read-out kernels) both instructions are no-ops.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait_for_previous_step() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// L2 prefetch of data that a block scheduled roughly one wave later will load: brings the
// DRAM fetch forward without holding registers or a scoreboard slot.
__device__ __forceinline__ void prefetch_l2(const void* p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
// The gather kernels' prefetches: a warp's 32 addresses of one link cover two to four 128-byte
// lines (one or two runs of consecutive sites), so only the lanes at which a line or a run can
// begin need to ask. HLB_PF_LANES: 0 = every lane (round 1), 1 = lanes 0, 15, 16, 31 (8-byte
// populations: line starts and ends of an aligned run, and both ends of the warp).
// Table links (REC = false: Morton / tiled orders) gather anywhere: every lane asks.
#ifndef HLB_PF_LANES
#define HLB_PF_LANES 1   // +0.5 % on the two-lattice kernel, neutral elsewhere (profiles/r02_tuning.md section 11)
#endif
template <bool REC>
__device__ __forceinline__ bool prefetch_lane() {
  if (!REC || !HLB_PF_LANES) return true;
  const unsigned l = threadIdx.x & 15u;
  return l == 0u || l == 15u;
}

// The even A-A kernel reads Q planes at the block's own 128 sites: the block pf sites ahead
// will read Q x (128 sizeof(ST) / 128) lines, one per thread -- one prefetch instruction per
// warp instead of Q per thread (and none of their 64-bit address arithmetic).
template <typename L, typename ST>
__device__ __forceinline__ void prefetch_block_planes(const ST* a, long long Ns, long long pf) {
  constexpr int LPP = SBLOCK * (int)sizeof(ST) / 128;  // lines per plane per block
  const ST* first = a + (long long)blockIdx.x * SBLOCK + pf;
  for (int l = threadIdx.x; l < L::Q * LPP; l += SBLOCK)
    prefetch_l2((const char*)(first + (long long)(l / LPP) * Ns) + (l % LPP) * 128);
}

// BFL interpolated walls inside the step kernels (V == 2 instantiations; BflFused in
// kernels.cuh). With i = opp(p) the direction from x to the wall and y = x + c_p behind x:
//   d <  1/2:  f_p(x,t+1) = 2d f*_i(x,t) + (1 - 2d) f*_i(y,t).  After the gather of step t+1,
//              h[p] is the bounced f*_i(x,t) and h[opp(p)] is f*_i(y,t), streamed from y: the
//              rule is applied to the gathered registers.
//   d >= 1/2:  f_p(x,t+1) = f*_i(x,t) / (2d) + (1 - 1/(2d)) f*_p(x,t).  Both are this site's
//              own post-collision values of step t: the rule is applied to the value the site
//              writes back for link p.
// Neither needs a memory access beyond the coefficients. Two links p and opp(p) of one site
// are never both interpolated (that needs x + c_p solid and fluid), so updating in place is safe.
// Both rules mix the two members of ONE opposite pair (p, opp(p)) only, and the two links of a
// pair are never both interpolated (an interpolated link needs the site behind x to be fluid,
// include/hlb.h), so a site's coefficients are one double per PAIR plus a word that says which
// member is the link: BflFused in kernels.cuh. And so the rule for the written value fits into
// the store-as-you-go shape of the common path: the pair-symmetric collision hands over both
// post-collision values of a pair at once (collide_emit_pairs), the rule is applied to them
// (branch-free: a coefficient of 0 selects the plain value) and both are stored. Every thread
// that is not a cap site takes that path; the long path is for cap sites alone, as without
// interpolated walls. (Round 2 first sent every warp with a flagged lane down a long path
// that stored nothing early: 17-19 % below the plain kernels; profiles/r02_tuning.md 12, 15.)
__device__ __forceinline__ uint2 load_bfl_word(const BflFused& bf, long long i) { return __ldg(bf.idx + (i >> 5)); }
// warp-uniform: does any site of this group of 32 carry an interpolated link? A warp without
// one runs the plain common path (a third of the warps when every wall link is interpolated).
__device__ __forceinline__ bool bfl_warp(uint2 w) {
  return w.x != 0u;
}
__device__ __forceinline__ long long bfl_index_of(uint2 w) {
  const unsigned lane = threadIdx.x & 31;
  if (!((w.x >> lane) & 1u)) return -1;
  return (long long)w.y + __popc(w.x & ((1u << lane) - 1u));
}
// (-DHLB_BOUNDS_CHECK: the row index must lie inside the nf rows of the table)
__device__ __forceinline__ long long bfl_index_of(const BflFused& bf, uint2 w) {
  const long long idx = bfl_index_of(w);
#ifdef HLB_BOUNDS_CHECK
  if (idx >= bf.nf) __trap();
#else
  (void)bf;
#endif
  return idx;
}
// A site's row: P = (Q-1)/2 coefficients, then the member word (bit k set: the interpolated
// link of pair k is 2k + 2, else 2k + 1), padded to an even count: 64 B for D3Q15, 80 B for
// D3Q19, 16-byte aligned.
template <typename L>
__host__ __device__ constexpr int bfl_row() { return ((L::Q - 1) / 2 + 2) / 2 * 2; }
// The coefficients are static: fetch them towards the SM before the populations are waited
// for, so that the dependent chain bits -> rank -> coef does not add a DRAM round trip.
template <typename L>
__device__ __forceinline__ void bfl_prefetch(const BflFused& bf, long long idx) {
  const char* row = (const char*)(bf.coef + idx * bfl_row<L>());
  asm volatile("prefetch.global.L1 [%0];" ::"l"(row));
  if ((bfl_row<L>() * 8) % 128 != 0) asm volatile("prefetch.global.L1 [%0];" ::"l"(row + bfl_row<L>() * 8 - 16));
}
// Interpolation a x + (1 - a) y in the form x + b (y - x), b = 1 - a computed once on the host:
// two operations with no data-dependent control flow, b = 0 (no interpolated link in this pair,
// or the wall exactly half a link away, d = 1/2) returns x exactly -- so plain links need no
// select, and BFL with d = 1/2 IS halfway bounce-back bit for bit. The stored coefficient is
// +b for a d < 1/2 link (b = 1 - 2d), -b for a d >= 1/2 link (b = 1 - 1/(2d)).
// d < 1/2, on the gathered values: h[p] += b (h[opp(p)] - h[p])
template <typename L>
__device__ __forceinline__ void bfl_gather(const BflFused& bf, long long idx, double (&h)[L::Q]) {
  constexpr int P = (L::Q - 1) / 2, R = bfl_row<L>();
  const double* row = bf.coef + idx * R;
  const unsigned member = (unsigned)__double_as_longlong(__ldg(row + P));
#pragma unroll
  for (int k = 0; k < P; k += 2) {  // two pairs per 16-byte load
    const double2 v = __ldg((const double2*)row + k / 2);
#pragma unroll
    for (int j = k; j < k + 2 && j < P; ++j) {
      const int a = 2 * j + 1, b = a + 1;
      const bool s = (member >> j) & 1u;
      const double cj = j == k ? v.x : v.y;
      const double cp = cj > 0.0 ? cj : 0.0;
      const double D = sub(h[a], h[b]);
      h[a] = fma_(s ? 0.0 : -cp, D, h[a]);
      h[b] = fma_(s ? cp : 0.0, D, h[b]);
    }
  }
}
// d >= 1/2 (coefficient < 0), on the values a site writes back: out[p], the value written for
// link p, is the bounced h*_opp(p) without interpolation, h*_opp(p) + b (h*_p - h*_opp(p)) with
// it. BflWrite: what a thread needs for that, read before the collision; the coefficients
// themselves are read pair by pair (L1 hits after bfl_gather / the prefetch), not kept in
// 14-18 registers.
struct BflWrite {
  const double* row;  // NULL: no interpolated link at this site
  unsigned member;
};
template <typename L>
__device__ __forceinline__ BflWrite bfl_write_begin(const BflFused& bf, long long idx) {
  BflWrite w;
  w.row = nullptr;
  w.member = 0u;
  if (idx >= 0) {
    w.row = bf.coef + idx * bfl_row<L>();
    asm volatile("" : "+l"(w.row));  // read again below, do not keep bfl_gather's copies alive
    w.member = (unsigned)__double_as_longlong(__ldg(w.row + (L::Q - 1) / 2));
  }
  return w;
}
// pair (a, a + 1) with post-collision values va, vb: oa = out[a], ob = out[a + 1]
__device__ __forceinline__ void bfl_pair(const BflWrite& w, int a, double va, double vb, double& oa, double& ob) {
  const int k = (a - 1) / 2;
  double c = 0.0;
  if (w.row) c = __ldg(w.row + k);
  const bool s = (w.member >> k) & 1u;
  const double cn = c < 0.0 ? c : 0.0;  // -b
  const double D = sub(va, vb);
  oa = fma_(s ? 0.0 : -cn, D, vb);
  ob = fma_(s ? cn : 0.0, D, va);
}
// the same on whole arrays, for the cap-site path. h: post-collision; out[p] as above
template <typename L>
__device__ __forceinline__ void bfl_write(const BflFused& bf, long long idx, const double (&h)[L::Q],
                                          double (&out)[L::Q]) {
  const BflWrite w = bfl_write_begin<L>(bf, idx);
#pragma unroll
  for (int a = 1; a < L::Q; a += 2) bfl_pair(w, a, h[a], h[a + 1], out[a], out[a + 1]);
}
// two-lattice: the value written back for link p is slot opp(p) of the site
template <typename L>
__device__ __forceinline__ void bfl_write_pull(const BflFused& bf, long long idx, double (&h)[L::Q]) {
  const BflWrite w = bfl_write_begin<L>(bf, idx);
#pragma unroll
  for (int a = 1; a < L::Q; a += 2) {
    double oa, ob;
    bfl_pair(w, a, h[a], h[a + 1], oa, ob);
    h[a + 1] = oa;
    h[a] = ob;
  }
}

// BFL interpolated walls (linear Bouzidi-Firdaouss-Lallemand rule; the paper's "BFL" wall
// option, ref [16]) as a PRE-PASS over a list of interpolated links,
// run on the state buffer before a READ-OUT that gathers from it (the step kernels apply the
// rules themselves, see above; the API passes the d < 1/2 links only, the d >= 1/2 rule being
// already in what the step kernels wrote -- the kernel handles both). Written out for the
// two-lattice scheme: slot opp(p) of site x holds f*_opp(p)(x, t-1) and is read by nobody but
// x itself, as the halfway bounce-back value of its wall link p; the pre-pass replaces it by
//   d <  1/2:  2d f*_opp(p)(x) + (1 - 2d) f*_opp(p)(x + c_p)      (slot opp(p) of the site behind)
//   d >= 1/2:  f*_opp(p)(x) / (2d) + (1 - 1/(2d)) f*_p(x)         (slot p of x itself)
// (evaluated as x + (1 - a) (y - x), like the step kernels)
// The sources are slots that no link of the list writes (a link is in the list only if the
// site behind it is fluid), so the pass has no ordering hazards. As the way to apply BFL on
// every step it cost 23-25 % of configs[3] against 12-18 % in registers (profiles/r01_tuning.md
// section 11).
// Where the three values live depends on what the state buffer holds (GatherMode of the state):
//   GATHER_PULL   (two-lattice, post-collision f*_r(z) in slot r of z):
//       target f*_i(x): slot i of x;  f*_i(y): slot i of y;  f*_q(x): slot q of x
//   GATHER_AA_ODD (A-A after the even kernel, f*_r(z) in slot opp(r) of z):
//       target: slot q of x;          f*_i(y): slot q of y;  f*_q(x): slot i of x
//   GATHER_OWN    (A-A after the odd kernel, f*_r(z) in slot r of z + c_r, bounced walls in
//                  slot opp(r) of z):
//       target: slot q of x;          f*_i(y): slot i of x (= y + c_i);  f*_q(x): slot q of y
// In every case the target is the slot the step kernel reads as the bounced f_q(x, t+1), no
// other link reads or writes it, and neither source is the target of another link (that
// would need y or x to be solid).
// Each thread takes BFL_UNROLL links (a block: BFL_UNROLL * BLOCK consecutive ones): the
// link data (static) are fetched before the wait on the previous step, then all population
// loads are in flight together -- the pass is latency-bound, not bandwidth-bound.
constexpr int BFL_UNROLL = 4;
template <typename ST>
__global__ void __launch_bounds__(BLOCK)
k_bfl_prepass(ST* __restrict__ buf, long long Ns, const int32_t* __restrict__ site,
              const int32_t* __restrict__ behind, const uint8_t* __restrict__ link,
              const double* __restrict__ dist, long long n, int mode) {
  const long long l0 = (long long)blockIdx.x * (BFL_UNROLL * BLOCK) + threadIdx.x;
  long long tgt[BFL_UNROLL], src[BFL_UNROLL];
  double dd[BFL_UNROLL];
  pdl_launch_dependents();
#pragma unroll
  for (int k = 0; k < BFL_UNROLL; ++k) {
    const long long l = l0 + (long long)k * BLOCK;
    dd[k] = -1.0;
    if (l < n) {
      const long long i = __ldg(site + l), y = __ldg(behind + l);
      const int p = __ldg(link + l), po = opp(p);
      dd[k] = __ldg(dist + l);
      tgt[k] = (long long)(mode == GATHER_PULL ? po : p) * Ns + i;
      if (dd[k] < 0.5)
        src[k] = mode == GATHER_PULL ? (long long)po * Ns + y
               : mode == GATHER_AA_ODD ? (long long)p * Ns + y : (long long)po * Ns + i;
      else
        src[k] = mode == GATHER_PULL ? (long long)p * Ns + i
               : mode == GATHER_AA_ODD ? (long long)po * Ns + i : (long long)p * Ns + y;
    }
  }
  pdl_wait_for_previous_step();
  double a[BFL_UNROLL], b[BFL_UNROLL];
#pragma unroll
  for (int k = 0; k < BFL_UNROLL; ++k)
    if (dd[k] > 0.0) {
      a[k] = to_real(buf[tgt[k]]);
      b[k] = to_real(buf[src[k]]);
    }
#pragma unroll
  for (int k = 0; k < BFL_UNROLL; ++k)
    if (dd[k] > 0.0) {
      // the step kernels' form and operation order (bitwise the same: a read-out between two
      // steps does not change an fp64 run): x + (1 - a) (y - x), 1 - a as the host computes it
      const double two_d = mul(2.0, dd[k]);
      const double w = dd[k] < 0.5 ? sub(1.0, two_d) : sub(1.0, __ddiv_rn(1.0, two_d));
      buf[tgt[k]] = to_store<ST>(fma_(w, sub(b[k], a[k]), a[k]));
    }
}

// ------------------------------------------------------------------ two-lattice pull
// src holds post-collision values h*(., t-1) (iolet slots substituted); one launch does
// gather -> moments -> BGK -> store of h*(., t) into dst (rows S1..S6 fused).
// pf > 0: also L2-prefetch what site i + pf will gather; to first order its links are those
// of site i shifted by pf (x-fastest order). The population buffers carry pf elements of
// padding, so only the one warp-uniform test is needed.
// Shape shared by the three step kernels. Common path (no iolet link at this site, no
// interpolated walls): gather, moments, and every post-collision value stored the moment it
// is known. Rare path (2-3 % of the warps): the populations are READ AGAIN (L1 / L2 hits) and
// the moments recomputed, so that nothing has to be kept for it across the common path -- the
// compiler otherwise parks copies of the gathered values in local memory on every thread
// (profiles/r02_tuning.md). Safe in the in-place kernels too: a site's read set is its own
// write set, so nobody else has written these slots, and this thread has not stored yet.
template <typename L, typename ST, bool REC, typename IT, int V>
__global__ void __launch_bounds__(SBLOCK, pull_minb<L, REC>() - pull_f64_drop<L, ST, REC>() + bfl_pull_add<L, ST, IT, V>())
k_pull(const ST* __restrict__ src, ST* __restrict__ dst, const int32_t* __restrict__ nbr,
       const uint4* __restrict__ rec, IoletIndex io, const double* __restrict__ iolet_par,
       long long Ns, Relax rx, Planes pl, long long pf, BflFused bf) {
  const long long i = (long long)blockIdx.x * SBLOCK + threadIdx.x;
  double h[L::Q];
  long long bidx = -1;
  pdl_launch_dependents();
  const bool ahead_ok = pf > 0 && i + pf < Ns;  // warp-uniform (pf, Ns: multiples of 128)
  const uint2 iow = load_iolet_word(io, i);
  uint2 bw = make_uint2(0u, 0u);
  if (V == 2) bw = load_bfl_word(bf, i);  // in flight together with the link records
  {
    IT off[L::Q - 1];
    link_offsets<L, GATHER_PULL, REC, IT>(nbr, rec, Ns, i, pl, off);
    if (V == 2) {  // the row request goes out before the gathers and travels with them
      bidx = bfl_index_of(bf, bw);
      if (bidx >= 0) bfl_prefetch<L>(bf, bidx);
    }
    pdl_wait_for_previous_step();
    h[0] = to_real(src[i]);
#pragma unroll
    for (int q = 1; q < L::Q; ++q) h[q] = to_real(src[off[q - 1]]);
    if (ahead_ok) {  // every thread prefetches its own gathers shifted by pf (exact inside a run)
      const ST* ahead = src + pf;
      asm volatile("" : "+l"(ahead));  // keep base + offset * size: one IMAD.WIDE per prefetch
      if (REC && (threadIdx.x & 31) < ((L::Q - 1) * 16 + 31) / 32)
        prefetch_l2((const char*)(rec + ((i + pf) >> 5) * (L::Q - 1)) + 32 * (threadIdx.x & 31));
      if (prefetch_lane<REC>()) {
        prefetch_l2(ahead + i);
#pragma unroll
        for (int q = 1; q < L::Q; ++q) prefetch_l2(ahead + off[q - 1]);
      }
    }
  }
  const int irow = iolet_row_of(iow);
  if (V == 2 && bidx >= 0 && bf.gather) bfl_gather<L>(bf, bidx, h);
  const Moments m = moments_of<L>(h);
  ST* d = dst + i;
  // (no second gather here, unlike the A-A kernels: the offsets are dead by now, and keeping
  // the gathered values for the rare path costs this kernel nothing measurable)
  if (irow < 0) {  // common path: every value is stored as soon as it is known
    if (V == 2 && bfl_warp(bw)) {  // slot opp(p) holds what link p reads next step
      const BflWrite w = bfl_write_begin<L>(bf, bidx);
      collide_emit_pairs<L, sizeof(ST) == 4>(h, m, rx, [&](double v) { d[0] = to_store<ST>(v); },
        [&](int a, double va, double vb) {
          double oa, ob;
          bfl_pair(w, a, va, vb, oa, ob);
          d[(long long)a * Ns] = to_store<ST>(ob);
          d[(long long)(a + 1) * Ns] = to_store<ST>(oa);
        });
    } else {
      collide_emit<L, sizeof(ST) == 4>(h, m, rx, [&](int q, double v) { d[(long long)q * Ns] = to_store<ST>(v); });
    }
    return;
  }
  collide<L, sizeof(ST) == 4>(h, m, rx, h);
  if (V == 2 && bidx >= 0) bfl_write_pull<L>(bf, bidx, h);
  if (irow >= 0) {  // sites on an inlet/outlet cap
    // slot opp(p) of this site is read back by link p next step
    double back[L::Q];
#pragma unroll
    for (int p = 1; p < L::Q; ++p) back[p] = h[opp(p)];
    iolet_substitute<L, (V >= 1)>(io, irow, i, m, iolet_par, bf.iolet_w, back);
#pragma unroll
    for (int p = 1; p < L::Q; ++p) h[opp(p)] = back[p];
  }
#pragma unroll
  for (int q = 0; q < L::Q; ++q) d[(long long)q * Ns] = to_store<ST>(h[q]);
}

// ------------------------------------------------------------------ A-A in place
// Even phase: read slot q of the site, write h*_q to slot opp(q) of the site (no table).
// Odd phase: read f_q from slot opp(q) of x - c_q (slot q of x at a wall), write h*_q to
// the address f_opp(q) was read from. Read set = write set per site in both phases, so one
// array and no inter-thread hazards (tests/test_aa_model.py).
template <typename L, typename ST, int V>
__global__ void __launch_bounds__(SBLOCK, aa_even_minb<L, ST>())
k_aa_even(ST* __restrict__ a, IoletIndex io, const double* __restrict__ iolet_par,
          long long Ns, Relax rx, long long pf, BflFused bf) {
  const long long i = (long long)blockIdx.x * SBLOCK + threadIdx.x;
  ST* p0 = a + i;
  double h[L::Q];
  long long bidx = -1;
  pdl_launch_dependents();
  const uint2 iow = load_iolet_word(io, i);
  uint2 bw = make_uint2(0u, 0u);
  if (V == 2) bw = load_bfl_word(bf, i);
  pdl_wait_for_previous_step();
#pragma unroll
  for (int q = 0; q < L::Q; ++q) h[q] = to_real(p0[(long long)q * Ns]);
  if (V == 2) {  // after the population loads are issued: waiting for the word must not delay them
    bidx = bfl_index_of(bf, bw);
    if (bidx >= 0) bfl_prefetch<L>(bf, bidx);
  }
  if (pf > 0 && i + pf < Ns) prefetch_block_planes<L, ST>(a, Ns, pf);  // block-uniform test
  opaque(Ns);  // the stores rebuild their addresses (else 15 address pairs stay live: spills)
  const int irow = iolet_row_of(iow);
  if (irow < 0) {  // common path: h*_q goes to slot opp(q) as soon as it is known
    if (V == 2 && bidx >= 0 && bf.gather) bfl_gather<L>(bf, bidx, h);
    const Moments m = moments_of<L>(h);
    if (V == 2 && bfl_warp(bw)) {
      const BflWrite w = bfl_write_begin<L>(bf, bidx);
      collide_emit_pairs<L, sizeof(ST) == 4>(h, m, rx, [&](double v) { p0[0] = to_store<ST>(v); },
        [&](int a, double va, double vb) {
          double oa, ob;
          bfl_pair(w, a, va, vb, oa, ob);
          p0[(long long)a * Ns] = to_store<ST>(oa);
          p0[(long long)(a + 1) * Ns] = to_store<ST>(ob);
        });
    } else {
      collide_emit<L, sizeof(ST) == 4>(h, m, rx, [&](int q, double v) { p0[(long long)opp(q) * Ns] = to_store<ST>(v); });
    }
    return;
  }
  {  // rare path (cap sites): read again
    const ST* again = relaunder(p0);
#pragma unroll
    for (int q = 0; q < L::Q; ++q) h[q] = to_real(again[(long long)q * Ns]);
  }
  if (V == 2 && bidx >= 0 && bf.gather) bfl_gather<L>(bf, bidx, h);
  const Moments m = moments_of<L>(h);
  collide<L, sizeof(ST) == 4>(h, m, rx, h);
  double out[L::Q];  // out[p] is written where f_p was read: the bounced h*_opp(p)
#pragma unroll
  for (int p = 0; p < L::Q; ++p) out[p] = h[opp(p)];
  if (V == 2 && bidx >= 0) bfl_write<L>(bf, bidx, h, out);
  if (irow >= 0) iolet_substitute<L, (V >= 1)>(io, irow, i, m, iolet_par, bf.iolet_w, out);
#pragma unroll
  for (int p = 0; p < L::Q; ++p) p0[(long long)p * Ns] = to_store<ST>(out[p]);
}

// The cap-site path of k_aa_odd for the instantiations with the full iolet rules (V >= 1), as a
// function of its own that starts from the site index again (decode, read, update, scatter).
// Inlined, its register needs made ptxas spill 7 of the 14 offsets where they are DEFINED -- in
// the decode every thread runs: 7 STL + 14 LDL per thread on the common path of the V = 1 kernel
// (ncu, profiles/r02_ncu_bfl_readout.md). A call keeps the two allocations apart; nothing is
// live across it. Used where it was measured to pay: V = 1, D3Q15 (configs[4] with a velocity
// inlet: odd kernel 1.525 -> 1.515 ms in fp64, 0.926 -> 0.907 with 4-byte storage; configs[3]
// unchanged). With interpolated walls (V = 2) and on D3Q19 the inlined form is 1-2 % faster.
template <typename L, typename ST, bool REC, typename IT, int V>
__device__ __noinline__ void aa_odd_cap_site(ST* __restrict__ a, const int32_t* __restrict__ nbr,
                                             const uint4* __restrict__ rec, IoletIndex io,
                                             int irow, const double* __restrict__ iolet_par, long long Ns,
                                             Relax rx, Planes pl, BflFused bf,  // by value: copied at the call, not in the kernel's prologue
                                             long long bidx, long long i) {
  IT off[L::Q - 1];
  link_offsets<L, GATHER_AA_ODD, REC, IT, false>(nbr, rec, Ns, i, pl, off);
  double h[L::Q];
  h[0] = to_real(a[i]);
#pragma unroll
  for (int q = 1; q < L::Q; ++q) h[q] = to_real(a[off[q - 1]]);
  if (V == 2 && bidx >= 0 && bf.gather) bfl_gather<L>(bf, bidx, h);
  const Moments m = moments_of<L>(h);
  collide<L, sizeof(ST) == 4>(h, m, rx, h);
  double out[L::Q];
#pragma unroll
  for (int p = 0; p < L::Q; ++p) out[p] = h[opp(p)];
  if (V == 2 && bidx >= 0) bfl_write<L>(bf, bidx, h, out);
  iolet_substitute<L, (V >= 1)>(io, irow, i, m, iolet_par, bf.iolet_w, out);
  a[i] = to_store<ST>(out[0]);
#pragma unroll
  for (int p = 1; p < L::Q; ++p) a[off[p - 1]] = to_store<ST>(out[p]);
}

template <typename L, typename ST, bool REC, typename IT, int V>
__global__ void __launch_bounds__(SBLOCK, aa_odd_minb<L, REC>() + odd_smem_minb_add<L, ST, REC, IT, V>())
k_aa_odd(ST* __restrict__ a, const int32_t* __restrict__ nbr, const uint4* __restrict__ rec,
         IoletIndex io, const double* __restrict__ iolet_par,
         long long Ns, Relax rx, Planes pl, long long pf, BflFused bf) {
  const long long i = (long long)blockIdx.x * SBLOCK + threadIdx.x;
  IT off[L::Q - 1];
  long long bidx = -1;
  pdl_launch_dependents();
  uint2 bw = make_uint2(0u, 0u);
  if (V == 2) bw = load_bfl_word(bf, i);  // in flight together with the link records
  const bool ahead_ok = pf > 0 && i + pf < Ns;  // warp-uniform (pf, Ns: multiples of 128)
  constexpr bool REC_SMEM = sizeof(ST) == 4 && REC;  // = odd_rec_smem<ST, REC>()
  link_offsets<L, GATHER_AA_ODD, REC, IT, REC_SMEM>(nbr, rec, Ns, i, pl, off);
  if (V == 2) {  // the row request goes out before the gathers and travels with them
    bidx = bfl_index_of(bf, bw);
    if (bidx >= 0) bfl_prefetch<L>(bf, bidx);
  }
  const uint2 iow = load_iolet_word(io, i);  // (not before the decode: its registers are the scarce ones)
  pdl_wait_for_previous_step();
  double h[L::Q];
  h[0] = to_real(a[i]);
#pragma unroll
  for (int q = 1; q < L::Q; ++q) h[q] = to_real(a[off[q - 1]]);
  if (ahead_ok) {  // every thread prefetches its own gathers shifted by pf (exact inside a run)
    const ST* ahead = a + pf;
    asm volatile("" : "+l"(ahead));  // keep base + offset * size: one IMAD.WIDE per prefetch
    if (REC && (threadIdx.x & 31) < ((L::Q - 1) * 16 + 31) / 32)
      prefetch_l2((const char*)(rec + ((i + pf) >> 5) * (L::Q - 1)) + 32 * (threadIdx.x & 31));
    if (prefetch_lane<REC>()) {
      prefetch_l2(ahead + i);
#pragma unroll
      for (int q = 1; q < L::Q; ++q) prefetch_l2(ahead + off[q - 1]);
    }
  }
#pragma unroll
  for (int q = 1; q < L::Q; ++q) opaque(off[q - 1]);
  const int irow = iolet_row_of(iow);
  if (irow < 0) {  // common path: h*_q goes where f_opp(q) was read, as soon as it is known
    if (V == 2 && bidx >= 0 && bf.gather) bfl_gather<L>(bf, bidx, h);
    const Moments m = moments_of<L>(h);
    if (V == 2 && bfl_warp(bw)) {
      const BflWrite w = bfl_write_begin<L>(bf, bidx);
      collide_emit_pairs<L, sizeof(ST) == 4>(h, m, rx, [&](double v) { a[i] = to_store<ST>(v); },
        [&](int p, double va, double vb) {
          double oa, ob;
          bfl_pair(w, p, va, vb, oa, ob);
          a[off[p - 1]] = to_store<ST>(oa);
          a[off[p]] = to_store<ST>(ob);
        });
    } else {
      collide_emit<L, sizeof(ST) == 4>(h, m, rx, [&](int q, double v) {
        if (q == 0) a[i] = to_store<ST>(v);
        else a[off[opp(q) - 1]] = to_store<ST>(v);
      });
    }
    return;
  }
  if (V == 1 && L::Q == 15) {  // cap sites, full iolet rules: a call (see aa_odd_cap_site)
    aa_odd_cap_site<L, ST, REC, IT, V>(a, nbr, rec, io, irow, iolet_par, Ns, rx, pl, bf, bidx, i);
    return;
  }
  {  // rare path (cap sites): read again
    const ST* again = relaunder(a);
    h[0] = to_real(again[i]);
#pragma unroll
    for (int q = 1; q < L::Q; ++q) h[q] = to_real(again[off[q - 1]]);
  }
  if (V == 2 && bidx >= 0 && bf.gather) bfl_gather<L>(bf, bidx, h);
  const Moments m = moments_of<L>(h);
  collide<L, sizeof(ST) == 4>(h, m, rx, h);
  double out[L::Q];
#pragma unroll
  for (int p = 0; p < L::Q; ++p) out[p] = h[opp(p)];
  if (V == 2 && bidx >= 0) bfl_write<L>(bf, bidx, h, out);
  if (irow >= 0) iolet_substitute<L, (V >= 1)>(io, irow, i, m, iolet_par, bf.iolet_w, out);
  a[i] = to_store<ST>(out[0]);
#pragma unroll
  for (int p = 1; p < L::Q; ++p) a[off[p - 1]] = to_store<ST>(out[p]);
}

// ------------------------------------------------------------------ resident multi-step kernels
// Small geometries (every block of the grid resident on the chip at once; BASELINE configs[0]
// is 99 blocks) are bound by the launch-to-launch gap, not by memory: one cooperative launch
// runs n time steps, a thread keeping its site and its decoded link offsets in registers for
// the whole run, with a grid-wide barrier between steps in place of the kernel boundary. The
// per-site arithmetic is the same device code as in the one-shot kernels (bitwise identical
// results). Populations written by other SMs are read with ld.global.cg (L2; never a stale L1
// line). The barrier is a monotone arrival counter in global memory: after step s every block
// adds 1 and waits until the counter reaches base + (s + 1) * gridDim.x (the host advances
// base by (n - 1) * gridDim.x per launch; 64 bits never wrap).
__device__ __forceinline__ void grid_barrier(unsigned long long* bar, unsigned long long target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    // release: this block's stores (ordered before by the bar.sync) are visible before the
    // arrival; a reduction, so nothing waits for the old value to come back
    asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(bar) : "memory");
    unsigned long long v;
    do {
      asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(bar) : "memory");
    } while (v < target);
  }
  __syncthreads();
}
template <typename ST>
__device__ __forceinline__ double load_l2(const ST* p) { return to_real(__ldcg(p)); }
// Occupancy does not matter here (the grid is at most one block per slot and the run is
// latency-bound): 4 blocks per SM leave 128 registers, enough to keep the link offsets, the
// populations and the loop state without spills. (A second instantiation for 6 blocks per SM,
// 80 registers with spills, gained 3-9 % at 96 k sites and lost 10-14 % at 112 k against the
// one-shot kernels; so did a looping form for L2-sized geometries: profiles/r01_tuning.md
// section 14.)
constexpr int RESIDENT_MINB = 4;

// One site update of the resident kernels (the bodies of k_aa_even / k_aa_odd and k_pull).
template <typename L, typename ST, typename IT, int V>
__device__ __forceinline__ void aa_site(ST* a, const IoletIndex& io, int irow,
                                        const double* __restrict__ iolet_par,
                                        const double* __restrict__ iolet_w, long long Ns,
                                        const Relax& rx, long long i, const IT (&off)[L::Q - 1],
                                        bool iolet, bool odd) {
  double h[L::Q];
  h[0] = load_l2(a + i);
  if (odd) {
#pragma unroll
    for (int q = 1; q < L::Q; ++q) h[q] = load_l2(a + off[q - 1]);
  } else {
#pragma unroll
    for (int q = 1; q < L::Q; ++q) h[q] = load_l2(a + (long long)q * Ns + i);
  }
  const Moments m = moments_of<L>(h);
  collide<L, sizeof(ST) == 4>(h, m, rx, h);
  double out[L::Q];
#pragma unroll
  for (int p = 0; p < L::Q; ++p) out[p] = h[opp(p)];
  if (iolet) iolet_substitute<L, (V >= 1)>(io, irow, i, m, iolet_par, iolet_w, out);
  a[i] = to_store<ST>(out[0]);
  if (odd) {
#pragma unroll
    for (int p = 1; p < L::Q; ++p) a[off[p - 1]] = to_store<ST>(out[p]);
  } else {
#pragma unroll
    for (int p = 1; p < L::Q; ++p) a[(long long)p * Ns + i] = to_store<ST>(out[p]);
  }
}
template <typename L, typename ST, typename IT, int V>
__device__ __forceinline__ void pull_site(const ST* src, ST* dst, const IoletIndex& io, int irow,
                                          const double* __restrict__ iolet_par,
                                          const double* __restrict__ iolet_w, long long Ns,
                                          const Relax& rx, long long i, const IT (&off)[L::Q - 1],
                                          bool iolet) {
  double h[L::Q];
  h[0] = load_l2(src + i);
#pragma unroll
  for (int q = 1; q < L::Q; ++q) h[q] = load_l2(src + off[q - 1]);
  const Moments m = moments_of<L>(h);
  collide<L, sizeof(ST) == 4>(h, m, rx, h);
  if (iolet) {
    double back[L::Q];
#pragma unroll
    for (int p = 1; p < L::Q; ++p) back[p] = h[opp(p)];
    iolet_substitute<L, (V >= 1)>(io, irow, i, m, iolet_par, iolet_w, back);
#pragma unroll
    for (int p = 1; p < L::Q; ++p) h[opp(p)] = back[p];
  }
#pragma unroll
  for (int q = 0; q < L::Q; ++q) dst[(long long)q * Ns + i] = to_store<ST>(h[q]);
}

template <typename L, typename ST, bool REC, typename IT, int V>
__global__ void __launch_bounds__(SBLOCK, RESIDENT_MINB)
k_aa_resident(ST* a, const int32_t* __restrict__ nbr, const uint4* __restrict__ rec,
              IoletIndex io, const double* __restrict__ iolet_par,
              const double* __restrict__ iolet_w, long long Ns, Relax rx, Planes pl, long long n_steps, int odd0, unsigned long long* bar,
              unsigned long long bar_base) {
  const long long i = (long long)blockIdx.x * SBLOCK + threadIdx.x;
  IT off[L::Q - 1];
  const int irow = iolet_row_of(load_iolet_word(io, i));
  link_offsets<L, GATHER_AA_ODD, REC, IT>(nbr, rec, Ns, i, pl, off);
  const bool iolet = irow >= 0;
  bool odd = odd0 != 0;
  for (long long s = 0; s < n_steps; ++s) {
    aa_site<L, ST, IT, V>(a, io, irow, iolet_par, iolet_w, Ns, rx, i, off, iolet, odd);
    odd = !odd;
    if (s + 1 < n_steps) grid_barrier(bar, bar_base + (unsigned long long)(s + 1) * gridDim.x);
  }
}

template <typename L, typename ST, bool REC, typename IT, int V>
__global__ void __launch_bounds__(SBLOCK, RESIDENT_MINB)
k_pull_resident(ST* b0, ST* b1, const int32_t* __restrict__ nbr, const uint4* __restrict__ rec,
                IoletIndex io, const double* __restrict__ iolet_par,
                const double* __restrict__ iolet_w, long long Ns, Relax rx, Planes pl, long long n_steps, unsigned long long* bar,
                unsigned long long bar_base) {
  const long long i = (long long)blockIdx.x * SBLOCK + threadIdx.x;
  IT off[L::Q - 1];
  const int irow = iolet_row_of(load_iolet_word(io, i));
  link_offsets<L, GATHER_PULL, REC, IT>(nbr, rec, Ns, i, pl, off);
  const bool iolet = irow >= 0;
  const ST* src = b0;
  ST* dst = b1;
  for (long long s = 0; s < n_steps; ++s) {
    pull_site<L, ST, IT, V>(src, dst, io, irow, iolet_par, iolet_w, Ns, rx, i, off, iolet);
    ST* t = const_cast<ST*>(src);
    src = dst;
    dst = t;
    if (s + 1 < n_steps) grid_barrier(bar, bar_base + (unsigned long long)(s + 1) * gridDim.x);
  }
}

// ------------------------------------------------------------------ read-out / init
// REC: the sources come from the 16-byte link records (7 B per site) instead of the int32 table
// (56 / 72 B per site) wherever the geometry has records -- the read-outs are HBM-bound like the
// step kernels, and the table was a quarter of what they moved. READOUT_MINB: the decode holds
// Q - 1 records of four words for a moment; without a bound ptxas takes 70-92 registers (two or
// three blocks of 256 per SM) and the two dependent round trips (records, then populations) are
// not covered (profiles/r02_tuning.md section 16).
#ifndef HLB_READOUT_MINB
#define HLB_READOUT_MINB 4
#endif
#ifndef HLB_READOUT_MINB_Q19
#define HLB_READOUT_MINB_Q19 3
#endif
template <typename L> constexpr int readout_minb() { return L::Q > 15 ? HLB_READOUT_MINB_Q19 : HLB_READOUT_MINB; }
template <typename L, typename ST, int MODE, bool REC, typename IT>
__device__ __forceinline__ void gather_precollision(const ST* __restrict__ buf,
                                                    const int32_t* __restrict__ nbr,
                                                    const uint4* __restrict__ rec, long long Ns,
                                                    const Planes& pl, long long i, double (&h)[L::Q]) {
  h[0] = to_real(buf[i]);
  if (REC && MODE != GATHER_OWN) {
    IT off[L::Q - 1];
    link_offsets<L, MODE, true, IT>(nbr, rec, Ns, i, pl, off);
#pragma unroll
    for (int q = 1; q < L::Q; ++q) h[q] = to_real(buf[off[q - 1]]);
    return;
  }
  int32_t e[L::Q - 1];
  if (MODE != GATHER_OWN) load_entries<L>(nbr, Ns, i, e);
#pragma unroll
  for (int q = 1; q < L::Q; ++q)
    h[q] = to_real(buf[slot_of<MODE>(q, MODE != GATHER_OWN ? e[q - 1] : 0, Ns, i)]);
}

template <typename L, typename ST, int MODE, bool REC, typename IT>
__global__ void __launch_bounds__(BLOCK, readout_minb<L>())
k_macroscopic(const ST* __restrict__ buf, const int32_t* __restrict__ nbr, const uint4* __restrict__ rec, Planes pl,
              const int32_t* __restrict__ canon, long long N, long long Ns,
              double* __restrict__ rho, double* __restrict__ u) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= N) return;
  double h[L::Q];
  gather_precollision<L, ST, MODE, REC, IT>(buf, nbr, rec, Ns, pl, i, h);
  const Moments m = moments_of<L>(h);
  const long long c = canon[i];
  if (rho) rho[c] = m.rho;
  if (u) {
    u[3 * c + 0] = m.ux;
    u[3 * c + 1] = m.uy;
    u[3 * c + 2] = m.uz;
  }
}

// Deviatoric (viscous) stress of the pre-collision state, canonical order, [N][6] in the
// order xx, yy, zz, xy, xz, yz:  sigma_ab = -(1 - omega / 2) sum_q c_qa c_qb (h_q - heq_q)
// (the shift w_q cancels in h - heq).
template <typename L, typename ST, int MODE, bool REC, typename IT>
__global__ void __launch_bounds__(BLOCK, readout_minb<L>())
k_stress(const ST* __restrict__ buf, const int32_t* __restrict__ nbr, const uint4* __restrict__ rec, Planes pl,
         const int32_t* __restrict__ canon, long long N, long long Ns, double omega,
         double* __restrict__ sigma) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= N) return;
  double h[L::Q];
  gather_precollision<L, ST, MODE, REC, IT>(buf, nbr, rec, Ns, pl, i, h);
  const Moments m = moments_of<L>(h);
  double pi[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int q = 1; q < L::Q; ++q) {  // c_0 = 0 contributes nothing
    const double neq = h[q] - heq_of<L>(q, m.drho, m.rho, m.ux, m.uy, m.uz);
    const int cx = L::cx(q), cy = L::cy(q), cz = L::cz(q);
    if (cx * cx) pi[0] += neq;
    if (cy * cy) pi[1] += neq;
    if (cz * cz) pi[2] += neq;
    if (cx * cy) pi[3] += (cx * cy > 0 ? neq : -neq);
    if (cx * cz) pi[4] += (cx * cz > 0 ? neq : -neq);
    if (cy * cz) pi[5] += (cy * cz > 0 ? neq : -neq);
  }
  const double pref = -(1.0 - 0.5 * omega);
  const long long c = canon[i];
#pragma unroll
  for (int k = 0; k < 6; ++k) sigma[c * 6 + k] = pref * pi[k];
}

// Wall shear stress from a stress tensor field and wall normals, both in canonical order:
// |t - (t.n) n| with t = sigma n and n the normalised normal; 0 where the normal is zero.
__global__ void __launch_bounds__(BLOCK)
k_wall_shear_stress(const double* __restrict__ sigma, const double* __restrict__ normals,
                    long long N, double* __restrict__ wss) {
  const long long c = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (c >= N) return;
  const double nx = normals[3 * c], ny = normals[3 * c + 1], nz = normals[3 * c + 2];
  const double len = sqrt(nx * nx + ny * ny + nz * nz);
  if (!(len > 0.0)) { wss[c] = 0.0; return; }
  const double n0 = nx / len, n1 = ny / len, n2 = nz / len;
  const double* s = sigma + 6 * c;  // xx yy zz xy xz yz
  const double t0 = s[0] * n0 + s[3] * n1 + s[4] * n2;
  const double t1 = s[3] * n0 + s[1] * n1 + s[5] * n2;
  const double t2 = s[4] * n0 + s[5] * n1 + s[2] * n2;
  const double tn = t0 * n0 + t1 * n1 + t2 * n2;
  const double a = t0 - tn * n0, b = t1 - tn * n1, d = t2 - tn * n2;
  wss[c] = sqrt(a * a + b * b + d * d);
}

template <typename L, typename ST, int MODE, bool REC, typename IT>
__global__ void __launch_bounds__(BLOCK, readout_minb<L>())
k_get_populations(const ST* __restrict__ buf, const int32_t* __restrict__ nbr, const uint4* __restrict__ rec, Planes pl,
                  const int32_t* __restrict__ canon, long long N, long long Ns,
                  double* __restrict__ f) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= N) return;
  double h[L::Q];
  gather_precollision<L, ST, MODE, REC, IT>(buf, nbr, rec, Ns, pl, i, h);
  const long long c = canon[i];
#pragma unroll
  for (int q = 0; q < L::Q; ++q) f[c * L::Q + q] = h[q] + L::weight(q);
}

// shifted initial population of direction q at internal site `site`
template <typename L>
__device__ __forceinline__ double initial_h(int q, long long site, const int32_t* __restrict__ canon,
                                            const double* __restrict__ rho_in,
                                            const double* __restrict__ u_in,
                                            const double* __restrict__ f_in) {
  const long long c = canon[site];
  if (f_in) return f_in[c * L::Q + q] - L::weight(q);
  const double r = rho_in ? rho_in[c] : 1.0;
  const double ux = u_in ? u_in[3 * c + 0] : 0.0, uy = u_in ? u_in[3 * c + 1] : 0.0,
               uz = u_in ? u_in[3 * c + 2] : 0.0;
  return heq_of<L>(q, r - 1.0, r, ux, uy, uz);
}

// MODE GATHER_OWN: buf[q][x] = h_q(x). MODE GATHER_PULL: slot (p, y) is read either by the
// fluid site y + c_p as its direction p, or (wall / iolet link) by y itself as direction
// opp(p); store the reader's initial population there, so that the first gather yields
// exactly f(., 0) = f_eq(rho0, u0) at every site and link.
template <typename L, typename ST, int MODE>
__global__ void __launch_bounds__(BLOCK)
k_init(ST* __restrict__ buf, const int32_t* __restrict__ nbr, const int32_t* __restrict__ canon,
       long long N, long long Ns, const double* __restrict__ rho_in,
       const double* __restrict__ u_in, const double* __restrict__ f_in) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= Ns) return;
  if (i >= N) {
#pragma unroll
    for (int q = 0; q < L::Q; ++q) buf[(long long)q * Ns + i] = to_store<ST>(0.0);
    return;
  }
  buf[i] = to_store<ST>(initial_h<L>(0, i, canon, rho_in, u_in, f_in));
#pragma unroll
  for (int p = 1; p < L::Q; ++p) {
    double v;
    if (MODE == GATHER_OWN) {
      v = initial_h<L>(p, i, canon, rho_in, u_in, f_in);
    } else {
      const int32_t e = __ldg(nbr + (long long)(opp(p) - 1) * Ns + i);  // pull source of opp(p) = y + c_p
      v = e >= 0 ? initial_h<L>(p, e, canon, rho_in, u_in, f_in)
                 : initial_h<L>(opp(p), i, canon, rho_in, u_in, f_in);
    }
    buf[(long long)p * Ns + i] = to_store<ST>(v);
  }
}

inline unsigned grid_for(long long n) { return (unsigned)((n + BLOCK - 1) / BLOCK); }

}  // namespace

int bfl_row_doubles(bool d3q19) { return d3q19 ? bfl_row<D3Q19>() : bfl_row<D3Q15>(); }
int resident_sites_per_sm_pull(bool d3q19, bool f32) {
  if (d3q19) return SBLOCK * pull_minb<D3Q19, true>();
  return SBLOCK * (f32 ? pull_minb<D3Q15, true>() - pull_f64_drop<D3Q15, float, true>()
                       : pull_minb<D3Q15, true>() - pull_f64_drop<D3Q15, double, true>());
}
int resident_kernel_sites_per_sm() { return SBLOCK * RESIDENT_MINB; }
int resident_sites_per_sm_aa(bool d3q19, bool f32) {  // of the odd (gather) kernel, the tighter of the two
  if (d3q19) return SBLOCK * (aa_odd_minb<D3Q19, true>() +
                              (f32 ? odd_smem_minb_add<D3Q19, float, true, uint32_t, 0>() : 0));
  return SBLOCK * (aa_odd_minb<D3Q15, true>() +
                   (f32 ? odd_smem_minb_add<D3Q15, float, true, uint32_t, 0>() : 0));
}

// ------------------------------------------------------------------ launchers
static Planes planes_of(const DeviceGeometry& g) {
  Planes pl;
  for (int q = 0; q < MAXQ; ++q) pl.p[q] = (uint32_t)((uint64_t)q * (uint64_t)g.Ns);
  return pl;
}
static IoletIndex iolet_index(const DeviceGeometry& g) {
  IoletIndex io;
  io.idx = (const uint2*)g.iolet_idx;
  io.links = (const uint4*)g.iolet_links;
  return io;
}
// Step kernels are launched with the programmatic-stream-serialization attribute when
// g.pdl is set (see pdl_launch_dependents above).
template <typename... KArgs, typename... Args>
static void launch_step(const DeviceGeometry& g, void (*kernel)(KArgs...), cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(g.Ns / SBLOCK));
  cfg.blockDim = dim3(SBLOCK);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = g.pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// -DHLB_TUNE_MIN (tuning builds only): compile just the instantiations the BASELINE configs run
// (D3Q15, link records, 32-bit offsets, lean iolet path) so that a kernel experiment builds in
// seconds; everything else aborts.
#ifdef HLB_TUNE_MIN
#define HLB_FULL_ONLY(...) do { fprintf(stderr, "HLB_TUNE_MIN build: instantiation not compiled\n"); abort(); } while (0)
#else
#define HLB_FULL_ONLY(...) __VA_ARGS__
#endif
#if defined(HLB_TUNE_MIN) && !defined(HLB_TUNE_BFL)
#define HLB_BFL_ONLY(...) HLB_FULL_ONLY(__VA_ARGS__)
#else
#define HLB_BFL_ONLY(...) __VA_ARGS__   // (-DHLB_TUNE_BFL: a tuning build that keeps the V = 2 kernels)
#endif
template <typename L, typename ST, bool REC, typename IT>
static void pull_launch(const DeviceGeometry& g, const void* src, void* dst, cudaStream_t s) {
#define HLB_PULL_ARGS s, (const ST*)src, (ST*)dst, g.nbr, (const uint4*)g.rec, iolet_index(g), g.iolet_par, \
                      (long long)g.Ns, make_relax<L>(g.omega), planes_of(g), (long long)g.prefetch_pull, g.bflf
  if (g.bfl_on) HLB_BFL_ONLY(launch_step(g, k_pull<L, ST, REC, IT, 2>, HLB_PULL_ARGS));
  else if (g.iolet_full) HLB_FULL_ONLY(launch_step(g, k_pull<L, ST, REC, IT, 1>, HLB_PULL_ARGS));
  else launch_step(g, k_pull<L, ST, REC, IT, 0>, HLB_PULL_ARGS);
#undef HLB_PULL_ARGS
}
template <typename L, typename ST>
static void pull_t(const DeviceGeometry& g, const void* src, void* dst, cudaStream_t s) {
  const bool idx32 = !g.index64;
  if (g.use_rec) {
    if (idx32) pull_launch<L, ST, true, uint32_t>(g, src, dst, s);
    else HLB_FULL_ONLY(pull_launch<L, ST, true, long long>(g, src, dst, s));
  } else {
    if (idx32) HLB_FULL_ONLY(pull_launch<L, ST, false, uint32_t>(g, src, dst, s));
    else HLB_FULL_ONLY(pull_launch<L, ST, false, long long>(g, src, dst, s));
  }
}
template <typename L, typename ST, bool REC, typename IT>
static void aa_odd_launch(const DeviceGeometry& g, void* a, cudaStream_t s) {
#define HLB_ODD_ARGS s, (ST*)a, g.nbr, (const uint4*)g.rec, iolet_index(g), g.iolet_par, (long long)g.Ns, \
                     make_relax<L>(g.omega), planes_of(g), (long long)g.prefetch_aa, g.bflf
  if (g.bfl_on) HLB_BFL_ONLY(launch_step(g, k_aa_odd<L, ST, REC, IT, 2>, HLB_ODD_ARGS));
  else if (g.iolet_full) HLB_FULL_ONLY(launch_step(g, k_aa_odd<L, ST, REC, IT, 1>, HLB_ODD_ARGS));
  else launch_step(g, k_aa_odd<L, ST, REC, IT, 0>, HLB_ODD_ARGS);
#undef HLB_ODD_ARGS
}
template <typename L, typename ST>
static void aa_t(const DeviceGeometry& g, void* a, bool odd, cudaStream_t s) {
  const bool idx32 = !g.index64;
  if (!odd) {
#define HLB_EVEN_ARGS s, (ST*)a, iolet_index(g), g.iolet_par, (long long)g.Ns, make_relax<L>(g.omega), \
                      (long long)g.prefetch_aa, g.bflf
    if (g.bfl_on) HLB_BFL_ONLY(launch_step(g, k_aa_even<L, ST, 2>, HLB_EVEN_ARGS));
    else if (g.iolet_full) HLB_FULL_ONLY(launch_step(g, k_aa_even<L, ST, 1>, HLB_EVEN_ARGS));
    else launch_step(g, k_aa_even<L, ST, 0>, HLB_EVEN_ARGS);
#undef HLB_EVEN_ARGS
  } else if (g.use_rec) {
    if (idx32) aa_odd_launch<L, ST, true, uint32_t>(g, a, s);
    else HLB_FULL_ONLY(aa_odd_launch<L, ST, true, long long>(g, a, s));
  } else {
    if (idx32) HLB_FULL_ONLY(aa_odd_launch<L, ST, false, uint32_t>(g, a, s));
    else HLB_FULL_ONLY(aa_odd_launch<L, ST, false, long long>(g, a, s));
  }
}
template <typename L, typename ST>
static void macroscopic_t(const DeviceGeometry& g, const void* buf, GatherMode mode, double* rho,
                          double* u, cudaStream_t s) {
  const unsigned grid = grid_for(g.N);
  const ST* b = (const ST*)buf;
  switch (mode) {
    case GATHER_PULL:
      if (g.use_rec && !g.index64) k_macroscopic<L, ST, GATHER_PULL, true, uint32_t><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, rho, u);
      else if (g.use_rec) HLB_FULL_ONLY((k_macroscopic<L, ST, GATHER_PULL, true, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, rho, u)));
      else HLB_FULL_ONLY((k_macroscopic<L, ST, GATHER_PULL, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, rho, u)));
      break;
    case GATHER_OWN: k_macroscopic<L, ST, GATHER_OWN, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, rho, u); break;
    case GATHER_AA_ODD:
      if (g.use_rec && !g.index64) k_macroscopic<L, ST, GATHER_AA_ODD, true, uint32_t><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, rho, u);
      else if (g.use_rec) HLB_FULL_ONLY((k_macroscopic<L, ST, GATHER_AA_ODD, true, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, rho, u)));
      else HLB_FULL_ONLY((k_macroscopic<L, ST, GATHER_AA_ODD, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, rho, u)));
      break;
  }
}
template <typename L, typename ST>
static void get_populations_t(const DeviceGeometry& g, const void* buf, GatherMode mode, double* f,
                              cudaStream_t s) {
  const unsigned grid = grid_for(g.N);
  const ST* b = (const ST*)buf;
  switch (mode) {
    case GATHER_PULL:
      if (g.use_rec && !g.index64) k_get_populations<L, ST, GATHER_PULL, true, uint32_t><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, f);
      else if (g.use_rec) HLB_FULL_ONLY((k_get_populations<L, ST, GATHER_PULL, true, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, f)));
      else HLB_FULL_ONLY((k_get_populations<L, ST, GATHER_PULL, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, f)));
      break;
    case GATHER_OWN: k_get_populations<L, ST, GATHER_OWN, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, f); break;
    case GATHER_AA_ODD:
      if (g.use_rec && !g.index64) k_get_populations<L, ST, GATHER_AA_ODD, true, uint32_t><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, f);
      else if (g.use_rec) HLB_FULL_ONLY((k_get_populations<L, ST, GATHER_AA_ODD, true, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, f)));
      else HLB_FULL_ONLY((k_get_populations<L, ST, GATHER_AA_ODD, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, f)));
      break;
  }
}
template <typename L, typename ST>
static void stress_t(const DeviceGeometry& g, const void* buf, GatherMode mode, double* sigma,
                     cudaStream_t s) {
  const unsigned grid = grid_for(g.N);
  const ST* b = (const ST*)buf;
  switch (mode) {
    case GATHER_PULL:
      if (g.use_rec && !g.index64) k_stress<L, ST, GATHER_PULL, true, uint32_t><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, g.omega, sigma);
      else if (g.use_rec) HLB_FULL_ONLY((k_stress<L, ST, GATHER_PULL, true, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, g.omega, sigma)));
      else HLB_FULL_ONLY((k_stress<L, ST, GATHER_PULL, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, g.omega, sigma)));
      break;
    case GATHER_OWN: k_stress<L, ST, GATHER_OWN, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, g.omega, sigma); break;
    case GATHER_AA_ODD:
      if (g.use_rec && !g.index64) k_stress<L, ST, GATHER_AA_ODD, true, uint32_t><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, g.omega, sigma);
      else if (g.use_rec) HLB_FULL_ONLY((k_stress<L, ST, GATHER_AA_ODD, true, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, (const uint4*)g.rec, planes_of(g), g.canon, g.N, g.Ns, g.omega, sigma)));
      else HLB_FULL_ONLY((k_stress<L, ST, GATHER_AA_ODD, false, long long><<<grid, BLOCK, 0, s>>>(b, g.nbr, nullptr, planes_of(g), g.canon, g.N, g.Ns, g.omega, sigma)));
      break;
  }
}
template <typename L, typename ST>
static void init_t(const DeviceGeometry& g, void* buf, GatherMode mode, const double* rho_in,
                   const double* u_in, const double* f_in, cudaStream_t s) {
  const unsigned grid = grid_for(g.Ns);
  if (mode == GATHER_PULL)
    k_init<L, ST, GATHER_PULL><<<grid, BLOCK, 0, s>>>((ST*)buf, g.nbr, g.canon, g.N, g.Ns, rho_in, u_in, f_in);
  else
    k_init<L, ST, GATHER_OWN><<<grid, BLOCK, 0, s>>>((ST*)buf, g.nbr, g.canon, g.N, g.Ns, rho_in, u_in, f_in);
}

// lattice x storage dispatch: F is a generic lambda called with (L{}, ST{})
template <typename F>
static void dispatch(const DeviceGeometry& g, F&& f) {
  if (g.d3q19) {
    if (g.f32) HLB_FULL_ONLY(f(D3Q19{}, float{}));
    else HLB_FULL_ONLY(f(D3Q19{}, double{}));
  } else {
    if (g.f32) f(D3Q15{}, float{});
    else f(D3Q15{}, double{});
  }
}

// Cooperative launch of a resident kernel: fails (without launching) with
// cudaErrorCooperativeLaunchTooLarge when the grid does not fit on the chip at once.
template <typename... KArgs, typename... Args>
static cudaError_t launch_resident(const DeviceGeometry& g, void (*kernel)(KArgs...), cudaStream_t s,
                                   Args... args) {
  std::tuple<KArgs...> vals{KArgs(args)...};
  void* ptrs[sizeof...(KArgs)];
  int k = 0;
  std::apply([&](auto&... v) { ((ptrs[k++] = (void*)&v), ...); }, vals);
  return cudaLaunchCooperativeKernel((const void*)kernel, dim3((unsigned)(g.Ns / SBLOCK)), dim3(SBLOCK),
                                     ptrs, 0, s);
}
template <typename L, typename ST, bool REC>
static cudaError_t resident_launch(const DeviceGeometry& g, bool aa, void* b0, void* b1, long long n,
                                   int odd0, unsigned long long* bar, unsigned long long base,
                                   cudaStream_t s) {
  using IT = uint32_t;
  if (aa) {
#define HLB_RES_ARGS s, (ST*)b0, g.nbr, (const uint4*)g.rec, iolet_index(g), g.iolet_par, g.bflf.iolet_w, \
                     (long long)g.Ns, make_relax<L>(g.omega), planes_of(g), n, odd0, bar, base
#ifndef HLB_TUNE_MIN
    if (g.iolet_full) return launch_resident(g, k_aa_resident<L, ST, REC, IT, 1>, HLB_RES_ARGS);
#endif
    return launch_resident(g, k_aa_resident<L, ST, REC, IT, 0>, HLB_RES_ARGS);
#undef HLB_RES_ARGS
  }
#define HLB_RES_ARGS s, (ST*)b0, (ST*)b1, g.nbr, (const uint4*)g.rec, iolet_index(g), g.iolet_par, \
                     g.bflf.iolet_w, (long long)g.Ns, make_relax<L>(g.omega), planes_of(g), n, bar, base
#ifndef HLB_TUNE_MIN
  if (g.iolet_full) return launch_resident(g, k_pull_resident<L, ST, REC, IT, 1>, HLB_RES_ARGS);
#endif
  return launch_resident(g, k_pull_resident<L, ST, REC, IT, 0>, HLB_RES_ARGS);
#undef HLB_RES_ARGS
}
cudaError_t launch_resident_steps(const DeviceGeometry& g, bool aa, void* b0, void* b1, long long n,
                                  int odd0, unsigned long long* bar, unsigned long long base,
                                  cudaStream_t s) {
  if (g.index64) return cudaErrorCooperativeLaunchTooLarge;  // 32-bit offsets only (small geometries)
  cudaError_t e = cudaSuccess;
  dispatch(g, [&](auto l, auto st) {
    using L = decltype(l);
    using ST = decltype(st);
    if (g.use_rec) e = resident_launch<L, ST, true>(g, aa, b0, b1, n, odd0, bar, base, s);
    else HLB_FULL_ONLY(e = resident_launch<L, ST, false>(g, aa, b0, b1, n, odd0, bar, base, s));
  });
  return e;
}

void launch_pull(const DeviceGeometry& g, const void* src, void* dst, cudaStream_t s) {
  dispatch(g, [&](auto l, auto st) { pull_t<decltype(l), decltype(st)>(g, src, dst, s); });
}
template <typename ST>
static void bfl_prepass_t(const DeviceGeometry& g, void* buf, GatherMode mode, cudaStream_t s) {
  const BflLinks& b = g.bfl;
  const long long per_block = (long long)BFL_UNROLL * BLOCK;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)((b.n + per_block - 1) / per_block));
  cfg.blockDim = dim3(BLOCK);
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = g.pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, k_bfl_prepass<ST>, (ST*)buf, (long long)g.Ns, b.site, b.behind, b.link, b.d,
                     (long long)b.n, (int)mode);
}
void launch_bfl_prepass(const DeviceGeometry& g, void* buf, GatherMode mode, cudaStream_t s) {
  if (g.bfl.n <= 0) return;
  if (g.f32) bfl_prepass_t<float>(g, buf, mode, s);
  else bfl_prepass_t<double>(g, buf, mode, s);
}
void launch_aa(const DeviceGeometry& g, void* a, bool odd, cudaStream_t s) {
  dispatch(g, [&](auto l, auto st) { aa_t<decltype(l), decltype(st)>(g, a, odd, s); });
}
void launch_macroscopic(const DeviceGeometry& g, const void* buf, GatherMode mode, double* rho,
                        double* u, cudaStream_t s) {
  dispatch(g, [&](auto l, auto st) { macroscopic_t<decltype(l), decltype(st)>(g, buf, mode, rho, u, s); });
}
void launch_get_populations(const DeviceGeometry& g, const void* buf, GatherMode mode, double* f,
                            cudaStream_t s) {
  dispatch(g, [&](auto l, auto st) { get_populations_t<decltype(l), decltype(st)>(g, buf, mode, f, s); });
}
void launch_stress(const DeviceGeometry& g, const void* buf, GatherMode mode, double* sigma,
                   cudaStream_t s) {
  dispatch(g, [&](auto l, auto st) { stress_t<decltype(l), decltype(st)>(g, buf, mode, sigma, s); });
}
// ------------------------------------------------------------------ static scratch (no-allocation entry point)
// sigma [NOALLOC_MAX_SITES][6] of hlb_get_wall_shear_stress_noalloc. Uninitialised device
// memory of the module (12 MiB per GPU that loads the library, until exit; not in the file).
// Host code must NOT pass `g_noalloc_sigma` itself to a kernel -- in host code the name is a
// host-side shadow of the symbol -- but the address cudaGetSymbolAddress returns for the device
// that is current.
static __device__ __align__(256) double g_noalloc_sigma[NOALLOC_MAX_SITES * 6];
namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
double* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};
std::mutex g_noalloc_mutex;
}  // namespace
cudaError_t noalloc_scratch_setup() {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (g_noalloc_ptr[dev]) return cudaSuccess;  // once per device
  double* ptr = nullptr;
  e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_sigma);
  if (e != cudaSuccess) return e;
  if (!ptr) return cudaErrorInvalidSymbol;
  g_noalloc_ptr[dev] = ptr;
  return cudaSuccess;
}
double* noalloc_scratch() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NOALLOC_MAX_DEVICES) return nullptr;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  return g_noalloc_ptr[dev];
}

void launch_wall_shear_stress(const double* sigma, const double* normals, long long N, double* wss,
                              cudaStream_t s) {
  k_wall_shear_stress<<<grid_for(N), BLOCK, 0, s>>>(sigma, normals, N, wss);
}
void launch_init(const DeviceGeometry& g, void* buf, GatherMode mode, const double* rho_in,
                 const double* u_in, const double* f_in, cudaStream_t s) {
  dispatch(g, [&](auto l, auto st) { init_t<decltype(l), decltype(st)>(g, buf, mode, rho_in, u_in, f_in, s); });
}

}  // namespace hlb
