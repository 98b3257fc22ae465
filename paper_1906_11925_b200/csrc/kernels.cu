// kernels.cu -- fused D3Q15 LBGK collide-and-stream kernels for sm_100a.
//
// One thread per fluid site, structure-of-arrays populations buf[slot][site] with plane
// stride Ns (a multiple of 128, planes 1 KiB aligned), so the own-site loads and all stores
// of a warp are single fully-coalesced 256-byte (fp64) / 128-byte (fp32) requests; the 14
// gathers follow the int32 pull-neighbour table. The work is
// an indirect gather/scatter stream at ~0.9 flop/byte: HBM-bound, no tensor cores, no
// shared memory (no intra-block reuse: every population is read exactly once per step).
//
// Memory-level parallelism: all 14 index loads are issued first, then all 15 population
// loads, then the arithmetic (Guideline 7 of the Blackwell guide).
//
// Sites i in [N, Ns) are padding: their table entries are all "wall", their populations
// are 0 (rest state in shifted form) and stay exactly 0, so no kernel needs a bounds
// branch inside a warp.
#include "kernels.cuh"

#include "lbgk.cuh"

namespace hlb {
namespace {

constexpr int BLOCK = 256;

__device__ __forceinline__ int iolet_of(int32_t e) {  // -1: not an iolet link
  return e < 0 ? (int)(e & 0x7fffffff) - 1 : -1;
}

template <typename ST>
__device__ __forceinline__ void load_entries(const int32_t* __restrict__ nbr, long long Ns,
                                             long long i, int32_t (&e)[Q - 1]) {
#pragma unroll
  for (int q = 1; q < Q; ++q) e[q - 1] = __ldg(nbr + (long long)(q - 1) * Ns + i);
}

// Address (element offset) where the pre-collision f_q(x) of link q lives.
template <int MODE>
__device__ __forceinline__ long long slot_of(int q, int32_t e, long long Ns, long long i) {
  if (MODE == GATHER_OWN) return (long long)q * Ns + i;
  const bool wall = e < 0;
  if (MODE == GATHER_PULL)  // post-collision buffer: wall -> own opposite slot
    return wall ? (long long)opp(q) * Ns + i : (long long)q * Ns + e;
  // GATHER_AA_ODD: slot opp(q) of the source site, slot q of the site itself at walls
  return wall ? (long long)q * Ns + i : (long long)opp(q) * Ns + e;
}

// Replace, for every iolet link p of this site, the value that will be read back as
// f_p(x, t+1) by the constant-density equilibrium f_eq_p(rho_k, u(x, t)) (reading A6).
// out[p] is that value; for non-iolet links it keeps the bounced post-collision value.
__device__ __forceinline__ void iolet_substitute(const int32_t (&e)[Q - 1], const Moments& m,
                                                 const double* __restrict__ iolet_rho,
                                                 double (&out)[Q]) {
#pragma unroll
  for (int p = 1; p < Q; ++p) {
    const int k = iolet_of(e[p - 1]);
    if (k >= 0) {
      const double rk = __ldg(iolet_rho + k);
      out[p] = heq_of(p, rk - 1.0, rk, m.ux, m.uy, m.uz);
    }
  }
}

// ------------------------------------------------------------------ two-lattice pull
// src holds post-collision values h*(., t-1) (iolet slots substituted); one launch does
// gather -> moments -> BGK -> store of h*(., t) into dst (rows S1..S6 fused).
template <typename ST>
__global__ void __launch_bounds__(BLOCK)
k_pull(const ST* __restrict__ src, ST* __restrict__ dst, const int32_t* __restrict__ nbr,
       const double* __restrict__ iolet_rho, long long Ns, double omega) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= Ns) return;
  int32_t e[Q - 1];
  load_entries<ST>(nbr, Ns, i, e);
  double h[Q];
  h[0] = to_real(src[i]);
  int io = 0;
#pragma unroll
  for (int q = 1; q < Q; ++q) {
    h[q] = to_real(src[slot_of<GATHER_PULL>(q, e[q - 1], Ns, i)]);
    io |= e[q - 1] < 0 ? (e[q - 1] & 0x7fffffff) : 0;
  }
  const Moments m = moments_of(h);
  double hs[Q];
  collide(h, m, omega, hs);
  if (io) {  // rare: sites on an inlet/outlet cap
    // slot opp(p) of this site is read back by link p next step
    double back[Q];
#pragma unroll
    for (int p = 1; p < Q; ++p) back[p] = hs[opp(p)];
    iolet_substitute(e, m, iolet_rho, back);
#pragma unroll
    for (int p = 1; p < Q; ++p) hs[opp(p)] = back[p];
  }
#pragma unroll
  for (int q = 0; q < Q; ++q) dst[(long long)q * Ns + i] = to_store<ST>(hs[q]);
}

// ------------------------------------------------------------------ A-A in place
// Even phase: read slot q of the site, write h*_q to slot opp(q) of the site (no table).
// Odd phase: read f_q from slot opp(q) of x - c_q (slot q of x at a wall), write h*_q to
// the address f_opp(q) was read from. Read set = write set per site in both phases, so one
// array and no inter-thread hazards.
template <typename ST, bool ODD>
__global__ void __launch_bounds__(BLOCK)
k_aa(ST* __restrict__ a, const int32_t* __restrict__ nbr, const uint32_t* __restrict__ iolet_bits,
     const double* __restrict__ iolet_rho, long long Ns, double omega) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= Ns) return;
  int32_t e[Q - 1];
  bool io;
  if (ODD) {
    load_entries<ST>(nbr, Ns, i, e);
    int any = 0;
#pragma unroll
    for (int q = 1; q < Q; ++q) any |= e[q - 1] < 0 ? (e[q - 1] & 0x7fffffff) : 0;
    io = any != 0;
  } else {
    io = (__ldg(iolet_bits + (i >> 5)) >> (i & 31)) & 1u;
    if (io) load_entries<ST>(nbr, Ns, i, e);
  }
  long long addr[Q];
  double h[Q];
  addr[0] = i;
#pragma unroll
  for (int q = 1; q < Q; ++q)
    addr[q] = ODD ? slot_of<GATHER_AA_ODD>(q, e[q - 1], Ns, i) : slot_of<GATHER_OWN>(q, 0, Ns, i);
#pragma unroll
  for (int q = 0; q < Q; ++q) h[q] = to_real(a[addr[q]]);
  const Moments m = moments_of(h);
  double hs[Q];
  collide(h, m, omega, hs);
  double out[Q];  // out[p] is written where f_p was read: the bounced h*_opp(p)
  out[0] = hs[0];
#pragma unroll
  for (int p = 1; p < Q; ++p) out[p] = hs[opp(p)];
  if (io) iolet_substitute(e, m, iolet_rho, out);
#pragma unroll
  for (int p = 0; p < Q; ++p) a[addr[p]] = to_store<ST>(out[p]);
}

// ------------------------------------------------------------------ read-out / init
template <typename ST, int MODE>
__device__ __forceinline__ void gather_precollision(const ST* __restrict__ buf,
                                                    const int32_t* __restrict__ nbr, long long Ns,
                                                    long long i, double (&h)[Q]) {
  int32_t e[Q - 1];
  if (MODE != GATHER_OWN) load_entries<ST>(nbr, Ns, i, e);
  h[0] = to_real(buf[i]);
#pragma unroll
  for (int q = 1; q < Q; ++q)
    h[q] = to_real(buf[slot_of<MODE>(q, MODE != GATHER_OWN ? e[q - 1] : 0, Ns, i)]);
}

template <typename ST, int MODE>
__global__ void __launch_bounds__(BLOCK)
k_macroscopic(const ST* __restrict__ buf, const int32_t* __restrict__ nbr,
              const int32_t* __restrict__ canon, long long N, long long Ns,
              double* __restrict__ rho, double* __restrict__ u) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= N) return;
  double h[Q];
  gather_precollision<ST, MODE>(buf, nbr, Ns, i, h);
  const Moments m = moments_of(h);
  const long long c = canon[i];
  if (rho) rho[c] = m.rho;
  if (u) {
    u[3 * c + 0] = m.ux;
    u[3 * c + 1] = m.uy;
    u[3 * c + 2] = m.uz;
  }
}

template <typename ST, int MODE>
__global__ void __launch_bounds__(BLOCK)
k_get_populations(const ST* __restrict__ buf, const int32_t* __restrict__ nbr,
                  const int32_t* __restrict__ canon, long long N, long long Ns,
                  double* __restrict__ f) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= N) return;
  double h[Q];
  gather_precollision<ST, MODE>(buf, nbr, Ns, i, h);
  const long long c = canon[i];
#pragma unroll
  for (int q = 0; q < Q; ++q) f[c * Q + q] = h[q] + weight(q);
}

// shifted initial population of direction q at internal site `site`
__device__ __forceinline__ double initial_h(int q, long long site, const int32_t* __restrict__ canon,
                                            const double* __restrict__ rho_in,
                                            const double* __restrict__ u_in,
                                            const double* __restrict__ f_in) {
  const long long c = canon[site];
  if (f_in) return f_in[c * Q + q] - weight(q);
  const double r = rho_in ? rho_in[c] : 1.0;
  const double ux = u_in ? u_in[3 * c + 0] : 0.0, uy = u_in ? u_in[3 * c + 1] : 0.0,
               uz = u_in ? u_in[3 * c + 2] : 0.0;
  return heq_of(q, r - 1.0, r, ux, uy, uz);
}

// MODE GATHER_OWN: buf[q][x] = h_q(x). MODE GATHER_PULL: slot (p, y) is read either by the
// fluid site y + c_p as its direction p, or (wall / iolet link) by y itself as direction
// opp(p); store the reader's initial population there, so that the first gather yields
// exactly f(., 0) = f_eq(rho0, u0) at every site and link.
template <typename ST, int MODE>
__global__ void __launch_bounds__(BLOCK)
k_init(ST* __restrict__ buf, const int32_t* __restrict__ nbr, const int32_t* __restrict__ canon,
       long long N, long long Ns, const double* __restrict__ rho_in,
       const double* __restrict__ u_in, const double* __restrict__ f_in) {
  const long long i = (long long)blockIdx.x * BLOCK + threadIdx.x;
  if (i >= Ns) return;
  if (i >= N) {
#pragma unroll
    for (int q = 0; q < Q; ++q) buf[(long long)q * Ns + i] = to_store<ST>(0.0);
    return;
  }
  buf[i] = to_store<ST>(initial_h(0, i, canon, rho_in, u_in, f_in));
#pragma unroll
  for (int p = 1; p < Q; ++p) {
    double v;
    if (MODE == GATHER_OWN) {
      v = initial_h(p, i, canon, rho_in, u_in, f_in);
    } else {
      const int32_t e = __ldg(nbr + (long long)(opp(p) - 1) * Ns + i);  // pull source of opp(p) = y + c_p
      v = e >= 0 ? initial_h(p, e, canon, rho_in, u_in, f_in)
                 : initial_h(opp(p), i, canon, rho_in, u_in, f_in);
    }
    buf[(long long)p * Ns + i] = to_store<ST>(v);
  }
}

inline unsigned grid_for(long long n) { return (unsigned)((n + BLOCK - 1) / BLOCK); }

}  // namespace

void launch_pull(const DeviceGeometry& g, const void* src, void* dst, cudaStream_t s) {
  if (g.f32)
    k_pull<float><<<grid_for(g.Ns), BLOCK, 0, s>>>((const float*)src, (float*)dst, g.nbr,
                                                   g.iolet_rho, g.Ns, g.omega);
  else
    k_pull<double><<<grid_for(g.Ns), BLOCK, 0, s>>>((const double*)src, (double*)dst, g.nbr,
                                                    g.iolet_rho, g.Ns, g.omega);
}

void launch_aa(const DeviceGeometry& g, void* a, bool odd, cudaStream_t s) {
  const unsigned grid = grid_for(g.Ns);
  if (g.f32) {
    if (odd) k_aa<float, true><<<grid, BLOCK, 0, s>>>((float*)a, g.nbr, g.iolet_bits, g.iolet_rho, g.Ns, g.omega);
    else k_aa<float, false><<<grid, BLOCK, 0, s>>>((float*)a, g.nbr, g.iolet_bits, g.iolet_rho, g.Ns, g.omega);
  } else {
    if (odd) k_aa<double, true><<<grid, BLOCK, 0, s>>>((double*)a, g.nbr, g.iolet_bits, g.iolet_rho, g.Ns, g.omega);
    else k_aa<double, false><<<grid, BLOCK, 0, s>>>((double*)a, g.nbr, g.iolet_bits, g.iolet_rho, g.Ns, g.omega);
  }
}

template <typename ST>
static void macroscopic_t(const DeviceGeometry& g, const void* buf, GatherMode mode, double* rho,
                          double* u, cudaStream_t s) {
  const unsigned grid = grid_for(g.N);
  const ST* b = (const ST*)buf;
  switch (mode) {
    case GATHER_PULL: k_macroscopic<ST, GATHER_PULL><<<grid, BLOCK, 0, s>>>(b, g.nbr, g.canon, g.N, g.Ns, rho, u); break;
    case GATHER_OWN: k_macroscopic<ST, GATHER_OWN><<<grid, BLOCK, 0, s>>>(b, g.nbr, g.canon, g.N, g.Ns, rho, u); break;
    case GATHER_AA_ODD: k_macroscopic<ST, GATHER_AA_ODD><<<grid, BLOCK, 0, s>>>(b, g.nbr, g.canon, g.N, g.Ns, rho, u); break;
  }
}
void launch_macroscopic(const DeviceGeometry& g, const void* buf, GatherMode mode, double* rho,
                        double* u, cudaStream_t s) {
  if (g.f32) macroscopic_t<float>(g, buf, mode, rho, u, s);
  else macroscopic_t<double>(g, buf, mode, rho, u, s);
}

template <typename ST>
static void get_populations_t(const DeviceGeometry& g, const void* buf, GatherMode mode, double* f,
                              cudaStream_t s) {
  const unsigned grid = grid_for(g.N);
  const ST* b = (const ST*)buf;
  switch (mode) {
    case GATHER_PULL: k_get_populations<ST, GATHER_PULL><<<grid, BLOCK, 0, s>>>(b, g.nbr, g.canon, g.N, g.Ns, f); break;
    case GATHER_OWN: k_get_populations<ST, GATHER_OWN><<<grid, BLOCK, 0, s>>>(b, g.nbr, g.canon, g.N, g.Ns, f); break;
    case GATHER_AA_ODD: k_get_populations<ST, GATHER_AA_ODD><<<grid, BLOCK, 0, s>>>(b, g.nbr, g.canon, g.N, g.Ns, f); break;
  }
}
void launch_get_populations(const DeviceGeometry& g, const void* buf, GatherMode mode, double* f,
                            cudaStream_t s) {
  if (g.f32) get_populations_t<float>(g, buf, mode, f, s);
  else get_populations_t<double>(g, buf, mode, f, s);
}

template <typename ST>
static void init_t(const DeviceGeometry& g, void* buf, GatherMode mode, const double* rho_in,
                   const double* u_in, const double* f_in, cudaStream_t s) {
  const unsigned grid = grid_for(g.Ns);
  if (mode == GATHER_PULL)
    k_init<ST, GATHER_PULL><<<grid, BLOCK, 0, s>>>((ST*)buf, g.nbr, g.canon, g.N, g.Ns, rho_in, u_in, f_in);
  else
    k_init<ST, GATHER_OWN><<<grid, BLOCK, 0, s>>>((ST*)buf, g.nbr, g.canon, g.N, g.Ns, rho_in, u_in, f_in);
}
void launch_init(const DeviceGeometry& g, void* buf, GatherMode mode, const double* rho_in,
                 const double* u_in, const double* f_in, cudaStream_t s) {
  if (g.f32) init_t<float>(g, buf, mode, rho_in, u_in, f_in, s);
  else init_t<double>(g, buf, mode, rho_in, u_in, f_in, s);
}

}  // namespace hlb
