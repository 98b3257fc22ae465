// kernels.cuh -- launchers of the CUDA kernels (sm_100a). Host-callable, defined in kernels.cu.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace hlb {

// BFL interpolated walls, list form (used by the pre-pass before a read-out): the interpolated
// links with d < 1/2. Link l belongs to internal site site[l], is its pull link link[l]
// (1 .. Q-1), has the wall at the fraction d[l] of its length, and behind[l] is the internal
// index of the fluid site x + c_p behind it.
struct BflLinks {
  const int32_t* site = nullptr;
  const int32_t* behind = nullptr;
  const uint8_t* link = nullptr;
  const double* d = nullptr;
  long long n = 0;
};

// BFL interpolated walls, site form (used inside the step kernels, by value as a kernel
// argument): idx[i / 32] = {bits, rank}: bit i % 32 of bits marks the sites with an interpolated
// link; such a site has the dense index rank + popcount(bits below lane i % 32). ONE 8-byte word
// per group, loaded with the kernel's first loads: as two arrays read one after the other (bits,
// then rank only where flagged) they put two dependent memory round trips in front of the link
// records (profiles/r02_tuning.md section 12). A site's row coef[idx * row ...] (row =
// bfl_row_doubles() doubles, 16-byte aligned) holds ONE coefficient per opposite pair of links
// (2k + 1, 2k + 2), k = 0 .. (Q-1)/2 - 1 -- the two are never both interpolated --, then a
// 64-bit word whose bit k says which member is the interpolated link (1: 2k + 2). The
// coefficient is, for that pull link,  1 - 2d  where d < 1/2 (applied while gathering),
// -(1 - 1/(2d))  where d >= 1/2 (applied to the value the site writes back for that link),  0 = plain
// bounce-back. gather = 0 when the d < 1/2 part is already in the state buffer (pre-pass
// run for a read-out) or does not apply (the initial state).
struct BflFused {
  const uint2* idx = nullptr;      // [Ns/32] {bits, rank}
  const double* coef = nullptr;    // [nf][row]
  long long nf = 0;
  int gather = 0;
  // The other per-site option that travels in this by-value argument: velocity weights of the
  // Ladd iolets (hlb_set_iolet_weight), [Ns] in internal site order, read on the rare iolet
  // path only; NULL = no weights.
  const double* iolet_w = nullptr;
};

struct DeviceGeometry {
  int64_t N = 0;                        // fluid sites
  int64_t Ns = 0;                       // plane stride (multiple of 128), arrays are [Q][Ns]
  const int32_t* nbr = nullptr;         // [Q-1][Ns] pull-neighbour table (include/hlb.h)
  const void* iolet_idx = nullptr;      // [Ns/32] {bits, rank} (preprocess.h: iolet index)
  const void* iolet_links = nullptr;    // [iolet sites + 1] rows of link -> iolet id bytes
  const void* rec = nullptr;            // [Ns/32][Q-1] 16-byte link records (include/hlb.h)
  bool use_rec = false;                 // step kernels read rec instead of nbr
  BflLinks bfl;                         // applied by launch_bfl_prepass when the API says so
  BflFused bflf;                        // used by the step kernels when bfl_on
  bool bfl_on = false;                  // interpolated walls are set
  bool iolet_full = false;              // some iolet is a velocity iolet or has a normal
  bool pdl = true;                      // programmatic dependent launch of the step kernels
  bool index64 = false;                 // flat offsets need (or are forced to) 64 bits
  // > 0: every thread L2-prefetches what site i + prefetch_* will load (about 3/4 of the
  // sites resident on the chip at once, i.e. the blocks scheduled just under a wave later)
  int64_t prefetch_pull = 0, prefetch_aa = 0;
  const int32_t* canon = nullptr;       // [N] internal -> canonical rank
  const double* iolet_par = nullptr;    // [n_iolets][4]: {rho_k, nx, ny, nz} constant density
                                        // (unit normal or 0,0,0);
                                        // {-1, ux, uy, uz} Ladd velocity iolet
  double omega = 1.0;                   // 1 / tau
  bool f32 = false;                     // HLB_STORE_F32
  bool d3q19 = false;                   // HLB_LATTICE_D3Q19 (else D3Q15)
};

int bfl_row_doubles(bool d3q19);
// Sites resident on an SM at once (threads per block x resident blocks) per step kernel.
int resident_sites_per_sm_pull(bool d3q19, bool f32);
int resident_sites_per_sm_aa(bool d3q19, bool f32);
// Sites per SM the resident multi-step kernels (launch_resident_steps) are sized for.
int resident_kernel_sites_per_sm();

// One time step, two-lattice pull: dst <- collide(gather(src)).
void launch_pull(const DeviceGeometry& g, const void* src, void* dst, cudaStream_t s);
// One time step, A-A in place; `odd` selects the phase.
void launch_aa(const DeviceGeometry& g, void* a, bool odd, cudaStream_t s);

// n >= 1 time steps in ONE cooperative launch (small geometries: the whole grid of Ns / 128
// blocks must be resident at once, else cudaErrorCooperativeLaunchTooLarge and nothing is
// launched). A-A: b0 is the array, odd0 the phase of the first step; two-lattice: the first
// step reads b0 and writes b1, then they alternate. bar: a zero-initialised device counter owned
// by the geometry; base: its value before the launch (the launch adds (n - 1) * Ns / 128).
// Plain iolet rules only (no interpolated walls).
cudaError_t launch_resident_steps(const DeviceGeometry& g, bool aa, void* b0, void* b1, long long n,
                                  int odd0, unsigned long long* bar, unsigned long long base,
                                  cudaStream_t s);

// How the pre-collision populations f(., n) are found in a buffer.
enum GatherMode {
  GATHER_PULL = 0,   // two-lattice buffer holding post-collision values: pull through the table
  GATHER_OWN = 1,    // A-A after an even number of steps: slot q of the site itself
  GATHER_AA_ODD = 2  // A-A after an odd number of steps: slot opp(q) of x - c_q (slot q at walls)
};
// Rewrite, in the state buffer `buf` (its layout given by `mode`), the bounce-back slots of the
// interpolated links (see kernels.cu); run once per state, before the step or read-out that
// gathers from it.
void launch_bfl_prepass(const DeviceGeometry& g, void* buf, GatherMode mode, cudaStream_t s);
// rho [N] / u [N][3] (device, canonical order; either may be NULL)
void launch_macroscopic(const DeviceGeometry& g, const void* buf, GatherMode mode, double* rho,
                        double* u, cudaStream_t s);
// sigma [N][6] deviatoric stress xx, yy, zz, xy, xz, yz (device, canonical order)
void launch_stress(const DeviceGeometry& g, const void* buf, GatherMode mode, double* sigma,
                   cudaStream_t s);
// wss [N] from sigma [N][6] and normals [N][3] (all device, canonical order)
void launch_wall_shear_stress(const double* sigma, const double* normals, long long N, double* wss,
                              cudaStream_t s);
// The static device scratch of hlb_get_wall_shear_stress_noalloc (include/hlb.h): `max_sites`
// x 6 doubles in a file-scope __device__ array of kernels.cu. noalloc_scratch_setup() takes its
// DEVICE address for the CURRENT device (cudaGetSymbolAddress; the array's name in host code is
// only a host-side stand-in) and remembers it per device; call it at set-up, with the device
// current. noalloc_scratch() returns the remembered address for the current device, or NULL.
constexpr long long NOALLOC_MAX_SITES = 262144;
cudaError_t noalloc_scratch_setup();
double* noalloc_scratch();
// f [N][Q] raw populations (device, canonical order)
void launch_get_populations(const DeviceGeometry& g, const void* buf, GatherMode mode, double* f,
                            cudaStream_t s);
// Initialise a buffer so that gathering in `mode` (GATHER_PULL or GATHER_OWN) yields
//   f_q(x) = f_in[canon(x)][q]                       if f_in != NULL, else
//   f_q(x) = f_eq_q(rho_in[canon(x)], u_in[canon(x)])  (NULL rho => 1, NULL u => 0).
void launch_init(const DeviceGeometry& g, void* buf, GatherMode mode, const double* rho_in,
                 const double* u_in, const double* f_in, cudaStream_t s);

}  // namespace hlb
