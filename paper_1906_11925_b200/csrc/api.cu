// api.cu -- the C-ABI entry points declared in include/hlb.h (argument checking, device
// buffers through the caller's allocator, stream-ordered kernel launches). Every step of
// the hot path runs in the kernels of kernels.cu; nothing here computes on the host.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/hlb.h"
#include "lattice.h"
#include "kernels.cuh"
#include "preprocess.h"
#include "render.cuh"

using namespace hlb;

namespace {
thread_local std::string g_err = "";

int fail(int code, const std::string& msg) {
  g_err = msg;
  return code;
}
int cuda_fail(cudaError_t e, const char* what) {
  g_err = std::string(what) + ": " + cudaGetErrorString(e);
  return HLB_ECUDA;
}
#define HLB_CUDA(call)                                   \
  do {                                                   \
    cudaError_t e__ = (call);                            \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
  } while (0)

SiteOrder order_of(uint32_t flags, bool& ok) {
  ok = true;
  switch (flags & HLB_ORDER_MASK) {
    case HLB_ORDER_AUTO: return ORDER_RASTER;
    case HLB_ORDER_MORTON: return ORDER_MORTON;
    case HLB_ORDER_RASTER: return ORDER_RASTER;
    case HLB_ORDER_TILED: return ORDER_TILED;
  }
  ok = false;
  return ORDER_MORTON;
}
}  // namespace

struct hlb_geometry {
  hlb_params p{};
  cudaStream_t stream = nullptr;
  bool aa = false, f32 = false;
  int Q = 15;                         // populations per site (15 or 19)
  int64_t N = 0, Ns = 0;
  std::vector<int64_t> canon_voxels;  // [N] ascending
  std::vector<double> iolet_rho;
  std::vector<uint8_t> iolet_kind;    // 0 constant density, 1 Ladd velocity
  std::vector<double> iolet_u;        // [n_iolets][3]
  std::vector<double> iolet_n;        // [n_iolets][3] unit normals of density iolets, 0 = none
  std::vector<double> iolet_par;      // [n_iolets][4] as uploaded: {rho or -1, ux, uy, uz}
  double* d_iolet_par = nullptr;      // device copy of iolet_par (dg.iolet_par points here, or
                                      // into d_wave while a waveform is set)
  // hlb_set_iolet_waveform: one [n_iolets][4] slice per time level, the rows of velocity
  // iolets carrying u[t][k]; the step at time t is launched with the slice t mod wave_nt
  std::vector<double> wave_u;         // [wave_nt][n_iolets][3] as given
  std::vector<double> wave_par;       // [wave_nt][n_iolets][4] as uploaded
  int64_t wave_nt = 0;
  double* d_wave = nullptr;
  size_t wave_cap = 0;                // doubles d_wave can hold
  double* d_iolet_w = nullptr;        // [Ns] velocity weights, internal order (hlb_set_iolet_weight)
  DeviceGeometry dg;
  void* buf[2] = {nullptr, nullptr};  // population arrays [15][Ns]; A-A uses buf[0] only
  int cur = 0;                        // two-lattice: buffer the next step reads
  double* scratch = nullptr;          // [4 N] doubles: staging of rho [N], u [N][3] transfers
  cudaStream_t copy_stream = nullptr; // params.copy_stream (hlb_get_macroscopic_async)
  double* scratch_out = nullptr;      // [4 N] doubles: its own staging buffer (lazy), so that an
                                      // upload through `scratch` may overlap the copies
  cudaEvent_t ev_ready = nullptr, ev_copied = nullptr;  // read-out done / copies done
  double* scratch_in = nullptr;       // [4 N] doubles: staging buffer of hlb_stage_state (lazy)
  cudaEvent_t ev_staged = nullptr, ev_consumed = nullptr;  // upload done / init kernel has read it
  bool staged = false, staged_rho = false, staged_u = false;
  double* scratch_pop = nullptr;      // [N][15] doubles, allocated by the first
                                      // hlb_get_populations / hlb_set_populations call
  int64_t steps = 0, launches = 0, device_bytes = 0;
  double sentinel_fraction = 0.0;     // of the (group, q) link records
  // hlb_step(n) replays a captured CUDA graph of GRAPH_STEPS steps while n allows: removes
  // the per-launch host cost that dominates small geometries (BASELINE configs[0], [2])
  float* volume = nullptr;            // [nz][ny][nx] floats for hlb_render (lazy)
  long long* d_voxels = nullptr;      // [N] canonical voxel index on the device (lazy)
  unsigned char* occ = nullptr;       // macro-cell emptiness of the volume (solid cells; lazy)
  cudaArray_t vol_array = nullptr;    // 3-D array copy of the volume behind a point-sampled
  cudaTextureObject_t vol_tex = 0;    // texture object (render_through_texture(); cudaMalloc3DArray,
  cudaSurfaceObject_t vol_surf = 0;   // not the caller's allocator: CUDA arrays are opaque)
  float* d_image = nullptr;           // staging image for hlb_render
  size_t d_image_floats = 0;
  cudaError_t noalloc_setup = cudaSuccess;  // result of noalloc_scratch_setup() at create
  bool bfl_set = false;               // wall distances given (hlb_set_wall_distance)
  int64_t bfl_sites = 0;              // sites with at least one interpolated link
  int64_t bfl_links = 0;              // interpolated links
  void* bfl_mem[7] = {};              // device tables of hlb_set_wall_distance, kept for reuse
  size_t bfl_cap_links = 0, bfl_cap_coef = 0;
  cudaGraphExec_t graph_exec = nullptr;
  bool graph_failed = false;
  // resident multi-step kernel (small geometries; kernels.cuh launch_resident_steps)
  unsigned long long* d_bar = nullptr;  // grid-barrier arrival counter
  unsigned long long bar_base = 0;      // its value once everything enqueued so far has run
  int64_t resident_max_sites = 0;       // Ns up to which the whole grid is resident at once
  bool resident_failed = false;         // a cooperative launch was refused: do not try again
  // The captured launches fix the kernel instantiation and the by-value arguments: drop the
  // graph whenever one of them changes (iolet kinds / normals, wall distances).
  void drop_graph() {
    if (graph_exec) {
      cudaStreamSynchronize(stream);
      cudaGraphExecDestroy(graph_exec);
      graph_exec = nullptr;
    }
  }
  std::vector<void*> owned;           // cudaMalloc'ed (no allocator callback)

  int alloc(size_t bytes, void** out) {
    void* ptr = nullptr;
    if (p.alloc) {
      ptr = p.alloc(bytes, p.alloc_user);
      if (!ptr) return fail(HLB_ENOMEM, "allocator callback returned NULL");
    } else {
      cudaError_t e = cudaMalloc(&ptr, bytes);
      if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? fail(HLB_ENOMEM, "cudaMalloc: out of memory")
                                              : cuda_fail(e, "cudaMalloc");
      }
      owned.push_back(ptr);
    }
    device_bytes += (int64_t)bytes;
    *out = ptr;
    return HLB_OK;
  }
  // Give back a buffer of alloc() that was replaced by a larger one (the stream is idle).
  void release(void* ptr, size_t bytes) {
    if (!ptr) return;
    if (p.alloc) {
      if (!p.free) return;  // stays with the caller until destroy
      p.free(ptr, p.alloc_user);
    } else {
      auto it = std::find(owned.begin(), owned.end(), ptr);
      if (it == owned.end()) return;
      owned.erase(it);
      cudaFree(ptr);
    }
    device_bytes -= (int64_t)bytes;
  }
  size_t store_bytes() const { return f32 ? 4 : 8; }
  GatherMode gather_mode() const {
    if (!aa) return GATHER_PULL;
    return (steps & 1) ? GATHER_AA_ODD : GATHER_OWN;
  }
  const void* state_buf() const { return aa ? buf[0] : buf[cur]; }
  // The BFL interpolation belongs to the propagation. Its d >= 1/2 part is in what the step
  // kernels write; its d < 1/2 part is applied to every state when it is gathered from --
  // by the next step kernel in registers (gather_bfl()), or, before a read-out, once by a
  // pre-pass that rewrites the bounce-back slots in the state buffer (ensure_bfl()) -- except
  // to the freshly initialised state f(., 0), which is given, not propagated.
  bool bfl_applied = false;  // the pre-pass has run on the current state buffer
  bool gather_bfl() const { return bfl_set && steps > 0 && !bfl_applied; }
  void ensure_bfl() {
    if (bfl_set && steps > 0 && !bfl_applied) {
      launch_bfl_prepass(dg, aa ? buf[0] : buf[cur], gather_mode(), stream);
      bfl_applied = true;
      if (dg.bfl.n > 0) ++launches;
    }
  }
};

extern "C" {

const char* hlb_last_error(void) { return g_err.c_str(); }

int hlb_lattice(uint32_t flags, int32_t* c, double* w, int32_t* o) {
  const LatticeDesc& lat = lattice_desc((flags & HLB_LATTICE_D3Q19) != 0);
  for (int q = 0; q < lat.Q; ++q) {
    if (c) { c[3 * q + 0] = lat.c[q][0]; c[3 * q + 1] = lat.c[q][1]; c[3 * q + 2] = lat.c[q][2]; }
    if (w) w[q] = lat.w[q];
    if (o) o[q] = opp(q);
  }
  return lat.Q;
}
void hlb_velocity_set(int32_t* c, double* w, int32_t* o) { (void)hlb_lattice(0, c, w, o); }

static int check_params(const uint8_t* site_type, const hlb_params* p, SiteOrder& order) {
  if (!site_type || !p) return fail(HLB_EINVAL, "NULL argument");
  if (p->nx <= 0 || p->ny <= 0 || p->nz <= 0) return fail(HLB_EINVAL, "non-positive box extent");
  if (p->n_iolets < 0 || p->n_iolets > 253) return fail(HLB_EINVAL, "n_iolets must be in 0..253");
  if (p->n_iolets > 0 && !p->iolet_rho) return fail(HLB_EINVAL, "iolet_rho is NULL");
  for (int k = 0; k < p->n_iolets; ++k)
    if (!(p->iolet_rho[k] > 0.0)) return fail(HLB_EINVAL, "iolet densities must be positive");
  if (p->periodic & ~7u) return fail(HLB_EINVAL, "unknown periodic bits");
  if (p->flags & ~(uint32_t)(HLB_STORE_F32 | HLB_AA | HLB_ORDER_MASK | HLB_NO_GRAPH |
                             HLB_LINKS_TABLE | HLB_LINKS_RECORDS | HLB_NO_PREFETCH | HLB_INDEX64 |
                             HLB_LATTICE_D3Q19 | HLB_NO_PDL | HLB_NO_RESIDENT | HLB_SCHEME_AUTO))
    return fail(HLB_EINVAL, "unknown flag bits");
  if ((p->flags & HLB_LINKS_TABLE) && (p->flags & HLB_LINKS_RECORDS))
    return fail(HLB_EINVAL, "HLB_LINKS_TABLE and HLB_LINKS_RECORDS are exclusive");
  bool ok;
  order = order_of(p->flags, ok);
  if (!ok) return fail(HLB_EINVAL, "unknown HLB_ORDER_* value");
  return HLB_OK;
}

int hlb_preprocess_count(const uint8_t* site_type, const hlb_params* p, int64_t* n_sites,
                         int64_t* stride) {
  SiteOrder order;
  int rc = check_params(site_type, p, order);
  if (rc) return rc;
  GeometryTables t;
  std::string err;
  rc = preprocess(site_type, p->nx, p->ny, p->nz, p->periodic, p->n_iolets, order,
                  lattice_desc((p->flags & HLB_LATTICE_D3Q19) != 0), true, t, err);
  if (rc) return fail(rc, err);
  if (n_sites) *n_sites = t.N;
  if (stride) *stride = t.Ns;
  return HLB_OK;
}

int hlb_preprocess_tables(const uint8_t* site_type, const hlb_params* p, int64_t* voxel_of_site,
                          int32_t* canon_of_site, int32_t* nbr) {
  SiteOrder order;
  int rc = check_params(site_type, p, order);
  if (rc) return rc;
  GeometryTables t;
  std::string err;
  rc = preprocess(site_type, p->nx, p->ny, p->nz, p->periodic, p->n_iolets, order,
                  lattice_desc((p->flags & HLB_LATTICE_D3Q19) != 0), false, t, err);
  if (rc) return fail(rc, err);
  if (voxel_of_site) std::memcpy(voxel_of_site, t.voxel_of_site.data(), sizeof(int64_t) * (size_t)t.N);
  if (canon_of_site) std::memcpy(canon_of_site, t.canon_of_site.data(), sizeof(int32_t) * (size_t)t.N);
  if (nbr) std::memcpy(nbr, t.nbr.data(), sizeof(int32_t) * t.nbr.size());
  return HLB_OK;
}

// {rho_k, nx, ny, nz} for a constant-density iolet, {-1, ux, uy, uz} for a velocity iolet
static int upload_iolets(hlb_geometry* g) {
  const int n = g->p.n_iolets;
  if (n == 0) return HLB_OK;
  HLB_CUDA(cudaStreamSynchronize(g->stream));  // the previous upload may still read iolet_par
  g->iolet_par.assign((size_t)n * 4, 0.0);
  const bool was_full = g->dg.iolet_full;
  g->dg.iolet_full = false;
  for (int k = 0; k < n; ++k) {
    if (g->iolet_kind[(size_t)k] == 1 || g->iolet_n[(size_t)k * 3] != 0.0 ||
        g->iolet_n[(size_t)k * 3 + 1] != 0.0 || g->iolet_n[(size_t)k * 3 + 2] != 0.0)
      g->dg.iolet_full = true;
    if (g->iolet_kind[(size_t)k] == 1) {
      g->iolet_par[(size_t)k * 4] = -1.0;
      for (int a = 0; a < 3; ++a) g->iolet_par[(size_t)k * 4 + 1 + a] = g->iolet_u[(size_t)k * 3 + a];
    } else {
      g->iolet_par[(size_t)k * 4] = g->iolet_rho[(size_t)k];
      for (int a = 0; a < 3; ++a) g->iolet_par[(size_t)k * 4 + 1 + a] = g->iolet_n[(size_t)k * 3 + a];
    }
  }
  if (g->dg.iolet_full != was_full) g->drop_graph();  // another instantiation of the step kernels
  HLB_CUDA(cudaMemcpyAsync(g->d_iolet_par, g->iolet_par.data(), sizeof(double) * 4 * (size_t)n,
                           cudaMemcpyHostToDevice, g->stream));
  if (g->wave_nt > 0) {
    // every time level is the slice above with the velocity rows replaced by u[t][k]
    const size_t slice = 4 * (size_t)n, total = slice * (size_t)g->wave_nt;
    if (total > g->wave_cap) {
      void* ptr = nullptr;
      const int rc = g->alloc(sizeof(double) * total, &ptr);
      if (rc) return rc;
      g->release(g->d_wave, sizeof(double) * g->wave_cap);  // (the stream was synchronised above)
      g->d_wave = (double*)ptr;
      g->wave_cap = total;
    }
    g->wave_par.resize(total);
    for (int64_t t = 0; t < g->wave_nt; ++t) {
      double* row = g->wave_par.data() + (size_t)t * slice;
      std::memcpy(row, g->iolet_par.data(), sizeof(double) * slice);
      for (int k = 0; k < n; ++k)
        if (g->iolet_kind[(size_t)k] == 1)
          for (int a = 0; a < 3; ++a)
            row[(size_t)k * 4 + 1 + a] = g->wave_u[((size_t)t * (size_t)n + (size_t)k) * 3 + (size_t)a];
    }
    HLB_CUDA(cudaMemcpyAsync(g->d_wave, g->wave_par.data(), sizeof(double) * total,
                             cudaMemcpyHostToDevice, g->stream));
  }
  return HLB_OK;
}

int hlb_preprocess_records(const int32_t* nbr, int32_t n_links, int64_t stride, uint32_t* rec,
                           int64_t* n_sentinel) {
  if (!nbr || !rec) return fail(HLB_EINVAL, "NULL argument");
  if (n_links != 14 && n_links != 18) return fail(HLB_EINVAL, "n_links must be 14 (D3Q15) or 18 (D3Q19)");
  if (stride <= 0 || stride % 32) return fail(HLB_EINVAL, "stride must be a positive multiple of 32");
  const int64_t n = build_link_records(nbr, n_links, stride, rec);
  if (n_sentinel) *n_sentinel = n;
  return HLB_OK;
}

int hlb_preprocess_bfl(const int32_t* nbr, const int32_t* canon_of_site, int32_t n_links, int64_t n_sites,
                       int64_t stride, const double* d27, uint32_t* index, double* coef, int64_t coef_rows,
                       int64_t* n_flagged, int64_t* n_interpolated) {
  if (!nbr || !canon_of_site || !d27) return fail(HLB_EINVAL, "NULL argument");
  if (n_links != 14 && n_links != 18) return fail(HLB_EINVAL, "n_links must be 14 (D3Q15) or 18 (D3Q19)");
  if (stride <= 0 || stride % 32 || n_sites < 0 || n_sites > stride)
    return fail(HLB_EINVAL, "stride must be a positive multiple of 32 and at least n_sites");
  BflTables bt;
  build_bfl_tables(nbr, canon_of_site, n_links + 1, n_sites, stride, d27, bt);
  if (n_flagged) *n_flagged = bt.n_sites;
  if (n_interpolated) *n_interpolated = (int64_t)bt.site.size();
  if (index) std::memcpy(index, bt.index.data(), sizeof(uint32_t) * bt.index.size());
  if (coef) {
    if (coef_rows < bt.n_sites) return fail(HLB_EINVAL, "coef_rows is smaller than the number of flagged sites");
    std::memcpy(coef, bt.coef.data(), sizeof(double) * bt.row * (size_t)bt.n_sites);
  }
  return HLB_OK;
}

int hlb_geometry_create(const uint8_t* site_type, const hlb_params* p, hlb_geometry** out) {
  if (out) *out = nullptr;
  if (!out) return fail(HLB_EINVAL, "out is NULL");
  SiteOrder order;
  int rc = check_params(site_type, p, order);
  if (rc) return rc;
  if (!(p->tau > 0.5)) return fail(HLB_EINVAL, "tau must be > 0.5");
  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev == 0) {
    (void)cudaGetLastError();
    return fail(HLB_ECUDA, "no CUDA device: the site update has no CPU fallback");
  }
  GeometryTables t;
  std::string err;
  rc = preprocess(site_type, p->nx, p->ny, p->nz, p->periodic, p->n_iolets, order,
                  lattice_desc((p->flags & HLB_LATTICE_D3Q19) != 0), false, t, err);
  if (rc) return fail(rc, err);

  hlb_geometry* g = new hlb_geometry();
  g->p = *p;
  g->p.iolet_rho = nullptr;
  g->stream = (cudaStream_t)p->stream;
  g->copy_stream = (cudaStream_t)p->copy_stream;
  g->aa = (p->flags & HLB_AA) != 0;
  if (p->flags & HLB_SCHEME_AUTO) {
    // A-A in place (half the launches read no links; one array in L2 for the mid sizes) except
    //  * where the resident multi-step kernel applies: two-lattice is the faster one there
    //    (5.4 k vs 5.0 k MSUPS on configs[0]);
    //  * where the whole grid is ONE wave of the two-lattice kernel (5 % slack) but more than
    //    one wave of the A-A kernels, i.e. where the two-lattice kernel has the larger register
    //    budget in blocks per SM (D3Q19: 5 against 4): the second, nearly empty wave costs A-A
    //    8-20 % there.
    // profiles/r02_tuning.md section 7.
    int dev = 0, sms = 0;
    const bool have = cudaGetDevice(&dev) == cudaSuccess &&
                      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess;
    const bool q19 = (p->flags & HLB_LATTICE_D3Q19) != 0;
    const int64_t blocks = t.Ns / 128;
    const int64_t slots_pull = (int64_t)sms * resident_sites_per_sm_pull(q19, (p->flags & HLB_STORE_F32) != 0) / 128;
    const int64_t slots_aa = (int64_t)sms * resident_sites_per_sm_aa(q19, (p->flags & HLB_STORE_F32) != 0) / 128;
    const bool resident = have && !(p->flags & (HLB_NO_GRAPH | HLB_NO_RESIDENT)) &&
                          t.Ns <= (int64_t)sms * resident_kernel_sites_per_sm();
    const bool one_pull_wave = have && blocks > slots_aa && blocks * 100 <= slots_pull * 105;
    g->aa = !(resident || one_pull_wave);
  }
  g->f32 = (p->flags & HLB_STORE_F32) != 0;
  g->Q = (p->flags & HLB_LATTICE_D3Q19) ? 19 : 15;
  const int Q = g->Q;
  g->N = t.N;
  g->Ns = t.Ns;
  g->iolet_rho.assign(p->iolet_rho, p->iolet_rho + p->n_iolets);
  g->iolet_kind.assign((size_t)p->n_iolets, 0);
  g->iolet_u.assign((size_t)p->n_iolets * 3, 0.0);
  g->iolet_n.assign((size_t)p->n_iolets * 3, 0.0);
  g->canon_voxels.resize((size_t)t.N);
  for (int64_t i = 0; i < t.N; ++i) g->canon_voxels[(size_t)t.canon_of_site[(size_t)i]] = t.voxel_of_site[(size_t)i];

  void *d_nbr = nullptr, *d_bits = nullptr, *d_canon = nullptr, *d_rho = nullptr, *d_scratch = nullptr;
  void *d_rec = nullptr, *d_iolinks = nullptr;
  g->sentinel_fraction = (double)t.n_rec_fallback / (double)((t.Ns / 32) * (Q - 1));
  const bool use_rec = (p->flags & HLB_LINKS_RECORDS) ? true
                       : (p->flags & HLB_LINKS_TABLE) ? false
                                                      : g->sentinel_fraction <= 0.5;
  if (!(p->flags & HLB_NO_PREFETCH)) {
    // L2 prefetch distance: 3/4 of the sites resident on the chip (measured optimum on
    // B200: 0.6 .. 0.9, profiles/r01_tuning.md). HLB_PREFETCH_SITES overrides it (tuning).
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
      cuda_fail(cudaGetLastError(), "cudaDeviceGetAttribute");
      delete g;
      return HLB_ECUDA;
    }
    // The distance is one in BYTES per plane: with 4-byte populations twice as many sites
    // (same-box sweep of the fp32-storage kernels: 0.82 / 1.00 ms at this many sites, 0.72 /
    // 0.97 ms at twice as many; profiles/r02_tuning.md).
    const int64_t per8 = g->f32 ? 2 : 1;
    g->dg.prefetch_pull = (int64_t)sms * resident_sites_per_sm_pull(Q == 19, g->f32) * 3 / 4 / 128 * 128 * per8;
    g->dg.prefetch_aa = (int64_t)sms * resident_sites_per_sm_aa(Q == 19, g->f32) * 3 / 4 / 128 * 128 * per8;
    // A state that fits half of the L2 stays there from step to step: the prefetches are then
    // only instructions (296 k sites, A-A: 10.54 -> 10.05 us per step without them, D3Q19 13.18 ->
    // 12.61; at 89 MB of state, configs[2] in place, no difference; beyond, they pay:
    // profiles/r02_tuning.md section 18).
    {
      int l2 = 0;
      const size_t state_bytes = (size_t)Q * (size_t)t.Ns * g->store_bytes() * (g->aa ? 1 : 2);
      if (cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev) == cudaSuccess && l2 > 0 &&
          state_bytes <= (size_t)l2 / 2)
        g->dg.prefetch_pull = g->dg.prefetch_aa = 0;
      else
        (void)cudaGetLastError();
    }
    if (const char* e = std::getenv("HLB_PREFETCH_SITES")) {
      const long long v = std::atoll(e);
      g->dg.prefetch_pull = g->dg.prefetch_aa = v > 0 ? (v < (1ll << 24) ? v : (1ll << 24)) : 0;
    }
  }
  // tail padding: a prefetch reaches at most `distance` elements past the last plane
  const size_t pad_bytes =
      (size_t)std::max(g->dg.prefetch_pull, g->dg.prefetch_aa) * g->store_bytes();
  const size_t pop_bytes = (size_t)Q * (size_t)t.Ns * g->store_bytes();
  auto bail = [&](int code) { hlb_geometry_destroy(g); return code; };
  if ((rc = g->alloc(sizeof(int32_t) * t.nbr.size(), &d_nbr))) return bail(rc);
  if ((rc = g->alloc(sizeof(uint32_t) * t.iolet_idx.size(), &d_bits))) return bail(rc);
  if ((rc = g->alloc(t.iolet_links.size(), &d_iolinks))) return bail(rc);
  if (use_rec && (rc = g->alloc(sizeof(uint32_t) * t.rec.size(), &d_rec))) return bail(rc);
  if ((rc = g->alloc(sizeof(int32_t) * (size_t)t.N, &d_canon))) return bail(rc);
  if ((rc = g->alloc(sizeof(double) * 4 * (size_t)(p->n_iolets > 0 ? p->n_iolets : 1), &d_rho))) return bail(rc);
  if ((rc = g->alloc(pop_bytes + pad_bytes, &g->buf[0]))) return bail(rc);
  if (!g->aa && (rc = g->alloc(pop_bytes + pad_bytes, &g->buf[1]))) return bail(rc);
  if ((rc = g->alloc(sizeof(double) * 4 * (size_t)t.N, &d_scratch))) return bail(rc);
  g->scratch = (double*)d_scratch;
  {
    int dev = 0, sms = 0, coop = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop) {
      void* d_bar = nullptr;
      if ((rc = g->alloc(256, &d_bar))) return bail(rc);
      g->d_bar = (unsigned long long*)d_bar;
      g->resident_max_sites = (int64_t)sms * resident_kernel_sites_per_sm();
    } else {
      (void)cudaGetLastError();
    }
  }

#define HLB_CUDA_G(call)                                                   \
  do {                                                                     \
    cudaError_t e__ = (call);                                              \
    if (e__ != cudaSuccess) { cuda_fail(e__, #call); return bail(HLB_ECUDA); } \
  } while (0)
  HLB_CUDA_G(cudaMemcpyAsync(d_nbr, t.nbr.data(), sizeof(int32_t) * t.nbr.size(), cudaMemcpyHostToDevice, g->stream));
  HLB_CUDA_G(cudaMemcpyAsync(d_bits, t.iolet_idx.data(), sizeof(uint32_t) * t.iolet_idx.size(), cudaMemcpyHostToDevice, g->stream));
  HLB_CUDA_G(cudaMemcpyAsync(d_iolinks, t.iolet_links.data(), t.iolet_links.size(), cudaMemcpyHostToDevice, g->stream));
  if (use_rec)
    HLB_CUDA_G(cudaMemcpyAsync(d_rec, t.rec.data(), sizeof(uint32_t) * t.rec.size(), cudaMemcpyHostToDevice, g->stream));
  if (g->d_bar) HLB_CUDA_G(cudaMemsetAsync(g->d_bar, 0, 256, g->stream));
  HLB_CUDA_G(cudaMemcpyAsync(d_canon, t.canon_of_site.data(), sizeof(int32_t) * (size_t)t.N, cudaMemcpyHostToDevice, g->stream));
  g->d_iolet_par = (double*)d_rho;
  g->dg.iolet_par = g->d_iolet_par;
  if ((rc = upload_iolets(g))) return bail(rc);
  g->dg.N = t.N;
  g->dg.Ns = t.Ns;
  g->dg.nbr = (const int32_t*)d_nbr;
  g->dg.iolet_idx = d_bits;
  g->dg.iolet_links = d_iolinks;
  g->dg.rec = d_rec;
  g->dg.use_rec = use_rec;
  g->dg.pdl = !(p->flags & HLB_NO_PDL);
  g->dg.index64 = (p->flags & HLB_INDEX64) != 0 || (int64_t)Q * t.Ns >= ((int64_t)1 << 32);
  g->dg.canon = (const int32_t*)d_canon;
  g->dg.omega = 1.0 / p->tau;
  g->dg.f32 = g->f32;
  g->dg.d3q19 = Q == 19;
  // set-up of the static scratch of hlb_get_wall_shear_stress_noalloc: its device address, once
  // per device, with this geometry's device current (kept, not fatal: only that call needs it)
  g->noalloc_setup = noalloc_scratch_setup();
  if (g->noalloc_setup != cudaSuccess) (void)cudaGetLastError();
  // the host tables die at the end of this call: finish the uploads first
  HLB_CUDA_G(cudaStreamSynchronize(g->stream));
  rc = hlb_set_state(g, nullptr, nullptr);
  if (rc) return bail(rc);
  HLB_CUDA_G(cudaStreamSynchronize(g->stream));
#undef HLB_CUDA_G
  *out = g;
  return HLB_OK;
}

void hlb_geometry_destroy(hlb_geometry* g) {
  if (!g) return;
  if (g->graph_exec) cudaGraphExecDestroy(g->graph_exec);
  if (g->ev_ready || g->ev_staged) cudaStreamSynchronize(g->copy_stream);
  if (g->ev_ready) {
    cudaEventDestroy(g->ev_ready);
    cudaEventDestroy(g->ev_copied);
  }
  if (g->ev_staged) {
    cudaEventDestroy(g->ev_staged);
    cudaEventDestroy(g->ev_consumed);
  }
  if (g->vol_array) {
    cudaStreamSynchronize(g->stream);
    if (g->vol_tex) cudaDestroyTextureObject(g->vol_tex);
    if (g->vol_surf) cudaDestroySurfaceObject(g->vol_surf);
    cudaFreeArray(g->vol_array);
  }
  if (!g->owned.empty()) {
    cudaStreamSynchronize(g->stream);
    for (void* ptr : g->owned) cudaFree(ptr);
  }
  delete g;
}

static int init_from(hlb_geometry* g, const double* d_rho, const double* d_u, const double* d_f) {
  const GatherMode mode = g->aa ? GATHER_OWN : GATHER_PULL;
  g->cur = 0;
  g->steps = 0;
  g->bfl_applied = false;
  launch_init(g->dg, g->buf[0], mode, d_rho, d_u, d_f, g->stream);
  HLB_CUDA(cudaGetLastError());
  return HLB_OK;
}

static int ensure_scratch_pop(hlb_geometry* g) {
  if (g->scratch_pop) return HLB_OK;
  void* ptr = nullptr;
  const int rc = g->alloc(sizeof(double) * (size_t)g->Q * (size_t)g->N, &ptr);
  if (rc) return rc;
  g->scratch_pop = (double*)ptr;
  return HLB_OK;
}

int hlb_set_state(hlb_geometry* g, const double* rho, const double* u) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  double *d_rho = nullptr, *d_u = nullptr;
  const size_t n = (size_t)g->N;
  if (rho) {
    d_rho = g->scratch;
    HLB_CUDA(cudaMemcpyAsync(d_rho, rho, sizeof(double) * n, cudaMemcpyHostToDevice, g->stream));
  }
  if (u) {
    d_u = g->scratch + n;
    HLB_CUDA(cudaMemcpyAsync(d_u, u, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, g->stream));
  }
  const int rc = init_from(g, d_rho, d_u, nullptr);
  // the caller may reuse or free rho / u as soon as this returns (pinned memory makes the
  // copies truly asynchronous)
  if (!rc && (rho || u)) HLB_CUDA(cudaStreamSynchronize(g->stream));
  return rc;
}

int hlb_set_populations(hlb_geometry* g, const double* f) {
  if (!g || !f) return fail(HLB_EINVAL, "NULL argument");
  int rc = ensure_scratch_pop(g);
  if (rc) return rc;
  HLB_CUDA(cudaMemcpyAsync(g->scratch_pop, f, sizeof(double) * (size_t)g->Q * (size_t)g->N, cudaMemcpyHostToDevice, g->stream));
  rc = init_from(g, nullptr, nullptr, g->scratch_pop);
  if (!rc) HLB_CUDA(cudaStreamSynchronize(g->stream));  // f has been read when this returns
  return rc;
}

int hlb_set_iolet_density(hlb_geometry* g, const double* iolet_rho) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (g->p.n_iolets == 0) return HLB_OK;
  if (!iolet_rho) return fail(HLB_EINVAL, "iolet_rho is NULL");
  for (int k = 0; k < g->p.n_iolets; ++k)
    if (!(iolet_rho[k] > 0.0)) return fail(HLB_EINVAL, "iolet densities must be positive");
  g->iolet_rho.assign(iolet_rho, iolet_rho + g->p.n_iolets);
  return upload_iolets(g);
}

int hlb_set_iolet_normal(hlb_geometry* g, const double* normals) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  const int n = g->p.n_iolets;
  for (int k = 0; k < n; ++k) {
    double v[3] = {0.0, 0.0, 0.0};
    if (normals) {
      const double* s = normals + k * 3;
      const double len = std::sqrt(s[0] * s[0] + s[1] * s[1] + s[2] * s[2]);
      if (len > 0.0) { v[0] = s[0] / len; v[1] = s[1] / len; v[2] = s[2] / len; }
    }
    for (int a = 0; a < 3; ++a) g->iolet_n[(size_t)k * 3 + a] = v[a];
  }
  return upload_iolets(g);
}

int hlb_set_wall_distance(hlb_geometry* g, const double* d27) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (g->steps != 0) return fail(HLB_EINVAL, "set the wall distances before the first step (steps_done == 0)");
  g->drop_graph();
  if (!d27) {
    g->bfl_set = false;
    g->dg.bfl = BflLinks();
    const double* keep_w = g->dg.bflf.iolet_w;  // the velocity weights travel in the same argument
    g->dg.bflf = BflFused();
    g->dg.bflf.iolet_w = keep_w;
    g->dg.bfl_on = false;
    return HLB_OK;
  }
  const int Q = g->Q;
  const int64_t N = g->N, Ns = g->Ns;
  // the link table and the canonical ranks live on the device only: fetch them
  std::vector<int32_t> nbr((size_t)(Q - 1) * (size_t)Ns), canon((size_t)N);
  HLB_CUDA(cudaStreamSynchronize(g->stream));
  HLB_CUDA(cudaMemcpy(nbr.data(), g->dg.nbr, sizeof(int32_t) * nbr.size(), cudaMemcpyDeviceToHost));
  HLB_CUDA(cudaMemcpy(canon.data(), g->dg.canon, sizeof(int32_t) * canon.size(), cudaMemcpyDeviceToHost));
  BflTables bt;
  build_bfl_tables(nbr.data(), canon.data(), Q, N, Ns, d27, bt);
  if (bt.row != (size_t)bfl_row_doubles(Q == 19)) return fail(HLB_EINVAL, "internal: BFL row size mismatch");
  const int64_t n_sites = bt.n_sites;
  const size_t nf = bt.nf;
  const std::vector<double>& coef = bt.coef;
  const std::vector<int32_t>& a_site = bt.site;
  // list form for the read-out pre-pass: the links with d < 1/2 only (the others are already
  // in what the step kernels write)
  std::vector<int32_t> l_site, l_behind;
  std::vector<uint8_t> l_link;
  std::vector<double> l_d;
  for (size_t l = 0; l < bt.site.size(); ++l)
    if (bt.d[l] < 0.5) {
      l_site.push_back(bt.site[l]);
      l_behind.push_back(bt.behind[l]);
      l_link.push_back(bt.link[l]);
      l_d.push_back(bt.d[l]);
    }
  const size_t nl = l_site.size();
  void *d_site = nullptr, *d_behind = nullptr, *d_link = nullptr, *d_d = nullptr;
  void *d_bits = nullptr, *d_rank = nullptr, *d_coef = nullptr;
  int rc;
  const size_t cap = nl > 0 ? nl : 1;
  if (g->bfl_mem[0] && cap <= g->bfl_cap_links && coef.size() <= g->bfl_cap_coef) {
    // tables of an earlier call are large enough: reuse them
    d_site = g->bfl_mem[0]; d_behind = g->bfl_mem[1]; d_link = g->bfl_mem[2]; d_d = g->bfl_mem[3];
    d_bits = g->bfl_mem[4]; d_rank = g->bfl_mem[5]; d_coef = g->bfl_mem[6];
    HLB_CUDA(cudaStreamSynchronize(g->stream));
  } else {
    if ((rc = g->alloc(sizeof(int32_t) * cap, &d_site))) return rc;
    if ((rc = g->alloc(sizeof(int32_t) * cap, &d_behind))) return rc;
    if ((rc = g->alloc(sizeof(uint8_t) * cap, &d_link))) return rc;
    if ((rc = g->alloc(sizeof(double) * cap, &d_d))) return rc;
    if ((rc = g->alloc(sizeof(uint32_t) * bt.index.size(), &d_bits))) return rc;  // {bits, rank} words
    if ((rc = g->alloc(sizeof(double) * coef.size(), &d_coef))) return rc;
    void* mem[7] = {d_site, d_behind, d_link, d_d, d_bits, d_rank, d_coef};
    if (g->bfl_mem[0]) {  // smaller tables of an earlier call
      HLB_CUDA(cudaStreamSynchronize(g->stream));
      const size_t old_bytes[7] = {sizeof(int32_t) * g->bfl_cap_links, sizeof(int32_t) * g->bfl_cap_links,
                                   sizeof(uint8_t) * g->bfl_cap_links, sizeof(double) * g->bfl_cap_links,
                                   sizeof(uint32_t) * bt.index.size(), 0,
                                   sizeof(double) * g->bfl_cap_coef};
      for (int k = 0; k < 7; ++k) g->release(g->bfl_mem[k], old_bytes[k]);
    }
    for (int k = 0; k < 7; ++k) g->bfl_mem[k] = mem[k];
    g->bfl_cap_links = cap;
    g->bfl_cap_coef = coef.size();
  }
  if (nl > 0) {
    HLB_CUDA(cudaMemcpy(d_site, l_site.data(), sizeof(int32_t) * nl, cudaMemcpyHostToDevice));
    HLB_CUDA(cudaMemcpy(d_behind, l_behind.data(), sizeof(int32_t) * nl, cudaMemcpyHostToDevice));
    HLB_CUDA(cudaMemcpy(d_link, l_link.data(), sizeof(uint8_t) * nl, cudaMemcpyHostToDevice));
    HLB_CUDA(cudaMemcpy(d_d, l_d.data(), sizeof(double) * nl, cudaMemcpyHostToDevice));
  }
  HLB_CUDA(cudaMemcpy(d_bits, bt.index.data(), sizeof(uint32_t) * bt.index.size(), cudaMemcpyHostToDevice));
  HLB_CUDA(cudaMemcpy(d_coef, coef.data(), sizeof(double) * coef.size(), cudaMemcpyHostToDevice));
  g->dg.bfl.site = (const int32_t*)d_site;
  g->dg.bfl.behind = (const int32_t*)d_behind;
  g->dg.bfl.link = (const uint8_t*)d_link;
  g->dg.bfl.d = (const double*)d_d;
  g->dg.bfl.n = (long long)nl;
  g->dg.bflf.idx = (const uint2*)d_bits;
  g->dg.bflf.coef = (const double*)d_coef;
  g->dg.bflf.nf = (long long)nf;
  g->dg.bflf.gather = 0;
  g->dg.bfl_on = true;
  g->bfl_set = true;
  g->bfl_applied = false;
  g->bfl_sites = n_sites;
  g->bfl_links = (int64_t)a_site.size();
  return HLB_OK;
}

int64_t hlb_num_bfl_sites(const hlb_geometry* g) { return g ? (g->bfl_set ? g->bfl_sites : 0) : (int64_t)HLB_EINVAL; }

int hlb_set_iolet_velocity(hlb_geometry* g, const uint8_t* kind, const double* u) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  const int n = g->p.n_iolets;
  if (n == 0) return HLB_OK;
  for (int k = 0; k < n; ++k) {
    if (kind && kind[k] > 1) return fail(HLB_EINVAL, "iolet kind must be 0 (density) or 1 (velocity)");
    if (kind && kind[k] == 1 && !u) return fail(HLB_EINVAL, "u is NULL but a velocity iolet is requested");
  }
  for (int k = 0; k < n; ++k) {
    g->iolet_kind[(size_t)k] = kind ? kind[k] : 0;
    for (int a = 0; a < 3; ++a) g->iolet_u[(size_t)k * 3 + a] = u ? u[k * 3 + a] : 0.0;
  }
  return upload_iolets(g);
}

int hlb_set_iolet_weight(hlb_geometry* g, const double* weight) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (!weight) {
    if (g->dg.bflf.iolet_w) g->drop_graph();  // captured launches carry the pointer
    g->dg.bflf.iolet_w = nullptr;
    return HLB_OK;
  }
  const size_t N = (size_t)g->N, Ns = (size_t)g->Ns;
  for (size_t c = 0; c < N; ++c)
    if (!std::isfinite(weight[c])) return fail(HLB_EINVAL, "non-finite velocity weight");
  if (!g->d_iolet_w) {
    void* ptr = nullptr;
    const int rc = g->alloc(sizeof(double) * Ns, &ptr);
    if (rc) return rc;
    g->d_iolet_w = (double*)ptr;
  }
  // canonical -> internal order (the ranks live on the device only: fetch them)
  std::vector<int32_t> canon(N);
  HLB_CUDA(cudaStreamSynchronize(g->stream));
  HLB_CUDA(cudaMemcpy(canon.data(), g->dg.canon, sizeof(int32_t) * N, cudaMemcpyDeviceToHost));
  std::vector<double> w(Ns, 1.0);
  host_parallel_for((int64_t)N, 1 << 18, [&](int64_t b, int64_t e) {
    for (int64_t i = b; i < e; ++i) w[(size_t)i] = weight[(size_t)canon[(size_t)i]];
  });
  HLB_CUDA(cudaMemcpy(g->d_iolet_w, w.data(), sizeof(double) * Ns, cudaMemcpyHostToDevice));
  if (g->dg.bflf.iolet_w != g->d_iolet_w) g->drop_graph();
  g->dg.bflf.iolet_w = g->d_iolet_w;
  return HLB_OK;
}

int hlb_set_iolet_waveform(hlb_geometry* g, const double* u, int64_t n_t) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (n_t < 0) return fail(HLB_EINVAL, "n_t < 0");
  const int n = g->p.n_iolets;
  if (n_t > 0 && n == 0) return fail(HLB_EINVAL, "a waveform needs at least one iolet");
  g->drop_graph();
  if (!u || n_t == 0) {
    g->wave_nt = 0;
    g->wave_u.clear();
    return HLB_OK;
  }
  const size_t count = (size_t)n_t * (size_t)n * 3;
  for (size_t j = 0; j < count; ++j)
    if (!std::isfinite(u[j])) return fail(HLB_EINVAL, "non-finite waveform velocity");
  HLB_CUDA(cudaStreamSynchronize(g->stream));  // an earlier upload may still read wave_par
  g->wave_u.assign(u, u + count);
  g->wave_nt = n_t;
  const int rc = upload_iolets(g);
  if (rc) {
    g->wave_nt = 0;
    g->wave_u.clear();
  }
  return rc;
}

constexpr int64_t GRAPH_STEPS = 32;  // even: the buffer / phase parity is back where it started

static void enqueue_one_step(hlb_geometry* g) {
  g->dg.bflf.gather = g->gather_bfl() ? 1 : 0;
  // the iolet parameters of this time level (hlb_set_iolet_waveform), else the constant ones
  g->dg.iolet_par = g->wave_nt > 0
                        ? g->d_wave + (size_t)(g->steps % g->wave_nt) * 4 * (size_t)g->p.n_iolets
                        : g->d_iolet_par;
  if (g->aa) {
    launch_aa(g->dg, g->buf[0], (g->steps & 1) != 0, g->stream);
    g->bfl_applied = false;  // every slot has been rewritten in place
  } else {
    launch_pull(g->dg, g->buf[g->cur], g->buf[g->cur ^ 1], g->stream);
    g->bfl_applied = false;  // the new state buffer is untouched
    g->cur ^= 1;
  }
  ++g->steps;
  ++g->launches;
}

// Capture GRAPH_STEPS steps starting at even parity (two-lattice: cur == 0; A-A: even
// phase). Any failure just disables the graph path: the direct launches are equivalent.
static void build_step_graph(hlb_geometry* g) {
  cudaGraph_t graph = nullptr;
  const int64_t steps0 = g->steps, launches0 = g->launches;
  const int cur0 = g->cur;
  if (cudaStreamBeginCapture(g->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    (void)cudaGetLastError();
    g->graph_failed = true;
    return;
  }
  for (int64_t s = 0; s < GRAPH_STEPS; ++s) enqueue_one_step(g);
  const cudaError_t e = cudaStreamEndCapture(g->stream, &graph);
  g->steps = steps0;
  g->launches = launches0;
  g->cur = cur0;
  if (e != cudaSuccess || !graph ||
      cudaGraphInstantiate(&g->graph_exec, graph, 0) != cudaSuccess) {
    (void)cudaGetLastError();
    g->graph_exec = nullptr;
    g->graph_failed = true;
  }
  if (graph) cudaGraphDestroy(graph);
}

int hlb_step(hlb_geometry* g, int64_t n) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (n < 0) return fail(HLB_EINVAL, "n < 0");
  // graphs pay off only when a step is short next to the launch cost
  // (a captured launch carries its arguments: not with a waveform, whose slice changes per step)
  const bool want_graph = !(g->p.flags & HLB_NO_GRAPH) && !g->graph_failed && g->stream != nullptr &&
                          g->N <= (int64_t)4 << 20 && g->wave_nt == 0;
  // small geometry: all n steps in one cooperative launch of the resident kernel
  if (n >= 2 && g->d_bar && !(g->p.flags & (HLB_NO_GRAPH | HLB_NO_RESIDENT)) && !g->resident_failed &&
      !g->bfl_set && g->wave_nt == 0 && g->Ns <= g->resident_max_sites) {
    g->dg.iolet_par = g->d_iolet_par;
    const cudaError_t e = launch_resident_steps(
        g->dg, g->aa, g->aa ? g->buf[0] : g->buf[g->cur], g->aa ? nullptr : g->buf[g->cur ^ 1],
        (long long)n, (int)(g->steps & 1), g->d_bar, g->bar_base, g->stream);
    if (e == cudaSuccess) {
      g->bar_base += (unsigned long long)(n - 1) * (unsigned long long)(g->Ns / 128);
      g->steps += n;
      if (!g->aa && (n & 1)) g->cur ^= 1;
      ++g->launches;
      return HLB_OK;
    }
    (void)cudaGetLastError();  // refused (e.g. too large for this instantiation): step by step
    g->resident_failed = true;
  }
  int64_t left = n;
  while (left > 0) {
    const bool even = g->aa ? (g->steps & 1) == 0 : g->cur == 0;
    // with interpolated walls the captured steps all apply the gather-side rule: not from
    // the initial state, nor right after a read-out's pre-pass
    const bool uniform = !g->bfl_set || g->gather_bfl();
    if (want_graph && even && uniform && left >= GRAPH_STEPS && !g->graph_failed) {
      if (!g->graph_exec) build_step_graph(g);
      if (g->graph_exec) {
        HLB_CUDA(cudaGraphLaunch(g->graph_exec, g->stream));
        g->steps += GRAPH_STEPS;
        g->launches += GRAPH_STEPS;
        left -= GRAPH_STEPS;
        continue;
      }
    }
    enqueue_one_step(g);
    --left;
  }
  if (n > 0) HLB_CUDA(cudaGetLastError());
  return HLB_OK;
}

int hlb_get_macroscopic_device(hlb_geometry* g, double* rho_dev, double* u_dev) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (!rho_dev && !u_dev) return HLB_OK;
  g->ensure_bfl();
  launch_macroscopic(g->dg, g->state_buf(), g->gather_mode(), rho_dev, u_dev, g->stream);
  HLB_CUDA(cudaGetLastError());
  return HLB_OK;
}

int hlb_get_macroscopic(hlb_geometry* g, double* rho, double* u) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  const size_t n = (size_t)g->N;
  double* d_rho = g->scratch;
  double* d_u = g->scratch + n;
  int rc = hlb_get_macroscopic_device(g, rho ? d_rho : nullptr, u ? d_u : nullptr);
  if (rc) return rc;
  if (rho) HLB_CUDA(cudaMemcpyAsync(rho, d_rho, sizeof(double) * n, cudaMemcpyDeviceToHost, g->stream));
  if (u) HLB_CUDA(cudaMemcpyAsync(u, d_u, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, g->stream));
  HLB_CUDA(cudaStreamSynchronize(g->stream));
  return HLB_OK;
}

int hlb_get_macroscopic_async(hlb_geometry* g, double* rho, double* u) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (!g->copy_stream) return fail(HLB_EINVAL, "hlb_get_macroscopic_async needs params.copy_stream");
  if (!rho && !u) return HLB_OK;
  const size_t n = (size_t)g->N;
  if (!g->scratch_out) {
    void* ptr = nullptr;
    const int rc = g->alloc(sizeof(double) * 4 * n, &ptr);
    if (rc) return rc;
    g->scratch_out = (double*)ptr;
    HLB_CUDA(cudaEventCreateWithFlags(&g->ev_ready, cudaEventDisableTiming));
    HLB_CUDA(cudaEventCreateWithFlags(&g->ev_copied, cudaEventDisableTiming));
    HLB_CUDA(cudaEventRecord(g->ev_copied, g->copy_stream));
  }
  // the previous copies out of the staging buffer must be done before it is rewritten
  HLB_CUDA(cudaStreamWaitEvent(g->stream, g->ev_copied, 0));
  double* d_rho = g->scratch_out;
  double* d_u = g->scratch_out + n;
  int rc = hlb_get_macroscopic_device(g, rho ? d_rho : nullptr, u ? d_u : nullptr);
  if (rc) return rc;
  HLB_CUDA(cudaEventRecord(g->ev_ready, g->stream));
  HLB_CUDA(cudaStreamWaitEvent(g->copy_stream, g->ev_ready, 0));
  if (rho) HLB_CUDA(cudaMemcpyAsync(rho, d_rho, sizeof(double) * n, cudaMemcpyDeviceToHost, g->copy_stream));
  if (u) HLB_CUDA(cudaMemcpyAsync(u, d_u, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, g->copy_stream));
  HLB_CUDA(cudaEventRecord(g->ev_copied, g->copy_stream));
  return HLB_OK;
}

int hlb_wait_copies(hlb_geometry* g) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (g->copy_stream && (g->ev_ready || g->ev_staged)) HLB_CUDA(cudaStreamSynchronize(g->copy_stream));
  return HLB_OK;
}

int hlb_stage_state(hlb_geometry* g, const double* rho, const double* u) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (!g->copy_stream) return fail(HLB_EINVAL, "hlb_stage_state needs params.copy_stream");
  const size_t n = (size_t)g->N;
  if (!g->scratch_in) {
    void* ptr = nullptr;
    const int rc = g->alloc(sizeof(double) * 4 * n, &ptr);
    if (rc) return rc;
    g->scratch_in = (double*)ptr;
    HLB_CUDA(cudaEventCreateWithFlags(&g->ev_staged, cudaEventDisableTiming));
    HLB_CUDA(cudaEventCreateWithFlags(&g->ev_consumed, cudaEventDisableTiming));
    HLB_CUDA(cudaEventRecord(g->ev_consumed, g->stream));
  }
  // the init kernel of the previous hlb_set_state_staged must have read the buffer
  HLB_CUDA(cudaStreamWaitEvent(g->copy_stream, g->ev_consumed, 0));
  if (rho) HLB_CUDA(cudaMemcpyAsync(g->scratch_in, rho, sizeof(double) * n, cudaMemcpyHostToDevice, g->copy_stream));
  if (u) HLB_CUDA(cudaMemcpyAsync(g->scratch_in + n, u, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, g->copy_stream));
  HLB_CUDA(cudaEventRecord(g->ev_staged, g->copy_stream));
  g->staged = true;
  g->staged_rho = rho != nullptr;
  g->staged_u = u != nullptr;
  return HLB_OK;
}

int hlb_set_state_staged(hlb_geometry* g) {
  if (!g) return fail(HLB_EINVAL, "NULL geometry");
  if (!g->staged) return fail(HLB_EINVAL, "hlb_set_state_staged without a staged state (hlb_stage_state)");
  HLB_CUDA(cudaStreamWaitEvent(g->stream, g->ev_staged, 0));
  const int rc = init_from(g, g->staged_rho ? g->scratch_in : nullptr,
                           g->staged_u ? g->scratch_in + (size_t)g->N : nullptr, nullptr);
  if (rc) return rc;
  HLB_CUDA(cudaEventRecord(g->ev_consumed, g->stream));
  g->staged = false;
  return HLB_OK;
}

int hlb_get_stress_device(hlb_geometry* g, double* sigma_dev) {
  if (!g || !sigma_dev) return fail(HLB_EINVAL, "NULL argument");
  g->ensure_bfl();
  launch_stress(g->dg, g->state_buf(), g->gather_mode(), sigma_dev, g->stream);
  HLB_CUDA(cudaGetLastError());
  return HLB_OK;
}

int hlb_get_stress(hlb_geometry* g, double* sigma) {
  if (!g || !sigma) return fail(HLB_EINVAL, "NULL argument");
  int rc = ensure_scratch_pop(g);  // [N][Q >= 15] doubles hold [N][6]
  if (rc) return rc;
  rc = hlb_get_stress_device(g, g->scratch_pop);
  if (rc) return rc;
  HLB_CUDA(cudaMemcpyAsync(sigma, g->scratch_pop, sizeof(double) * 6 * (size_t)g->N, cudaMemcpyDeviceToHost, g->stream));
  HLB_CUDA(cudaStreamSynchronize(g->stream));
  return HLB_OK;
}

int hlb_get_wall_shear_stress(hlb_geometry* g, const double* normals, double* wss) {
  if (!g || !normals || !wss) return fail(HLB_EINVAL, "NULL argument");
  int rc = ensure_scratch_pop(g);  // [N][Q >= 15]: sigma [N][6] | normals [N][3] | wss [N]
  if (rc) return rc;
  const size_t n = (size_t)g->N;
  double* d_sigma = g->scratch_pop;
  double* d_normals = d_sigma + 6 * n;
  double* d_wss = d_normals + 3 * n;
  HLB_CUDA(cudaMemcpyAsync(d_normals, normals, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, g->stream));
  rc = hlb_get_stress_device(g, d_sigma);
  if (rc) return rc;
  launch_wall_shear_stress(d_sigma, d_normals, g->N, d_wss, g->stream);
  HLB_CUDA(cudaGetLastError());
  HLB_CUDA(cudaMemcpyAsync(wss, d_wss, sizeof(double) * n, cudaMemcpyDeviceToHost, g->stream));
  HLB_CUDA(cudaStreamSynchronize(g->stream));
  return HLB_OK;
}

int64_t hlb_noalloc_max_sites(void) { return (int64_t)NOALLOC_MAX_SITES; }
static_assert(NOALLOC_MAX_SITES == HLB_NOALLOC_MAX_SITES, "include/hlb.h and kernels.cuh disagree");

int hlb_get_wall_shear_stress_noalloc(hlb_geometry* g, const double* normals_dev, double* wss_dev) {
  if (!g || !normals_dev || !wss_dev) return fail(HLB_EINVAL, "NULL argument");
  if (g->N > (int64_t)NOALLOC_MAX_SITES)
    return fail(HLB_ETOOLARGE, "hlb_get_wall_shear_stress_noalloc: " + std::to_string((long long)g->N) +
                               " sites exceed the static scratch of HLB_NOALLOC_MAX_SITES = " +
                               std::to_string((long long)NOALLOC_MAX_SITES) +
                               " sites; use hlb_get_wall_shear_stress");
  if (g->noalloc_setup != cudaSuccess)
    return cuda_fail(g->noalloc_setup, "cudaGetSymbolAddress(static scratch) at hlb_geometry_create");
  double* d_sigma = noalloc_scratch();  // the DEVICE address taken at set-up, not the symbol's name
  if (!d_sigma) return fail(HLB_ECUDA, "static scratch not set up on the current device "
                                       "(the geometry was created on another one)");
  // k_stress writes sigma[c][0..5] for every c < N, k_wall_shear_stress reads exactly those:
  // nothing of an earlier call is read, nothing needs clearing. No allocation on this path
  // (the BFL pre-pass, if due, is a plain launch).
  const int rc = hlb_get_stress_device(g, d_sigma);
  if (rc) return rc;
  launch_wall_shear_stress(d_sigma, normals_dev, g->N, wss_dev, g->stream);
  HLB_CUDA(cudaGetLastError());
  return HLB_OK;
}

static int check_view(const hlb_view* v, const float* lut, RenderSetup& r) {
  if (!v || !lut) return fail(HLB_EINVAL, "NULL argument");
  if (v->width <= 0 || v->height <= 0) return fail(HLB_EINVAL, "image size must be positive");
  if (!(v->zoom > 0.0f) || !(v->step > 0.0f)) return fail(HLB_EINVAL, "zoom and step must be > 0");
  r.width = v->width; r.height = v->height;
  for (int k = 0; k < 9; ++k) r.rot[k] = v->rot[k];
  r.zoom = v->zoom; r.step = v->step; r.tf_scale = v->tf_scale; r.tf_offset = v->tf_offset;
  r.opacity = v->opacity;
  return HLB_OK;
}

// HLB_RENDER_NO_SKIP=1 in the environment turns the empty-space skipping off (same image; for
// measurement only)
// hlb_render samples the volume through a POINT-sampled 3-D texture object over a CUDA array
// (the paper's "3D texture unit"): same values, same in-kernel trilinear
// arithmetic, bit-identical image, and the array's 3-D tiling keeps the eight corner fetches
// of neighbouring rays close whatever the view direction (1024^3 configs[3] box, 1024^2
// frames turning about y: 1.85 ms per frame against 2.76 ms from the linear array; a view
// along z: 3.30 against 3.20 ms; profiles/r02_render.md). HLB_RENDER_LINEAR=1 keeps the
// linear array (measurement only).
static bool render_through_texture() {
  static const bool off = [] { const char* e = getenv("HLB_RENDER_LINEAR"); return e && *e && *e != '0'; }();
  return !off;
}
static bool render_skip_disabled() {
  static const bool off = [] { const char* e = getenv("HLB_RENDER_NO_SKIP"); return e && *e && *e != '0'; }();
  return off;
}

int hlb_render_volume(const float* volume, int32_t nx, int32_t ny, int32_t nz, const hlb_view* view,
                      const float* lut, float* image, void* stream) {
  if (!volume || !image) return fail(HLB_EINVAL, "NULL argument");
  if (nx <= 0 || ny <= 0 || nz <= 0) return fail(HLB_EINVAL, "non-positive volume extent");
  RenderSetup r;
  int rc = check_view(view, lut, r);
  if (rc) return rc;
  r.nx = nx; r.ny = ny; r.nz = nz;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t vbytes = sizeof(float) * (size_t)nx * (size_t)ny * (size_t)nz;
  const size_t ibytes = sizeof(float) * 4 * (size_t)view->width * (size_t)view->height;
  float *d_vol = nullptr, *d_img = nullptr;
  unsigned char* d_occ = nullptr;
  auto done = [&](int code) { cudaFree(d_vol); cudaFree(d_img); cudaFree(d_occ); return code; };
  if (cudaMalloc((void**)&d_vol, vbytes) != cudaSuccess || cudaMalloc((void**)&d_img, ibytes) != cudaSuccess ||
      cudaMalloc((void**)&d_occ, (size_t)occupancy_cells(nx, ny, nz)) != cudaSuccess) {
    const cudaError_t e = cudaGetLastError();
    return done(e == cudaErrorMemoryAllocation ? fail(HLB_ENOMEM, "cudaMalloc: out of memory")
                                               : cuda_fail(e, "cudaMalloc"));
  }
  cudaError_t e = cudaMemcpyAsync(d_vol, volume, vbytes, cudaMemcpyHostToDevice, s);
  if (e == cudaSuccess) { launch_occupancy(d_vol, nx, ny, nz, d_occ, s); e = cudaGetLastError(); }
  if (e == cudaSuccess) { launch_raymarch(r, lut, d_vol, 0, render_skip_disabled() ? nullptr : d_occ, d_img, s); e = cudaGetLastError(); }
  if (e == cudaSuccess) e = cudaMemcpyAsync(image, d_img, ibytes, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return done(cuda_fail(e, "hlb_render_volume"));
  return done(HLB_OK);
}

int hlb_render_device(hlb_geometry* g, const hlb_view* view, const float* lut, float* image_dev) {
  if (!g || !image_dev) return fail(HLB_EINVAL, "NULL argument");
  RenderSetup r;
  int rc = check_view(view, lut, r);
  if (rc) return rc;
  if (view->field != 0 && view->field != 1) return fail(HLB_EINVAL, "field must be 0 (speed) or 1 (rho - 1)");
  r.nx = g->p.nx; r.ny = g->p.ny; r.nz = g->p.nz;
  const size_t nvox = (size_t)r.nx * (size_t)r.ny * (size_t)r.nz;
  if (!g->volume) {
    // both buffers or neither: a half-finished set-up must not look finished to the next call
    void *vol = nullptr, *vox = nullptr;
    if ((rc = g->alloc(sizeof(float) * nvox, &vol))) return rc;
    if ((rc = g->alloc(sizeof(long long) * (size_t)g->N, &vox))) {
      g->release(vol, sizeof(float) * nvox);
      return rc;
    }
    static_assert(sizeof(long long) == sizeof(int64_t), "voxel index width");
    HLB_CUDA(cudaMemcpyAsync(vox, g->canon_voxels.data(), sizeof(int64_t) * (size_t)g->N,
                             cudaMemcpyHostToDevice, g->stream));
    HLB_CUDA(cudaMemsetAsync(vol, 0, sizeof(float) * nvox, g->stream));  // solid voxels stay 0
    g->volume = (float*)vol;
    g->d_voxels = (long long*)vox;
  }
  if (render_through_texture() && !g->vol_tex) {
    cudaChannelFormatDesc fmt = cudaCreateChannelDesc<float>();
    cudaArray_t arr = nullptr;
    HLB_CUDA(cudaMalloc3DArray(&arr, &fmt, make_cudaExtent((size_t)r.nx, (size_t)r.ny, (size_t)r.nz),
                               cudaArraySurfaceLoadStore));
    cudaResourceDesc res = {};
    res.resType = cudaResourceTypeArray;
    res.res.array.array = arr;
    cudaTextureDesc td = {};
    td.addressMode[0] = td.addressMode[1] = td.addressMode[2] = cudaAddressModeClamp;
    td.filterMode = cudaFilterModePoint;
    td.readMode = cudaReadModeElementType;
    td.normalizedCoords = 0;
    cudaTextureObject_t tex = 0;
    cudaSurfaceObject_t surf = 0;
    cudaError_t e = cudaCreateTextureObject(&tex, &res, &td, nullptr);
    if (e == cudaSuccess) e = cudaCreateSurfaceObject(&surf, &res);
    // solid voxels stay 0: clear the array once through a copy of the (zeroed) linear volume
    cudaMemcpy3DParms cp = {};
    cp.srcPtr = make_cudaPitchedPtr(g->volume, (size_t)r.nx * sizeof(float), (size_t)r.nx, (size_t)r.ny);
    cp.dstArray = arr;
    cp.extent = make_cudaExtent((size_t)r.nx, (size_t)r.ny, (size_t)r.nz);
    cp.kind = cudaMemcpyDeviceToDevice;
    if (e == cudaSuccess) e = cudaMemcpy3DAsync(&cp, g->stream);
    if (e != cudaSuccess) {
      if (tex) cudaDestroyTextureObject(tex);
      if (surf) cudaDestroySurfaceObject(surf);
      cudaFreeArray(arr);
      return cuda_fail(e, "3-D texture set-up");
    }
    g->vol_array = arr; g->vol_tex = tex; g->vol_surf = surf;
    g->device_bytes += (int64_t)(sizeof(float) * nvox);
  }
  double* d_rho = g->scratch;
  double* d_u = g->scratch + g->N;
  rc = hlb_get_macroscopic_device(g, d_rho, d_u);
  if (rc) return rc;
  if (!g->occ && !render_skip_disabled()) {
    // Only fluid voxels are ever written, so a macro-cell without fluid stays empty for good:
    // mark every fluid voxel with a non-zero value once and take the occupancy of that.
    void* ptr = nullptr;
    if ((rc = g->alloc((size_t)occupancy_cells(r.nx, r.ny, r.nz), &ptr))) return rc;
    launch_scatter_field(d_rho, d_u, g->d_voxels, g->N, 2, g->volume, 0, r.nx, r.ny, g->stream);  // field 2: the constant 1
    launch_occupancy(g->volume, r.nx, r.ny, r.nz, (unsigned char*)ptr, g->stream);
    HLB_CUDA(cudaGetLastError());
    g->occ = (unsigned char*)ptr;
  }
  launch_scatter_field(d_rho, d_u, g->d_voxels, g->N, view->field, g->volume, g->vol_surf, r.nx, r.ny, g->stream);
  HLB_CUDA(cudaGetLastError());
  launch_raymarch(r, lut, g->volume, g->vol_tex, g->occ, image_dev, g->stream);
  HLB_CUDA(cudaGetLastError());
  return HLB_OK;
}

int hlb_render(hlb_geometry* g, const hlb_view* view, const float* lut, float* image) {
  if (!g || !image || !view) return fail(HLB_EINVAL, "NULL argument");
  if (view->width <= 0 || view->height <= 0) return fail(HLB_EINVAL, "image size must be positive");
  const size_t nfl = 4 * (size_t)view->width * (size_t)view->height;
  if (g->d_image_floats < nfl) {
    void* ptr = nullptr;
    int rc = g->alloc(sizeof(float) * nfl, &ptr);
    if (rc) return rc;
    HLB_CUDA(cudaStreamSynchronize(g->stream));
    g->release(g->d_image, sizeof(float) * g->d_image_floats);
    g->d_image = (float*)ptr;
    g->d_image_floats = nfl;
  }
  int rc = hlb_render_device(g, view, lut, g->d_image);
  if (rc) return rc;
  HLB_CUDA(cudaMemcpyAsync(image, g->d_image, sizeof(float) * nfl, cudaMemcpyDeviceToHost, g->stream));
  HLB_CUDA(cudaStreamSynchronize(g->stream));
  return HLB_OK;
}

int hlb_get_populations(hlb_geometry* g, double* f) {
  if (!g || !f) return fail(HLB_EINVAL, "NULL argument");
  int rc = ensure_scratch_pop(g);
  if (rc) return rc;
  g->ensure_bfl();
  launch_get_populations(g->dg, g->state_buf(), g->gather_mode(), g->scratch_pop, g->stream);
  HLB_CUDA(cudaGetLastError());
  HLB_CUDA(cudaMemcpyAsync(f, g->scratch_pop, sizeof(double) * (size_t)g->Q * (size_t)g->N, cudaMemcpyDeviceToHost, g->stream));
  HLB_CUDA(cudaStreamSynchronize(g->stream));
  return HLB_OK;
}

int hlb_num_q(const hlb_geometry* g) { return g ? g->Q : (int)HLB_EINVAL; }
int64_t hlb_num_sites(const hlb_geometry* g) { return g ? g->N : (int64_t)HLB_EINVAL; }
int64_t hlb_steps_done(const hlb_geometry* g) { return g ? g->steps : (int64_t)HLB_EINVAL; }
int64_t hlb_device_bytes(const hlb_geometry* g) { return g ? g->device_bytes : (int64_t)HLB_EINVAL; }
int64_t hlb_launch_count(const hlb_geometry* g) { return g ? g->launches : (int64_t)HLB_EINVAL; }
int hlb_offset_bits(const hlb_geometry* g) { return g ? (g->dg.index64 ? 64 : 32) : (int)HLB_EINVAL; }
int hlb_uses_aa(const hlb_geometry* g) { return g ? (g->aa ? 1 : 0) : (int)HLB_EINVAL; }
int hlb_uses_records(const hlb_geometry* g) { return g ? (g->dg.use_rec ? 1 : 0) : (int)HLB_EINVAL; }
double hlb_record_sentinel_fraction(const hlb_geometry* g) { return g ? g->sentinel_fraction : -1.0; }
int hlb_get_site_voxels(const hlb_geometry* g, int64_t* v) {
  if (!g || !v) return fail(HLB_EINVAL, "NULL argument");
  std::memcpy(v, g->canon_voxels.data(), sizeof(int64_t) * (size_t)g->N);
  return HLB_OK;
}

}  // extern "C"
