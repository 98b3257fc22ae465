/* hlb.h -- C-ABI boundary of the B200-native sparse lattice-Boltzmann site update.
 *
 * One thing lives behind this header: the per-timestep site update of a HemeLB-style
 * solver -- "a lattice of fluid sites, each equipped with a single-particle distribution
 * ... evolution of these particle distributions over consecutive propagation and collision
 * steps" (section II), with "simple bounce-back boundary condition"
 * (section IV) -- in the concrete form BASELINE.json `north_star` fixes:
 * fused D3Q15 LBGK collide-and-stream over a sparse, indirectly addressed list of fluid
 * sites, halfway bounce-back walls, constant-density inlets/outlets. The paper's own lattice,
 * D3Q19, is selected with HLB_LATTICE_D3Q19; Q below is the
 * lattice's population count (15 or 19). The formulas and the readings of every point the
 * paper leaves open are in DESIGN.md ("Readings").
 *
 * Conventions
 *   - Plain C ABI: no C++ or torch types. Every function returns HLB_OK (0) or a negative
 *     hlb_status and never throws; hlb_last_error() gives a thread-local message.
 *   - Voxel box nx*ny*nz, linear voxel index v = (z*ny + y)*nx + x.
 *   - CANONICAL SITE ORDER = ascending v over the fluid voxels. Every per-site array that
 *     crosses this boundary (rho, u, populations, site voxels) is in canonical order; the
 *     library's internal (Morton / blocked) order never leaks.
 *   - "host" / "device" is stated per pointer. Inputs are caller-owned and only read during
 *     the call. Outputs go to caller-allocated buffers.
 *   - Device memory comes from the caller's allocator callback (PyTorch in the Python
 *     binding) and is released by the caller after hlb_geometry_destroy(); with a NULL
 *     callback the library uses cudaMalloc / cudaFree itself.
 *   - All device work is enqueued on hlb_params.stream. The library never calls
 *     cudaSetDevice and creates no streams. hlb_step() is asynchronous; the calls that
 *     return data to the host synchronise that stream.
 *   - There is no CPU fallback: without a CUDA device every compute entry point fails
 *     with HLB_ECUDA. hlb_preprocess_* are host-only by design (the geometry preprocessor
 *     is host code) and work anywhere.
 */
#ifndef HLB_H_
#define HLB_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  HLB_OK = 0,
  HLB_EINVAL = -1,    /* NULL pointer, non-positive extent, tau <= 0.5, site type >=
                         2 + n_iolets, iolet density <= 0, n < 0, unknown flag combination */
  HLB_ENOFLUID = -2,  /* no voxel of type 1                                               */
  HLB_ETOOLARGE = -3, /* N >= 2^31 - 128 (site indices are int32)                         */
  HLB_ENOMEM = -4,    /* allocator returned NULL                                          */
  HLB_ECUDA = -5      /* a CUDA call failed (text in hlb_last_error())                    */
} hlb_status;

/* hlb_params.flags: one value from each group, OR-ed together. */
enum {
  HLB_STORE_F64 = 0x0,     /* populations stored as IEEE binary64                          */
  HLB_STORE_F32 = 0x1,     /* stored as binary32 (round-to-nearest-even on store, exact
                              widening on load); ALL arithmetic stays fp64; what is stored
                              is h_q = f_q - w_q (reading R-shift)               */
  HLB_TWO_LATTICE = 0x0,   /* two population arrays, pull (gather) form                    */
  HLB_AA = 0x2,            /* one array updated in place, A-A pattern (even/odd steps)     */
  HLB_SCHEME_AUTO = 0x1000,/* the library picks: A-A in place (one array; measured 1-25 %
                              faster than two-lattice above ~150 k sites), except where the
                              resident multi-step kernel applies and where the grid is one
                              wave of the two-lattice kernel but more than one of the A-A
                              kernels (DESIGN.md section 6 item 17); overrides HLB_AA.
                              hlb_uses_aa() tells which was taken                          */
  HLB_ORDER_AUTO = 0x0,    /* internal site order: the library's choice -- currently raster,
                              the fastest measured on B200       */
  HLB_ORDER_MORTON = 0x4,  /* Morton (Z) curve over voxel coordinates                      */
  HLB_ORDER_RASTER = 0x8,  /* internal order = canonical order (x fastest)                 */
  HLB_ORDER_TILED = 0xC,   /* Morton over 8x8x8 blocks, x-fastest raster inside a block    */
  HLB_ORDER_MASK = 0xC,
  HLB_NO_GRAPH = 0x10,     /* launch every step directly instead of replaying a captured
                              CUDA graph of steps or running the resident multi-step kernel
                              (debugging / profiling)                                      */
  HLB_NO_RESIDENT = 0x800, /* never use the resident multi-step kernel (see hlb_step)      */
  HLB_LINKS_AUTO = 0x0,    /* the step kernels read the run-length link records when at
                              least half of them are not sentinels, else the table         */
  HLB_LINKS_TABLE = 0x20,  /* always read the int32 table (ablation / profiling)           */
  HLB_LINKS_RECORDS = 0x40,/* always read the records                                     */
  HLB_NO_PREFETCH = 0x80,  /* step kernels issue no L2 prefetches (ablation / profiling;
                              the library issues none by itself where the populations fit
                              half of the L2 cache)                                        */
  HLB_INDEX64 = 0x100,     /* use the 64-bit flat-offset kernels even when Q * stride fits
                              32 bits (they are otherwise only taken above 286 M sites;
                              this flag lets small tests cover them)                       */
  HLB_NO_PDL = 0x400,      /* launch the step kernels without programmatic dependent launch
                              (by default step t+1 starts its blocks and fetches its link
                              records while the last blocks of step t finish)              */
  HLB_LATTICE_D3Q15 = 0x0, /* 15 velocities: rest, 6 axis, 8 cube diagonals (BASELINE.json) */
  HLB_LATTICE_D3Q19 = 0x200 /* 19 velocities: rest, 6 axis, 12 face diagonals -- the lattice
                              the paper names. Everywhere below
                              Q = 15 or 19 is the lattice's population count and Q - 1 its
                              link count                                                   */
};

typedef struct hlb_geometry hlb_geometry; /* opaque handle */

/* Returns a DEVICE pointer to `bytes` bytes, at least 256-byte aligned, or NULL. The
 * memory must stay valid until after hlb_geometry_destroy(). */
typedef void* (*hlb_alloc_fn)(size_t bytes, void* user);
/* Optional counterpart: called with a pointer hlb_alloc_fn returned once the library no longer
 * uses it and no enqueued work refers to it (a table that was regrown: a longer waveform, a
 * larger image, other wall distances). Without it such buffers stay with the caller until
 * hlb_geometry_destroy(). */
typedef void (*hlb_free_fn)(void* ptr, void* user);

typedef struct {
  int32_t nx, ny, nz;      /* voxel box, each >= 1                                         */
  uint32_t periodic;       /* bit0 = x, bit1 = y, bit2 = z wrap; a non-periodic axis has
                              solid outside the box                                        */
  double tau;              /* LBGK relaxation time, must be > 0.5; nu = (tau - 1/2)/3      */
  int32_t n_iolets;        /* 0..253                                                       */
  const double* iolet_rho; /* HOST, n_iolets densities in lattice units (may be NULL when
                              n_iolets == 0)                                               */
  uint32_t flags;          /* HLB_STORE_* | HLB_TWO_LATTICE/HLB_AA | HLB_ORDER_* | ...     */
  hlb_alloc_fn alloc;      /* device allocator or NULL (=> cudaMalloc)                     */
  void* alloc_user;
  void* stream;            /* cudaStream_t as void*; NULL = the legacy default stream      */
  hlb_free_fn free;        /* optional (NULL): releases one buffer of `alloc` early; called
                              with alloc_user                                              */
  void* copy_stream;       /* optional (NULL): a second cudaStream_t of the caller, used only by
                              hlb_get_macroscopic_async and hlb_stage_state for their copies
                              from / to the host, so that they overlap the steps on `stream` */
} hlb_params;

/* Build the geometry: extract the fluid sites, order them, build the int32 pull-neighbour
 * table (wall and iolet links encoded as bounce-back targets), upload, and initialise the
 * state to rho = 1, u = 0 (f = f_eq, step counter 0).
 *   site_type: HOST array of nx*ny*nz bytes. 0 = solid, 1 = fluid, 2+k = ghost voxel of
 *              iolet k (never simulated; it marks the links that cross iolet k).
 * Errors: HLB_EINVAL, HLB_ENOFLUID, HLB_ETOOLARGE, HLB_ENOMEM, HLB_ECUDA. On error *out
 * is set to NULL. */
int hlb_geometry_create(const uint8_t* site_type, const hlb_params* p, hlb_geometry** out);

/* Set f_q(x, 0) = f_eq_q(rho(x), u(x)) and the step counter to 0.
 *   rho: HOST [N] or NULL (=> 1);  u: HOST [N][3] or NULL (=> 0); canonical order.
 * The host arrays have been read when the call returns (it waits for its own copies; this
 * holds for every hlb_set_* call that takes host arrays). */
int hlb_set_state(hlb_geometry* g, const double* rho, const double* u);

/* Replace the n_iolets iolet densities (HOST array, each > 0). Takes effect from the next
 * step; the density of an iolet that is currently a velocity iolet is kept for later. */
int hlb_set_iolet_density(hlb_geometry* g, const double* iolet_rho);

/* Normals of the constant-density iolets ("normal-projected" pressure iolets): with a normal
 * n_k given, the rule f_q(x,t+1) = f_eq_q(rho_k, u(x,t)) uses only the part of u along n_k,
 * (u.n_k) n_k.  normals: HOST [n_iolets][3], any length (normalised here), a zero vector (or
 * NULL for all) = no projection, the default. Ignored for velocity iolets. Takes effect from
 * the next step. */
int hlb_set_iolet_normal(hlb_geometry* g, const double* normals);

/* Interpolated ("BFL") walls -- the paper's wall option (ref. [16]:
 * Bouzidi, Firdaouss & Lallemand), linear form. d27: HOST [N][27] in canonical site order;
 * entry (dz+1)*9 + (dy+1)*3 + (dx+1) is the fraction d in (0, 1] of the link from the site
 * along the lattice vector (dx, dy, dz) at which the wall cuts it (1/2 = the halfway
 * bounce-back default); <= 0 or > 1: no distance for that link. With i = opp(q) the direction
 * from x to the wall and y = x + c_q the site behind x, a solid-wall link q becomes
 *     d <  1/2:  f_q(x,t+1) = 2d f*_i(x,t) + (1 - 2d) f*_i(y,t)
 *     d >= 1/2:  f_q(x,t+1) = f*_i(x,t) / (2d) + (1 - 1/(2d)) f*_q(x,t)
 * where y is a fluid site; otherwise (y solid or iolet, or no distance) the link stays a
 * halfway bounce-back (reading R-bfl). Iolet links are not affected. NULL switches
 * the interpolation off. The step kernels of both schemes apply it in registers (the d >= 1/2
 * rule to the value a site writes back, the d < 1/2 rule to the values it gathers; no extra
 * launch per step); a read-out between steps first runs a pre-pass kernel over the d < 1/2
 * links of the state buffer. With HLB_STORE_F64 the pre-pass writes exactly what the next step
 * would have computed in registers, so reading out does not change the run. With HLB_STORE_F32
 * it rounds those interpolated values to binary32 one step earlier than a run without the
 * read-out would: a read-out (hlb_get_macroscopic, _stress, _populations, hlb_render) then
 * perturbs the trajectory at the level of the storage rounding itself (~1e-8 relative, inside
 * the 1e-5 bar; tests/test_gpu_parity.py). Only while hlb_steps_done() == 0
 * (after create / hlb_set_state / hlb_set_populations; it survives later hlb_set_state
 * calls). Allocates its tables through the allocator. Errors: HLB_EINVAL, HLB_ENOMEM,
 * HLB_ECUDA. hlb_num_bfl_sites: sites with at least one interpolated link (0 when off). */
int hlb_set_wall_distance(hlb_geometry* g, const double* d27);
int64_t hlb_num_bfl_sites(const hlb_geometry* g);

/* Choose, per iolet, between the constant-density rule (kind 0, the default:
 * f_q(x,t+1) = f_eq_q(rho_k, u(x,t))) and Ladd's velocity rule (kind 1, the paper's
 * "LADDIOLET" boundary, ref. [15]): a link whose source voxel is a
 * ghost voxel of velocity iolet k bounces back off a boundary moving with u_k,
 *     f_q(x,t+1) = f*_opp(q)(x,t) + 6 w_q rho(x,t) c_q.u_k      (reading R-ladd).
 *   kind: HOST [n_iolets] bytes 0 / 1, or NULL (all 0);  u: HOST [n_iolets][3] lattice
 *   velocities (read for kind 1; may be NULL when no kind is 1).
 * Takes effect from the next step, so a time-varying inlet (the paper's Fig. 8 waveform) is
 * hlb_step(n) / hlb_set_iolet_velocity(...) in turn. Errors: HLB_EINVAL. */
int hlb_set_iolet_velocity(hlb_geometry* g, const uint8_t* kind, const double* u);

/* Per-site velocity weights of the velocity iolets -- a velocity profile across the inlet
 * cap (the paper's build flag USE_VELOCITY_WEIGHTS_FILE; the file itself is
 * not in the paper): as seen from site x the boundary of a velocity iolet k moves with
 * omega(x) u_k,
 *     f_q(x,t+1) = f*_opp(q)(x,t) + 6 w_q rho(x,t) omega(x) c_q.u_k   (reading R-weights)
 * for every link q of x whose source voxel is a ghost voxel of a kind-1 iolet (with or without
 * a waveform). weight: HOST [N] in canonical site order, copied during the call (entries of
 * sites without such a link are ignored); NULL removes the weights (omega = 1). Takes effect
 * from the next step. Synchronises the stream. Errors: HLB_EINVAL (non-finite weight),
 * HLB_ENOMEM, HLB_ECUDA. */
int hlb_set_iolet_weight(hlb_geometry* g, const double* weight);

/* Device-resident velocity waveform for the velocity iolets (the paper drives its inlet from
 * a velocity file, Table I "inlet velocity" and line 126 Fig. 8): with a
 * waveform the step that advances the state from time t to t+1 (t = hlb_steps_done() before
 * it) applies Ladd's rule of hlb_set_iolet_velocity with
 *     u_k = u[t mod n_t][k]            (periodic in time, one vector per iolet and time level)
 * for every iolet k of kind 1, so hlb_step(n) covers n time levels with no host work between
 * the launches (calling hlb_set_iolet_velocity before every step gives the same result and
 * costs a stream synchronisation per step).
 *   u: HOST [n_t][n_iolets][3] lattice velocities, copied during the call; rows of iolets of
 *   kind 0 are ignored. n_t >= 1. u == NULL or n_t == 0 removes the waveform: velocity iolets
 *   go back to the constant vectors of hlb_set_iolet_velocity.
 * The kinds (hlb_set_iolet_velocity), densities and normals may be changed afterwards; the
 * waveform stays. hlb_set_state / hlb_set_populations reset the time to 0. The table
 * (n_t * n_iolets * 32 bytes) comes from the allocator. While a waveform is set the steps are
 * launched directly (no CUDA-graph replay: a captured launch fixes its time level).
 * Errors: HLB_EINVAL (n_t < 0, no iolets but n_t > 0, non-finite velocity), HLB_ENOMEM,
 * HLB_ECUDA. */
int hlb_set_iolet_waveform(hlb_geometry* g, const double* u, int64_t n_t);

/* Advance n >= 0 time steps: n launches of ONE fused collide-and-stream kernel (A-A:
 * alternating even/odd kernels), asynchronously on the stream. n == 0 is a no-op. A
 * kernel fault surfaces at the next synchronising call. For geometries of up to 2^22
 * sites on a non-NULL stream the launches are replayed from a captured CUDA graph in
 * chunks of 32 steps (same kernels, same order; HLB_NO_GRAPH switches it off).
 * Geometries small enough for all their thread blocks (128 sites each) to be resident on
 * the chip at once (about 10^5 sites on a B200) run a call of n >= 2 steps as ONE
 * cooperative launch of a resident kernel instead: every thread keeps its site and its link
 * offsets in registers for the n steps, with a grid-wide barrier between steps in place of
 * the kernel boundary (same per-site arithmetic, bitwise the same results; not with
 * interpolated walls or a waveform; HLB_NO_RESIDENT or HLB_NO_GRAPH switches it off). Such a
 * launch needs every SM slot it was sized for: it must not share the device with another
 * long-running kernel of the same process that waits on it. */
int hlb_step(hlb_geometry* g, int64_t n);

/* rho(x) = sum_q f_q, u(x) = sum_q c_q f_q / rho of the PRE-collision populations after
 * hlb_steps_done() steps (reading R-readout), canonical order.
 *   rho: HOST [N];  u: HOST [N][3]. Either may be NULL. Synchronises the stream. */
int hlb_get_macroscopic(hlb_geometry* g, double* rho, double* u);
/* The same, without waiting: the read-out kernel runs on `stream`, the copies to the HOST
 * arrays (pinned memory, or they are not asynchronous) on params.copy_stream once it is
 * done, and the call returns at once; work enqueued on `stream` afterwards (hlb_set_state,
 * hlb_step) overlaps the copies. The arrays are valid after hlb_wait_copies(), which also any
 * later hlb_get_macroscopic_async waits for before it reuses the staging buffer. Needs
 * params.copy_stream (else HLB_EINVAL). */
int hlb_get_macroscopic_async(hlb_geometry* g, double* rho, double* u);
int hlb_wait_copies(hlb_geometry* g);

/* The counterpart for the way in: hlb_stage_state uploads an initial state (HOST, pinned, as
 * hlb_set_state: rho [N] or NULL => 1, u [N][3] or NULL => 0) into a staging buffer on
 * params.copy_stream WITHOUT touching the simulation -- it may run under hlb_step calls still
 * in flight on `stream` -- and returns at once; the arrays must stay valid until the next
 * hlb_wait_copies(). hlb_set_state_staged then does what hlb_set_state does, from the staged
 * copy: `stream` waits for the upload, f = f_eq(rho, u), step counter 0. One staged state at
 * a time: a second hlb_stage_state waits (on the device) until the first has been consumed.
 * Errors: HLB_EINVAL (no copy stream; hlb_set_state_staged without a staged state),
 * HLB_ENOMEM (the first call allocates the staging buffer), HLB_ECUDA. */
int hlb_stage_state(hlb_geometry* g, const double* rho, const double* u);
int hlb_set_state_staged(hlb_geometry* g);

/* Same, into DEVICE buffers (rho [N], u [N][3]); enqueued on the stream, no sync. */
int hlb_get_macroscopic_device(hlb_geometry* g, double* rho_dev, double* u_dev);

/* Deviatoric (viscous) stress tensor of the same pre-collision state,
 *     sigma_ab(x) = -(1 - 1/(2 tau)) sum_q c_qa c_qb (f_q - f_eq_q(rho, u)),
 * the quantity wall shear stress is derived from ("pressure and velocity", PAPER.md line 27;
 * the pressure itself is rho / 3), canonical order, HOST [N][6] in the order xx, yy, zz, xy,
 * xz, yz. Synchronises the stream. The first call allocates a staging buffer through the
 * allocator (as hlb_get_populations). hlb_get_stress_device: DEVICE [N][6], no sync. */
int hlb_get_stress(hlb_geometry* g, double* sigma);
int hlb_get_stress_device(hlb_geometry* g, double* sigma_dev);

/* Wall shear stress: with t = sigma n the traction on the plane of unit normal n, the size of
 * its tangential part, |t - (t.n) n|.
 *   normals: HOST [N][3] canonical order, the wall normal at each site (any length; a zero
 *            vector marks a site away from the wall and gives 0). The voxel mask carries no
 *            normals, so they are the caller's (from the surface the mask was made from).
 *   wss:     HOST [N]. Synchronises the stream. */
int hlb_get_wall_shear_stress(hlb_geometry* g, const double* normals, double* wss);

/* The same wall shear stress for callers that must not allocate (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): this call allocates NOTHING
 * -- no cudaMalloc / cudaFree, no allocator callback, no allocating library routine -- and does
 * not synchronise. Its only scratch, the stress tensor sigma [N][6] between the two kernels, lives
 * in a file-scope static __device__ array of HLB_NOALLOC_MAX_SITES x 6 doubles (12 MiB) that
 * every GPU which loads the library holds until the process exits; its device address is taken
 * once per device when a geometry is created on it.
 *   normals: DEVICE [N][3] canonical order (as hlb_get_wall_shear_stress);  wss: DEVICE [N].
 * Both are the caller's; the two kernels are enqueued on the geometry's stream.
 * Limits: N <= HLB_NOALLOC_MAX_SITES (= hlb_noalloc_max_sites()), else HLB_ETOOLARGE and nothing
 * is launched. ALL geometries of a process share the one array on a device: two such calls that
 * overlap on the GPU (different streams, or graphs replayed concurrently) race on it -- order
 * them. The array keeps the last call's contents; every element a call reads it has written
 * itself first, so nothing needs clearing between calls.
 * Errors: HLB_EINVAL (NULL argument), HLB_ETOOLARGE, HLB_ECUDA (launch error, or the address of
 * the array could not be taken when the geometry was created: hlb_last_error says which). */
#define HLB_NOALLOC_MAX_SITES 262144
int hlb_get_wall_shear_stress_noalloc(hlb_geometry* g, const double* normals_dev, double* wss_dev);
int64_t hlb_noalloc_max_sites(void);

/* Pre-collision populations f_q(x) (not shifted) as fp64, HOST [N][Q], canonical site
 * order, q in the order of hlb_lattice(). For population-level parity checks. The
 * first call of this or of hlb_set_populations allocates a [N][Q] fp64 staging buffer
 * through the allocator (HLB_ENOMEM if that fails). */
int hlb_get_populations(hlb_geometry* g, double* f);

/* Set pre-collision populations f_q(x, 0) directly (HOST [N][Q], layout as above) and
 * the step counter to 0. */
int hlb_set_populations(hlb_geometry* g, const double* f);

int64_t hlb_num_sites(const hlb_geometry* g);  /* N, or HLB_EINVAL for NULL                */
int hlb_num_q(const hlb_geometry* g);          /* Q of the geometry's lattice (15 or 19)   */
int64_t hlb_steps_done(const hlb_geometry* g);
/* Linear voxel index of every site, HOST [N], canonical order (ascending). */
int hlb_get_site_voxels(const hlb_geometry* g, int64_t* v);
/* Bytes of device memory the geometry holds (populations + tables + scratch). */
int64_t hlb_device_bytes(const hlb_geometry* g);
/* Kernel launches enqueued by hlb_step() so far (graph replays count their nodes; a resident
 * multi-step launch counts once; with BFL
 * walls the pre-pass over the interpolated links counts too, also when a read-out runs it). */
int64_t hlb_launch_count(const hlb_geometry* g);
/* Width of the flat population offsets the step kernels compute: 32, or 64 when Q * stride
 * >= 2^32 (above 286 M sites for D3Q15) or HLB_INDEX64 was given. */
int hlb_offset_bits(const hlb_geometry* g);
/* 1 if the geometry steps in place (A-A), 0 if it uses two arrays (see HLB_SCHEME_AUTO). */
int hlb_uses_aa(const hlb_geometry* g);
/* 1 if the step kernels of this geometry read the link records, 0 if they read the table. */
int hlb_uses_records(const hlb_geometry* g);
/* Fraction of (group, q) link records that are sentinels (see hlb_preprocess_records). */
double hlb_record_sentinel_fraction(const hlb_geometry* g);

void hlb_geometry_destroy(hlb_geometry* g); /* NULL is a no-op                            */
const char* hlb_last_error(void);           /* thread-local, never NULL                   */

/* The library's D3Q15 set: c HOST [15][3], w HOST [15], opp HOST [15]. */
void hlb_velocity_set(int32_t* c, double* w, int32_t* opp);
/* The velocity set selected by the HLB_LATTICE_* bits of flags: c HOST [Q][3], w HOST [Q],
 * opp HOST [Q] (arrays of 19 entries always suffice; any may be NULL). Returns Q. */
int hlb_lattice(uint32_t flags, int32_t* c, double* w, int32_t* opp);

/* ---- volume rendering to a headless buffer -----------------------
 * The paper's own GPU kernel: "the volume rendering kernel based on the ray marching
 * algorithm", the look-up table and viewing parameters in constant memory, steering by zoom,
 * rotation and scale / offset of the transfer function. No window,
 * no OpenGL: the image is a float RGBA buffer. Definition (reading R-render):
 *   volume v[z][y][x] of nx*ny*nz floats, voxel centres at integer coordinates;
 *   orthographic camera along view +z; rot (row-major 3x3) maps view to volume space about
 *   the box centre; pixel (px, py) -> X = (px + 0.5 - width/2) / zoom, same for Y; samples
 *   k = 0 .. floor(2T/step) at view z = -T + k step, T = half the box diagonal; samples
 *   outside [0, n-1]^3 are skipped; trilinear interpolation; t = clamp(value * tf_scale +
 *   tf_offset, 0, 1); entry (int)(255 t + 0.5) of the 256-entry RGBA table; sample opacity
 *   a = clamp(lut.a * opacity, 0, 1); front-to-back: C += (1-A) a rgb, A += (1-A) a; stop at
 *   A >= 0.995. All arithmetic binary32. */
typedef struct {
  int32_t width, height;  /* image size in pixels, each >= 1                               */
  float rot[9];           /* row-major rotation, view -> volume                            */
  float zoom;             /* pixels per voxel, > 0                                         */
  float step;             /* distance between samples in voxels, > 0                       */
  float tf_scale, tf_offset; /* transfer function                                          */
  float opacity;          /* multiplies the table's alpha                                  */
  int32_t field;          /* hlb_render only: 0 = speed |u|, 1 = rho - 1                   */
} hlb_view;

/* Render a HOST volume [nz][ny][nx] with the HOST table lut [256][4] into the HOST image
 * [height][width][4]. Uses cudaMalloc for its scratch; work goes to `stream` (cudaStream_t as
 * void*, NULL = default) and is complete on return. Errors: HLB_EINVAL, HLB_ENOMEM, HLB_ECUDA. */
int hlb_render_volume(const float* volume, int32_t nx, int32_t ny, int32_t nz, const hlb_view* view,
                      const float* lut, float* image, void* stream);

/* Render the geometry's current state: the scalar field view->field of the pre-collision
 * state is written into a dense nx*ny*nz float volume on the device (0 outside the fluid;
 * allocated through the allocator on first use and kept), then ray-marched.
 *   hlb_render: image HOST [height][width][4], synchronises the stream.
 *   hlb_render_device: image DEVICE [height][width][4] (16-byte aligned), no sync. */
int hlb_render(hlb_geometry* g, const hlb_view* view, const float* lut, float* image);
int hlb_render_device(hlb_geometry* g, const hlb_view* view, const float* lut, float* image_dev);

/* ---- geometry preprocessor, host only (subsystem (b) of BASELINE.json north_star) ----
 * Two calls: hlb_preprocess_count() gives N and the plane stride Ns (N rounded up to a
 * multiple of 128); hlb_preprocess_tables() fills caller-allocated HOST arrays:
 *   voxel_of_site [N]      linear voxel index of internal site i
 *   canon_of_site [N]      canonical rank of internal site i
 *   nbr           [Q-1][Ns] entry (q-1)*Ns + i describes the pull source x - c_q of link q
 *                          (q = 1..Q-1) of internal site i:
 *                            >= 0            internal index of the fluid source site
 *                            0x80000000      solid (or outside a non-periodic box): the
 *                                            bounce-back target is slot opp(q) of site i
 *                            0x80000000 | (k+1)  ghost voxel of iolet k (also a bounce-back
 *                                            target; the kernel substitutes f_eq(rho_k, u))
 *                          entries i >= N of each plane are 0x80000000.
 * Only nx, ny, nz, periodic, n_iolets and the HLB_ORDER_* / HLB_LATTICE_* bits of p are read. */
int hlb_preprocess_count(const uint8_t* site_type, const hlb_params* p, int64_t* n_sites,
                         int64_t* stride);
int hlb_preprocess_tables(const uint8_t* site_type, const hlb_params* p, int64_t* voxel_of_site,
                          int32_t* canon_of_site, int32_t* nbr);

/* Run-length link records of a table (host only): the compressed form of nbr that the step
 * kernels read. A group is 32 consecutive internal sites (one warp). For group g and link q
 * the record rec[(g*n_links + (q-1))*4 .. +4] = { wall, runs, off0, off1 }:
 *   wall    bit l set: the entry of lane l is negative (solid or iolet: bounce-back target)
 *   runs    the non-wall lanes split into runs of lanes with consecutive entries (a wall
 *           lane or a jump in the entries ends a run). Bits 0..5: second = the lane at which
 *           run 1 starts, 32 if there is only one run (or none). Bit 6: there is a third run;
 *           then bits 7..11: third = the lane at which run 2 starts, and bits 12..31: the
 *           signed difference off2 - off1. All higher bits 0 without a third run.
 *   off0, off1: (entry of a lane of the run) - (internal index 32 g + l of that lane's own
 *           site), modulo 2^32, for run 0 and run 1; off1 = off0 when there is only one run
 * so that the entry of a non-wall lane l is 32 g + l + (l >= third ? off2 : l >= second ? off1 :
 * off0) (mod 2^32): the step kernels add the same delta to every lane's own index. A (g, q)
 * with more than three runs, or with a third run whose off2 - off1 does not fit 20 signed
 * bits, gets the sentinel { 0, 0xffffffff, 0, 0 } and the kernels read nbr for it instead.
 *   nbr: HOST [n_links][stride] as filled by hlb_preprocess_tables; stride a multiple of 32;
 *        n_links = Q - 1 = 14 or 18
 *   rec: HOST [stride/32][n_links][4] uint32, filled
 *   n_sentinel: number of (g, q) that got the sentinel (may be NULL) */
int hlb_preprocess_records(const int32_t* nbr, int32_t n_links, int64_t stride, uint32_t* rec,
                           int64_t* n_sentinel);

/* Interpolated-wall (BFL) tables of a geometry (host only): the site form hlb_set_wall_distance
 * builds for the step kernels, exposed so that it can be checked without a GPU. A link p
 * (1 .. n_links) of internal site i is interpolated when nbr[p-1][i] is a solid wall, the pull
 * source of opp(p) -- the site behind i -- is fluid, and 0 < d <= 1 is given for it, d =
 * d27[canon_of_site[i]][(1 - c_pz) * 9 + (1 - c_py) * 3 + (1 - c_px)] (the wall lies along -c_p).
 * opp(p) = ((p - 1) ^ 1) + 1, so links 2k + 1 and 2k + 2 form opposite pair k; the two links of a
 * pair are never both interpolated.
 *   index: HOST [stride/32][2] uint32 {bits, rank}: bit l of bits marks site 32 g + l as carrying
 *          an interpolated link; its row is rank + popcount(bits below l). May be NULL.
 *   coef:  HOST [coef_rows][row] doubles, row = ((n_links / 2 + 2) / 2) * 2 (8 for D3Q15, 10 for
 *          D3Q19): entries 0 .. n_links/2 - 1 are one coefficient per pair -- +(1 - 2d) for a
 *          d < 1/2 link (applied to the gathered value), -(1 - 1/(2d)) for a d >= 1/2 link (applied
 *          to the value written back), 0 without an interpolated link --, entry n_links/2 holds a
 *          64-bit word whose bit k is set when the link of pair k is 2k + 2 (else 2k + 1). May be
 *          NULL; else coef_rows must be at least the number of flagged sites (HLB_EINVAL).
 *   n_flagged, n_interpolated: sites with a row / interpolated links (may be NULL) */
int hlb_preprocess_bfl(const int32_t* nbr, const int32_t* canon_of_site, int32_t n_links, int64_t n_sites,
                       int64_t stride, const double* d27, uint32_t* index, double* coef, int64_t coef_rows,
                       int64_t* n_flagged, int64_t* n_interpolated);

#ifdef __cplusplus
}
#endif
#endif /* HLB_H_ */
