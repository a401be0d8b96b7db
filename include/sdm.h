/* sdm.h -- C ABI of libsdm: the super-droplet (particle-based) warm-rain step of
 * arxiv 1310.1905 (libcloudph++ 0.2, section 5) on one NVIDIA B200.
 *
 * The interface follows the paper's programming interface (PAPER.md :667-835,
 * Listings 5.1-5.7): options fixed at creation (opts_init_t), per-step options
 * (opts_t), array descriptors (arrinfo_t), a factory, step_sync / step_async
 * and the diag_* / outbuf methods.  C has no templates, so real_t is the
 * `real_bytes` field and backend_t is gone (CUDA only).
 *
 * Conventions
 *  - Every function returns SDM_OK (0) or a negative sdm_status; the message is
 *    available from sdm_last_error().  No exception crosses the boundary.
 *  - "DEVICE pointer" = memory of the CUDA device the context was created on,
 *    owned by the caller unless stated otherwise.  "HOST pointer" = ordinary
 *    host memory.  `stream` is a cudaStream_t passed as void* (NULL = legacy
 *    default stream).  Work is enqueued on that stream; functions documented
 *    as "blocking" synchronise with it.
 *  - Eulerian fields (th, rv, rhod, Courant numbers, outbuf) are IEEE double.  The real attributes of the
 *    super-droplets (rw2, rd3, kappa, x, y, z) are stored as double or float (real_bytes 8 or 4, the real_t of the
 *    paper's templates); the arithmetic is fp64 either way, values are rounded when stored.
 *  - There is no CPU fallback: sdm_create fails with SDM_ERR_NO_DEVICE when no
 *    sm_100 device is usable (PAPER.md :827 "does report an error").
 */
#ifndef SDM_H_
#define SDM_H_
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sdm_ctx sdm_ctx;

typedef enum {
  SDM_OK = 0,
  SDM_ERR_INVALID = -1,     /* bad argument (NULL, size, stride, option) */
  SDM_ERR_NO_DEVICE = -2,   /* no usable sm_100 CUDA device */
  SDM_ERR_CUDA = -3,        /* a CUDA runtime call or kernel failed */
  SDM_ERR_CAPACITY = -4,    /* more super-droplets than max_sd, or a cell holds more SDs than a CTA can sort */
  SDM_ERR_ORDER = -5        /* calls out of order (e.g. step_async without step_sync) */
} sdm_status;

/* PAPER.md Listing 5.3 (:722-726) has only `geometric`; BASELINE.json north_star adds the other two. */
typedef enum {
  SDM_KERNEL_GEOMETRIC = 0, /* eq. 28 with E = 1 */
  SDM_KERNEL_GOLOVIN = 1,   /* K = b (v_i + v_j) */
  SDM_KERNEL_HYDRO_TAB = 2  /* eq. 28 with E(r_large, r_small/r_large) bilinear from a table */
} sdm_kernel;

/* One lognormal mode of the initial dry-aerosol spectrum (eq. 3 :119, the same fields as blk_2m's
 * lognormal_mode_t :400-410).  dry_distros of Listing 5.2 (:703-708) maps kappa to a functor n(ln r_d); C has no
 * functors, so a spectrum is the sum of the modes that share one kappa, and distinct kappas are an external
 * mixture (:659) whose spectra share the super-droplets equally. */
typedef struct {
  double kappa;             /* hygroscopicity */
  double n_stp;             /* number concentration at STP [m^-3] */
  double r_mean;            /* mode radius [m] */
  double sigma_g;           /* geometric standard deviation (> 1) */
} sdm_lognormal_mode;

/* PAPER.md Listing 5.2 (:699-720) lgrngn::opts_init_t.  Copied by sdm_create. */
typedef struct {
  int nx, ny, nz;           /* Eulerian grid; 0 = dimension absent (:751: 0..3 Courant components) */
  double dx, dy, dz, dt;    /* grid steps [m] and time step [s]; an absent dimension still
                               contributes its d? to the cell volume dV = dx dy dz (2D: dy = 1 m; box: V) */
  double x0, y0, z0, x1, y1, z1; /* Lagrangian sub-domain (:713); used by sdm_init only; all zero = whole grid */
  double sd_conc_mean;      /* mean number of SDs per cell (:715); a sizing hint here */
  int kernel;               /* sdm_kernel */
  double golovin_b;         /* [1/s] for SDM_KERNEL_GOLOVIN */
  int n_eff_R, n_eff_q;     /* collision-efficiency table shape (HYDRO_TAB) */
  const double* eff_R;      /* HOST, n_eff_R collector radii [m], ascending */
  const double* eff_q;      /* HOST, n_eff_q radius ratios small/large, ascending */
  const double* eff_tab;    /* HOST, row-major [n_eff_R][n_eff_q] */
  uint64_t seed;            /* Philox-4x32-10 key (low word, high word) */
  int real_bytes;           /* 8 or 4: storage type of rw2, rd3, kappa, x, y, z (and of the arrays of
                               sdm_init_from_arrays / sdm_export_state) */
  int multi_coal;           /* 1: gamma = floor(p) + [u < frac(p)] (north_star); 0: gamma = [u < p] (PAPER.md :645) */
  uint64_t max_sd;          /* capacity in super-droplets (HBM is allocated once, at creation) */
  int n_modes;              /* dry_distros (:703-708): number of lognormal modes, 0..8 (0: sdm_init unavailable) */
  const sdm_lognormal_mode* modes; /* HOST, n_modes entries; copied */
  int open_x;               /* 0: x is periodic (PAPER.md :558).  1: this context is one slab of a domain decomposed along x
                               (SURVEY.md section 8e): SDs moved beyond x < 0 or x >= nx*dx keep their coordinate and must be
                               handed to the neighbour with sdm_pack_leavers before the next step_sync */
} sdm_opts_init;

/* PAPER.md Listing 5.1 (:677-689) lgrngn::opts_t */
typedef struct {
  int adve, sedi, cond, coal; /* process toggles */
  double RH_max;              /* RH limit for drop growth (:685) */
  int sstp_cond, sstp_coal;   /* numbers of substeps (:688) */
  double cond_adapt_tol;      /* 0 (default): every cell takes sstp_cond condensation substeps, as the paper does ("the number of
                                 subtimesteps is kept constant throughout the domain", :566).  > 0: the adaptive choice the paper
                                 plans (:566), per cell and step (reading R-adapt): with eps = |d r_v| / (r_v max(|RH - 1|,
                                 1e-3)), d r_v the vapour one explicit step of the cell's growth rates would take up (eq. 25), the cell
                                 takes the smallest divisor d of sstp_cond with d >= sstp_cond * eps / cond_adapt_tol substeps of dt / d.
                                 Changes results (by the time-discretisation error it trades); fp64-arithmetic condensation only
                                 (SDM_ERR_INVALID with sdm_set_cond_arith(ctx, 4)). */
  int coal_adapt_max;         /* 0 or 1 (default): every cell takes sstp_coal coalescence substeps.  > 1: the adaptive logic the paper
                                 plans (:645 "use the values of P_ij to control an adaptive timestep logic"; DESIGN.md reading
                                 R-adapt-coal): a cell takes sstp_coal * m substeps with new random pairs each, m = min(coal_adapt_max,
                                 ceil(P_max)), P_max the largest probability of eq. 27 among the pairs of its first grouping at
                                 dt / sstp_coal: enough for every such pair to have P <= 1.  Changes results wherever P_max > 1. */
} sdm_opts;

/* PAPER.md Listing 5.4 (:730-745) lgrngn::arrinfo_t: element (i,j,k) of the field lives at
 * data_zero[i*strides[0] + j*strides[1] + k*strides[2]] (strides in elements, one per PRESENT
 * dimension in x,y,z order; unused entries ignored).  data_zero == NULL means "argument omitted". */
typedef struct {
  double* data_zero;        /* DEVICE pointer to element (0,0,0) */
  int64_t strides[3];
} sdm_arrinfo;

typedef struct {
  uint64_t n_sd;            /* super-droplets in storage (live ones after the last step_sync) */
  uint64_t max_cell_count;  /* largest number of SDs in one cell at the last step_sync */
  uint64_t step;            /* completed steps */
  uint64_t kernel_launches; /* CUDA kernels launched by this context since creation */
  uint64_t pairs, collisions, near_ties; /* coalescence: candidate pairs, pairs with gamma > 0,
                                            pairs with |u - frac(p)| < 1e-12 (summed since creation) */
  uint64_t ill_posed;       /* condensation: SD-substeps that took the bracket branch of PAPER.md :579 */
  uint64_t newton_iters;    /* condensation: growth-rate evaluations (summed) */
  uint64_t sd_substeps;     /* condensation: SD-substeps solved */
  uint64_t cond_slow;       /* condensation: SD-substeps deferred to the second (compacted) solver pass */
  uint64_t recycled;        /* zero-multiplicity SDs recycled (sdm_set_recycle) */
  /* launch configuration chosen by the last step (it follows the cell occupancy, which drifts as rain forms) */
  uint64_t cond_variant;    /* condensation kernel: 1, 2, 3 = tile kernels of 800 / 1280 / 4096 SD slots, 0 = one cell per CTA in
                               place in global memory; 100 + v: the fp32-arithmetic tile kernel v */
  uint64_t cond_tile_cells; /* cells per condensation tile */
  uint64_t coal_tile_cells; /* cells per tile of the fused coalescence + movement kernel; 0 = the per-cell kernel ran */
  uint64_t host_syncs;      /* host synchronisations inside step_sync / step_async since creation */
} sdm_stats_t;

/* factory() of Listing 5.7 (:800-808).  Allocates all device memory for max_sd super-droplets on
 * the current CUDA device.  Blocking. */
int sdm_create(const sdm_opts_init* opts, sdm_ctx** out);
void sdm_destroy(sdm_ctx* ctx);
/* message of the last failed call on ctx (ctx == NULL: of the last failed sdm_create); library-owned */
const char* sdm_last_error(const sdm_ctx* ctx);

/* init() of Listing 5.5 (:759-766): the initialisation of PAPER.md section 5.1.6 (:653-665).  Creates
 * round(sd_conc_mean * cells of the Lagrangian domain) super-droplets with ids 0..N-1: positions uniform in
 * [x0,x1) x [y0,y1) x [z0,z1) (:655); ln r_d uniform between the limits at which an SD stands for at least one
 * particle (:657); multiplicity = n(ln r_d) * range / SDs per cell * dV * rho_d / rho_STP, rounded, at least 1
 * (:659); wet radius in equilibrium (zero growth rate in eq. 20) with min(RH, 0.95) of the SD's cell (:661-665);
 * theta and r_v are not changed (:663).  Random numbers: Philox-4x32-10 with the context's seed, counter
 * (id, 0, 0, tag), tag 2, 3, 4, 5 = x, y, z, ln r_d.  th, rv, rhod are mandatory, the Courant components are
 * those of the present dimensions (:751) and may be omitted (zero flow); all are DEVICE arrays, copied or read
 * before the call returns.  Fails with SDM_ERR_INVALID without modes, SDM_ERR_CAPACITY if N > max_sd.  Blocking. */
int sdm_init(sdm_ctx* ctx, sdm_arrinfo th, sdm_arrinfo rv, sdm_arrinfo rhod, sdm_arrinfo rhod_courant_1,
             sdm_arrinfo rhod_courant_2, sdm_arrinfo rhod_courant_3, void* stream);
/* The limits of ln r_d chosen by the rule of :657 for spectrum g (0-based, in order of first appearance of its
 * kappa among the modes); HOST outputs. */
int sdm_init_range(const sdm_ctx* ctx, int g, double* lnr_lo, double* lnr_hi);

/* Load a particle population (parity tests, the box set-up, checkpoint restart) instead of the
 * paper's init() (:759-766).  rhod and the Courant components (rho_d times Courant number on the
 * Arakawa-C grid, shapes (nx+1) x ny x nz, nx x (ny+1) x nz, nx x ny x (nz+1); in 2D the second
 * component is the vertical one and the third is omitted, :751) are copied into library-owned dense
 * arrays.  n (multiplicity, uint64), rw2 (wet radius squared), rd3 (dry radius cubed), kappa, x, y,
 * z, id (unique uint32) are DEVICE arrays of N elements, copied; coordinates of absent dimensions
 * may be NULL; rw2 .. z are arrays of real_bytes-sized reals.  Positions must lie inside the domain.  Blocking. */
int sdm_init_from_arrays(sdm_ctx* ctx, sdm_arrinfo rhod, sdm_arrinfo rhod_courant_1,
                         sdm_arrinfo rhod_courant_2, sdm_arrinfo rhod_courant_3, uint64_t N,
                         const uint64_t* n, const void* rw2, const void* rd3, const void* kappa,
                         const void* x, const void* y, const void* z, const uint32_t* id, void* stream);

/* step_sync() of Listing 5.5 (:768-775, :816): the part of a step that alters the Eulerian fields.
 * Removes N = 0 SDs, sorts the SDs by (cell, Philox key, id), and if opts->cond integrates
 * opts->sstp_cond condensation substeps (eq. 17-26).  th and rv are read and OVERWRITTEN (final when
 * the work enqueued on `stream` completes).  Courant components and rhod may be omitted
 * (data_zero == NULL) when unchanged since initialisation (:816).  Blocks the host only until the
 * sort histogram is known (it sizes the cell-resident launches). */
int sdm_step_sync(sdm_ctx* ctx, const sdm_opts* opts, sdm_arrinfo th, sdm_arrinfo rv,
                  sdm_arrinfo rhod_courant_1, sdm_arrinfo rhod_courant_2, sdm_arrinfo rhod_courant_3,
                  sdm_arrinfo rhod, void* stream);

/* step_async() of Listing 5.5 (:776-777, :816): coalescence (eq. 27-28), advection (eq. 16) and
 * sedimentation; only enqueues.  Must follow a step_sync of the same step. */
int sdm_step_async(sdm_ctx* ctx, const sdm_opts* opts, void* stream);
/* Waits for the last step_async and returns its rain flux through the bottom of the domain
 * (:816), as the mass of water that left during that step [kg]. */
int sdm_step_async_result(sdm_ctx* ctx, double* rain_flux);

/* The same step for a caller whose Eulerian fields live in HOST memory (the paper's CPU solver,
 * :845-848): copies th, rv (dense C order, nx*ny*nz doubles, pinned or pageable) to the device,
 * runs step_sync, copies them back, runs step_async.  The copies travel on a stream of the library's own: in while
 * the sort runs (the condensation kernel waits for them), out while coalescence and movement run (with pinned
 * buffers; pageable ones serialise in the driver).  Blocking; *rain_flux as above. */
int sdm_step_host(sdm_ctx* ctx, const sdm_opts* opts, double* th_host, double* rv_host,
                  double* rain_flux, void* stream);

/* diag_* of Listing 5.5 (:779-788, :818-823).  *_rng selects r in [r_mi, r_mx) for the following
 * *_mom calls; *_mom(k) computes eq. 29 per cell into the output buffer; sd_conc counts SDs per
 * cell.  Cells are those of the SDs' current positions.  Enqueue on `stream`. */
int sdm_diag_sd_conc(sdm_ctx* ctx, void* stream);
int sdm_diag_dry_rng(sdm_ctx* ctx, double r_mi, double r_mx);
int sdm_diag_wet_rng(sdm_ctx* ctx, double r_mi, double r_mx);
int sdm_diag_dry_mom(sdm_ctx* ctx, int k, void* stream);
int sdm_diag_wet_mom(sdm_ctx* ctx, int k, void* stream);
/* outbuf() (:788, :823): DEVICE pointer to nx*ny*nz doubles in dense C order, library-owned, valid
 * until the next diag_* call; contents are final when the stream work of that diag call completes. */
const double* sdm_outbuf(sdm_ctx* ctx);

/* Parity / checkpoint access.  sdm_n_sd: number of SDs in storage (blocking).  sdm_export_state:
 * copies the SoA state in storage order into DEVICE arrays of at least sdm_n_sd elements (NULL =
 * skip that attribute); SDs whose multiplicity reached 0 during the last step are still present
 * until the next step_sync.  sdm_export_order: after step_sync, the ids in sorted (cell, key, id)
 * order and the nx*ny*nz+1 segment offsets (DEVICE arrays).  All enqueue on `stream`. */
int sdm_n_sd(sdm_ctx* ctx, uint64_t* n_sd);
/* sdm_n_live: the name SURVEY.md section 8(b) gives this call; the same number (after step_sync every SD in storage is
 * live: the compaction of PAPER.md :641 is folded into the sort). */
int sdm_n_live(sdm_ctx* ctx, uint64_t* n_live);
int sdm_export_state(sdm_ctx* ctx, uint64_t* n, void* rw2, void* rd3, void* kappa,
                     void* x, void* y, void* z, uint32_t* id, void* stream);
int sdm_export_order(sdm_ctx* ctx, uint32_t* ids_sorted, uint32_t* seg_start, void* stream);
/* Counters (blocking: synchronises the context's last stream). */
int sdm_stats(sdm_ctx* ctx, sdm_stats_t* out);
/* Per-stage device timing.  With timing enabled every stage of step_sync / step_async is bracketed by
 * CUDA events on the launching stream.  sdm_stage_times synchronises that stream and returns, per
 * sdm_stage, the summed elapsed milliseconds and the number of timed launches since the last reset
 * (ms and launches: HOST arrays of SDM_N_STAGES elements; launches may be NULL). */
typedef enum {
  SDM_STAGE_HIST = 0,      /* a0-a1: cell index + histogram (compaction) */
  SDM_STAGE_SCAN = 1,      /* a2: segment offsets */
  SDM_STAGE_SCATTER = 2,   /* a3: reorder the state by cell */
  SDM_STAGE_RANK = 3,      /* a2: (Philox key, id) order inside each cell */
  SDM_STAGE_COND = 4,      /* a4: condensation substeps */
  SDM_STAGE_COAL_MOVE = 5, /* a5-a6: coalescence + advection + sedimentation */
  SDM_STAGE_RECYCLE = 6,   /* recycling of zero-multiplicity SDs (only with sdm_set_recycle) */
  SDM_N_STAGES = 7
} sdm_stage;
int sdm_set_timing(sdm_ctx* ctx, int enable);
int sdm_stage_times(sdm_ctx* ctx, double* ms, uint64_t* launches, int reset);
/* PAPER.md :641, :651: "Particles with zero multiplicity are 'recycled' at the begining of each timestep.  The
 * recycling procedure first looks for computational particles with highest multiplicites and then assignes their
 * properties to the recycled particles halving the multiplicity."  on = 0 (default): zero-multiplicity SDs are
 * removed by the compaction of step_sync (BASELINE.json north_star).  on = 1: at the beginning of step_sync, with k
 * zero-multiplicity SDs in storage, the first k SDs in the order (multiplicity descending, id ascending) among those
 * with multiplicity >= 2 give: the i-th of them to the zero-multiplicity SD of i-th smallest id, which takes its
 * r_w^2, r_d^3, kappa and position, keeps its own id and gets floor(N/2), the donor keeping N - floor(N/2); with fewer
 * donors than k the rest is compacted away.  The first call with on = 1 allocates 32 bytes of scratch per SD of
 * capacity (SDM_ERR_CUDA if that fails).  Adds one host synchronisation to step_sync. */
int sdm_set_recycle(sdm_ctx* ctx, int on);
/* Overrides the step counter used in the Philox counters (restart from a checkpoint, parity). */
int sdm_set_step(sdm_ctx* ctx, uint64_t step);
/* Tuning override for tests: threads cooperating on one cell in the cell-resident kernels
 * (0 = automatic; 4, 8, 16, 32 = sub-warp groups; 256 = one CTA per cell). */
int sdm_set_group_size(sdm_ctx* ctx, int group);
/* Arithmetic of the condensation sweep (a4).  8 (default): fp64, radii within 1e-9 of the oracle.  4: fp32 -- the
 * `real_t = float` of the paper's templates (PAPER.md :747; its timings are single precision, :908) -- allowed with
 * real_bytes = 4 only (SDM_ERR_INVALID otherwise); radii within 1e-4 of the fp64 oracle started from the same
 * fp32-representable state (BASELINE.json north_star).  The cells' thermodynamics, the feedback on th and rv (eq. 25-26)
 * and every SD whose bracket may hold several roots or whose iterate leaves the bracket stay fp64.  One crowded cell
 * beyond 4096 SDs is solved in fp64 either way. */
int sdm_set_cond_arith(sdm_ctx* ctx, int bytes);
/* Tuning override: growth-rate evaluations the dense condensation sweep spends on an SD before deferring it
 * to the compacted second pass (1..200, default 4).  Does not change results beyond the solver tolerance. */
int sdm_set_cond_kfast(sdm_ctx* ctx, int kfast);

/* Domain decomposition along x (PAPER.md :843 "in case of domain decomposition"): every stage but the
 * movement of eq. 16 is local to a cell, so a rank owns a slab of columns (a context created with open_x = 1 on its own nx
 * columns, coordinates relative to the slab) and after step_async exchanges the SDs that crossed its two faces.
 * sdm_sd_buffers: one SoA set of DEVICE arrays, caller-owned; rw2 .. z of real_bytes-sized reals; y, z may be NULL when absent. */
typedef struct {
  uint64_t* n;
  void *rw2, *rd3, *kappa, *x, *y, *z;
  uint32_t* id;
} sdm_sd_buffers;
/* Moves every live SD with x < 0 into `left` and every one with x >= nx*dx into `right` (coordinates unchanged, any order)
 * and marks its slot N = 0 (the next step_sync compacts it away).  cap: elements each buffer array holds.  *n_left,
 * *n_right: HOST outputs.  If either count exceeds cap nothing is moved and SDM_ERR_CAPACITY is returned with the counts
 * set.  To be called after step_async of the step; waits for it.  Blocking. */
int sdm_pack_leavers(sdm_ctx* ctx, uint64_t cap, const sdm_sd_buffers* left, const sdm_sd_buffers* right, uint64_t* n_left,
                     uint64_t* n_right, void* stream);
/* Appends N SDs (a neighbour's `right` list with x_shift = minus that neighbour's slab width, or its `left` list with
 * x_shift = plus this slab's width) behind the SDs in storage, x + x_shift being their coordinate in this slab.  Ids travel
 * with the SDs (they key the Philox streams).  SDM_ERR_CAPACITY beyond max_sd.  Enqueues on `stream`. */
int sdm_unpack_arrivals(sdm_ctx* ctx, uint64_t N, const sdm_sd_buffers* in, double x_shift, void* stream);

/* The "prototype transport equation solver" of PAPER.md Figure 7 and section 5.2.2 (:831-852): one first-order upstream
 * (donor-cell; :219-235) step of the scalar field psi (DEVICE, strided as the other Eulerian fields; overwritten) with the
 * rho_d x Courant arrays and rho_d the context holds since sdm_init* / the last step_sync (:751): psi' = psi - sum over the
 * dimensions of (F_hi - F_lo) / rho_d, F = max(rho_d C, 0) psi_donor-side + min(rho_d C, 0) psi_other at each face; periodic
 * in x and y, psi continued by its boundary value below and above.  This is what the host model does to theta and r_v
 * between step_sync and the next step_sync, on a stream of its own, while step_async runs (:816); the library's own step
 * never calls it.  Enqueues 2 kernels on `stream`; the first call allocates nx*ny*nz doubles of scratch. */
int sdm_upstream_advect(sdm_ctx* ctx, sdm_arrinfo psi, void* stream);

/* Measurement aid, not part of the step (the condensation kernel of PAPER.md eq. 17-24, which
 * "takes most of the simulation time" (:912), is bound by fp64 arithmetic, so its roofline needs a MEASURED fp64 peak):
 * runs a register-only kernel of independent fp64 FMA chains on every SM of the current device and returns the best of
 * five timed launches (CUDA events on `stream`).  *fma_tflops: 2 flop per FMA, in TFLOP/s.  *dfma_per_clk_per_sm (may be
 * NULL): thread-level FMAs retired per SM clock per SM, from clock64() inside the kernel (64 on sm_100).  HOST outputs;
 * allocates and frees 1.3 MB of device memory.  Blocking.  SDM_ERR_NO_DEVICE without a device. */
int sdm_measure_fp64_peak(double* fma_tflops, double* dfma_per_clk_per_sm, void* stream);

/* An entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  The operation is the scan of the counting sort by cell (SURVEY.md section 8
 * row a2; PAPER.md :641, the super-droplets are sorted by cell before the pairs are drawn): from the per-cell numbers of
 * super-droplets count[0..ncell) it writes the start of every cell's segment in the sorted order,
 *     seg[c] = count[0] + ... + count[c-1]   (c = 0..ncell;  seg[ncell] = the total),
 * exactly (32-bit unsigned arithmetic, as in the step; the total must fit 32 bits).
 * count: DEVICE, ncell words, read only (the step's own scan zeroes its histogram; this one does not).  seg: DEVICE,
 * ncell + 1 words, written.  Both caller-owned; they must not overlap.  Needs no context.  Enqueues 3 kernels on `stream`
 * of the current device and returns; no host synchronisation, no cudaMalloc / cudaFree / allocating library routine.
 * The block sums it needs live in a static device array of 16 KB inside the library (held by every GPU that loads the
 * library, until the process exits), which bounds the size: ncell <= SDM_NOALLOC_MAX_CELLS, beyond which the call is
 * refused with SDM_ERR_CAPACITY and enqueues nothing.  SDM_ERR_INVALID for NULL pointers or ncell < 0, SDM_ERR_NO_DEVICE
 * without a device, SDM_ERR_CUDA if a launch fails; the message is available from sdm_noalloc_last_error() (per host thread).
 * All calls on one device share that array, and it keeps the last call's contents (nothing in it has to start at zero:
 * every call overwrites what it reads).  Calls that OVERLAP on the GPU - different streams, or host threads, on the same
 * device without an ordering between them - race on it and give wrong offsets; calls on one stream are safe.
 * sdm_cell_offsets_noalloc_setup(): looks up the array's device address for the CURRENT device (cudaGetSymbolAddress, once
 * per device).  The entry point does this itself on its first call on a device; call the set-up beforehand, with the
 * device current, where that first call would come at a bad time (before starting a graph capture). */
#define SDM_NOALLOC_MAX_CELLS 16777216LL
int sdm_cell_offsets_noalloc_setup(void);
int sdm_cell_offsets_noalloc(const uint32_t* count, int64_t ncell, uint32_t* seg, void* stream);
const char* sdm_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SDM_H_ */
