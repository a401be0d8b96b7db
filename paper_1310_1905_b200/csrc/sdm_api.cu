// C ABI of libsdm (include/sdm.h): context, memory, launch sizing.  All arithmetic of the step runs in
// the kernels of sdm_sort.cu, sdm_cond.cu, sdm_coal_move.cu and sdm_diag.cu; there is no CPU path.
#include "../../include/sdm.h"
#include "sdm_kernels.cuh"
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

using namespace sdm;

namespace {
thread_local std::string g_create_error;
constexpr size_t kSmemLimit = 200 * 1024;   // dynamic shared memory we are willing to ask for per CTA
#ifndef SDM_COND_TILE_TARGET
#define SDM_COND_TILE_TARGET 660.0
#endif
constexpr double kCondTileTarget = SDM_COND_TILE_TARGET;   // SDs per condensation tile (mean); 5 sigma above fits the 800 slots of k_cond4
#ifndef SDM_SMALL_WAVES
#define SDM_SMALL_WAVES 1.0
#endif
#ifndef SDM_COND32_TILE_TARGET
#define SDM_COND32_TILE_TARGET 660.0
#endif
constexpr double kCond32TileTarget = SDM_COND32_TILE_TARGET;   // the same for the fp32-arithmetic kernel (sdm_set_cond_arith)
constexpr double kCondMaxCpb = 128.0;       // one thread per cell of the tile
// SD slots of the small tile kernels (sdm_cond.cu: SDM_COND_CAP, SDM_COND32_CAP)
#ifndef SDM_COND_TILE_SLOTS
#define SDM_COND_TILE_SLOTS 800.0
#endif
#ifndef SDM_COND32_TILE_SLOTS
#define SDM_COND32_TILE_SLOTS 800.0
#endif
}

struct sdm_ctx {
  sdm_opts_init o{};
  Grid g{};
  int device = 0;
  int n_sm = 148;
  u64 cap_sd = 0;
  SdArrays buf[2]{};
  int cur = 0;
  u32 *cell = nullptr, *off = nullptr, *count = nullptr, *blocksum = nullptr, *seg = nullptr;
  u16* rank = nullptr;
  u32* d_info = nullptr;     // [0],[1] slot counts (ping-pong), [2] max cell count, [3] error flag, [4..7] tile maxima
  u32* h_info = nullptr;     // pinned mirror
  int cn = 0;                // which of d_info[0..1] is current
  CellFields cf{};
  double *cx = nullptr, *cy = nullptr, *cz = nullptr;
  double* outbuf = nullptr;
  double* adv_tmp = nullptr;     // scratch of sdm_upstream_advect
  double* flux_slots = nullptr;
  double* flux_part = nullptr;   // per-CTA rain flux of k_coal_move_tile
  int n_flux_part = 0;
  bool hist_valid = false;       // cell, off, count of the next step were written by the last step_async
  double* d_flux = nullptr;  // [0] last step, [1] total, [2] the device error flag of the step (copied by k_flux_sum)
  unsigned long long* cnt_mem = nullptr;
  Counters cnt{};
  CoalParams kp{};
  InitParams ip{};           // dry spectra and the limits of :657, prepared at creation
  bool have_modes = false;
  double *d_effR = nullptr, *d_effq = nullptr, *d_efftab = nullptr;
  double *th_dense = nullptr, *rv_dense = nullptr;   // for sdm_step_host
  u64 nslots = 0;            // host-known number of slots in use
  u64 max_nc = 0;
  u32 tile_max[4] = {0, 0, 0, 0};   // most populated tile for the 4 candidate tile sizes of the last step_sync
  u64 step = 0;
  bool synced = false;       // step_sync of the current step done
  bool have_order = false;
  int G = 32;                // group size chosen by the last step_sync
  int group_override = 0;
  int cond_cpb0 = 1;         // candidate cells per condensation tile (halved up to 3 times if a tile overflows)
  int kfast = 4;
  int cond_arith = 8;        // 8: fp64 arithmetic in the condensation sweep; 4: fp32 (real_bytes == 4 only)
  cudaEvent_t ev_info = nullptr, ev_async = nullptr;
  // sdm_step_host: th, rv travel on a stream of their own, overlapped with the sort (in) and with coalescence + movement (out)
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_copy_go = nullptr, ev_h2d = nullptr, ev_fields = nullptr;
  bool wait_h2d = false;
  cudaStream_t last_stream = nullptr;
  u64 launches = 0;
  u64 host_syncs = 0;
  int last_cond_variant = 0, last_cond_cpb = 0, last_coal_cpb = 0;
  bool mv_valid = false;     // cf.mv matches cf.rhod and the Courant fields
  double dry_lo = 0, dry_hi = 1e300, wet_lo = 0, wet_hi = 1e300;
  // optional per-stage timing with CUDA events on the launching stream (sdm_set_timing)
  bool timing = false;
  std::vector<cudaEvent_t> tev[SDM_N_STAGES];   // start/stop pairs not yet folded into t_ms
  double t_ms[SDM_N_STAGES] = {0, 0, 0, 0, 0, 0, 0};
  uint64_t t_cnt[SDM_N_STAGES] = {0, 0, 0, 0, 0, 0, 0};
  // recycling (sdm_set_recycle): two item lists, histogram + info words on the device, pinned info mirror
  bool recycle = false;
  RecItem *rec_dead = nullptr, *rec_cand = nullptr;
  u32 *rec_hist = nullptr, *rec_info = nullptr, *h_rec = nullptr;
  u64 recycled = 0;
  std::vector<cudaEvent_t> ev_pool;
  std::string err;
};

namespace {

// the state arrays are stored in the double-typed struct; with real_bytes == 4 the same pointers are floats
template <typename R> const SdArraysT<R>& view(const SdArrays& b) { return reinterpret_cast<const SdArraysT<R>&>(b); }

int fail(sdm_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_create_error = msg;
  return code;
}
#define CK(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e__ = (call);                                                                      \
    if (e__ != cudaSuccess)                                                                        \
      return fail(ctx, SDM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e__));         \
  } while (0)

template <typename T>
cudaError_t dalloc(T** p, size_t n) { return cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(T)); }

Field make_field(const sdm_ctx* c, const sdm_arrinfo& a) {
  Field f{a.data_zero, 0, 0, 0};
  int idx = 0;
  if (c->g.hx) f.s0 = a.strides[idx++];
  if (c->g.hy) f.s1 = a.strides[idx++];
  if (c->g.hz) f.s2 = a.strides[idx++];
  return f;
}

// Courant component q (0-based among the PRESENT dimensions, PAPER.md :751) -> dense library copy
int copy_courants(sdm_ctx* ctx, const sdm_arrinfo* comps, cudaStream_t st) {
  const Grid& g = ctx->g;
  int q = 0;
  for (int dim = 0; dim < 3; ++dim) {
    const bool present = dim == 0 ? g.hx : dim == 1 ? g.hy : g.hz;
    if (!present) continue;
    const sdm_arrinfo& a = comps[q++];
    if (!a.data_zero) continue;
    double* dst = dim == 0 ? ctx->cx : dim == 1 ? ctx->cy : ctx->cz;
    launch_dense_copy(make_field(ctx, a), dst, g.NX + (dim == 0), g.NY + (dim == 1), g.NZ + (dim == 2), st);
    ctx->launches++;
    ctx->mv_valid = false;
  }
  CK(cudaGetLastError());
  return SDM_OK;
}

// stage timers: t_begin/t_end bracket the launches of one stage with events on the stream
void t_begin(sdm_ctx* c, int stage, cudaStream_t st) {
  if (!c->timing) return;
  cudaEvent_t e;
  if (!c->ev_pool.empty()) { e = c->ev_pool.back(); c->ev_pool.pop_back(); }
  else if (cudaEventCreate(&e) != cudaSuccess) return;
  cudaEventRecord(e, st);
  c->tev[stage].push_back(e);
}
void t_end(sdm_ctx* c, int stage, cudaStream_t st) {
  if (!c->timing || (c->tev[stage].size() & 1) == 0) return;
  cudaEvent_t e;
  if (!c->ev_pool.empty()) { e = c->ev_pool.back(); c->ev_pool.pop_back(); }
  else if (cudaEventCreate(&e) != cudaSuccess) { c->ev_pool.push_back(c->tev[stage].back()); c->tev[stage].pop_back(); return; }
  cudaEventRecord(e, st);
  c->tev[stage].push_back(e);
}
void t_fold(sdm_ctx* c) {   // caller has synchronised the stream
  for (int s = 0; s < SDM_N_STAGES; ++s) {
    auto& v = c->tev[s];
    for (size_t k = 0; k + 1 < v.size(); k += 2) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, v[k], v[k + 1]) == cudaSuccess) { c->t_ms[s] += ms; c->t_cnt[s]++; }
    }
    for (cudaEvent_t e : v) c->ev_pool.push_back(e);
    v.clear();
  }
  cudaGetLastError();
}

// The rank kernels of step_sync raise d_info[3] when a cell holds more SDs than the launch was sized for; the step's device work
// is complete when this is called, so the flag is that of THIS step.  Cleared once reported.
int check_device_flag(sdm_ctx* ctx, const char* who, double* rain_flux) {
  double h[3] = {0, 0, 0};   // flux of the step, total, error flag: one read-back
  CK(cudaMemcpy(h, ctx->d_flux, sizeof(h), cudaMemcpyDeviceToHost));
  if (rain_flux) *rain_flux = h[0];
  if (h[2] == 0.0) return SDM_OK;
  cudaMemset(ctx->d_info + 3, 0, sizeof(u32));
  return fail(ctx, SDM_ERR_CUDA, std::string(who) + ": device-side error flag set (a cell outgrew the launch its ranks were sized for)");
}

int pick_group(const sdm_ctx* c, double mean) {
  if (c->group_override) return c->group_override;
  if (mean < 12.0) return 4;
  if (mean < 28.0) return 8;
  if (mean < 80.0) return 16;
  if (mean < 400.0) return 32;
  return 256;
}
int ng_of(int G) { return (G <= 32 ? 128 : G) / G; }

}  // namespace

extern "C" {

const char* sdm_last_error(const sdm_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int sdm_create(const sdm_opts_init* o, sdm_ctx** out) {
  sdm_ctx* ctx = nullptr;
  if (!o || !out) return fail(nullptr, SDM_ERR_INVALID, "sdm_create: NULL argument");
  *out = nullptr;
  if (o->real_bytes != 8 && o->real_bytes != 4) return fail(nullptr, SDM_ERR_INVALID, "sdm_create: real_bytes must be 8 or 4");
  if (o->nx < 0 || o->ny < 0 || o->nz < 0 || !(o->dx > 0) || !(o->dy > 0) || !(o->dz > 0) || !(o->dt > 0))
    return fail(nullptr, SDM_ERR_INVALID, "sdm_create: grid sizes must be >= 0 and dx, dy, dz, dt > 0");
  if (o->kernel < 0 || o->kernel > 2) return fail(nullptr, SDM_ERR_INVALID, "sdm_create: unknown kernel");
  if (o->kernel == SDM_KERNEL_HYDRO_TAB && (o->n_eff_R < 2 || o->n_eff_q < 2 || !o->eff_R || !o->eff_q || !o->eff_tab))
    return fail(nullptr, SDM_ERR_INVALID, "sdm_create: hydro_tab kernel needs an efficiency table of at least 2 x 2");
  if (o->max_sd == 0 || o->max_sd >= 0xFFFFFFF0ull)
    return fail(nullptr, SDM_ERR_INVALID, "sdm_create: max_sd must be in [1, 2^32 - 16)");
  const long long ncell = (long long)std::max(o->nx, 1) * std::max(o->ny, 1) * std::max(o->nz, 1);
  if (ncell >= (1ll << 31) - 8) return fail(nullptr, SDM_ERR_INVALID, "sdm_create: too many cells");
  int ndev = 0, dev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(nullptr, SDM_ERR_NO_DEVICE, "sdm_create: no CUDA device (libsdm has no CPU fallback)");
  }
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
    return fail(nullptr, SDM_ERR_NO_DEVICE, "sdm_create: cannot query the current CUDA device");
  if (prop.major != 10)
    return fail(nullptr, SDM_ERR_NO_DEVICE, std::string("sdm_create: device '") + prop.name + "' is not sm_100 (B200)");

  ctx = new sdm_ctx();
  ctx->o = *o;
  ctx->device = dev;
  ctx->n_sm = prop.multiProcessorCount;
  Grid& g = ctx->g;
  g.NX = std::max(o->nx, 1); g.NY = std::max(o->ny, 1); g.NZ = std::max(o->nz, 1);
  g.hx = o->nx > 0; g.hy = o->ny > 0; g.hz = o->nz > 0;
  g.open_x = (o->open_x && g.hx) ? 1 : 0;
  g.ncell = (int)ncell;
  g.dx = o->dx; g.dy = o->dy; g.dz = o->dz; g.dt = o->dt;
  g.dV = o->dx * o->dy * o->dz;
  g.X = o->dx * g.NX; g.Y = o->dy * g.NY; g.Z = o->dz * g.NZ;
  ctx->cap_sd = o->max_sd;
  const size_t N = (size_t)o->max_sd;
  auto bail = [&](cudaError_t e, const char* what) {
    std::string m = std::string("sdm_create: ") + what + ": " + cudaGetErrorString(e);
    sdm_destroy(ctx);
    return fail(nullptr, SDM_ERR_CUDA, m);
  };
  cudaError_t e;
  for (int b = 0; b < 2; ++b) {
    SdArrays& a = ctx->buf[b];
    // 4 elements to spare: the bulk copies of k_coal_move_tile fetch whole 16-byte units around a tile's run
    const size_t NR = (o->real_bytes == 8 ? N : (N + 1) / 2) + 4;   // doubles that hold N reals
    if ((e = dalloc(&a.n, N + 4)) || (e = dalloc(&a.rw2, NR)) || (e = dalloc(&a.rd3, NR)) || (e = dalloc(&a.kappa, NR)) ||
        (e = dalloc(&a.x, g.hx ? NR : 4)) || (e = dalloc(&a.y, g.hy ? NR : 4)) || (e = dalloc(&a.z, g.hz ? NR : 4)) ||
        (e = dalloc(&a.id, N + 4)))
      return bail(e, "particle state");
  }
  const int nb = scan_num_blocks(g.ncell);
  if ((e = dalloc(&ctx->cell, N)) || (e = dalloc(&ctx->off, N)) || (e = dalloc(&ctx->rank, N + 8)) ||
      (e = dalloc(&ctx->count, (size_t)g.ncell)) || (e = dalloc(&ctx->blocksum, (size_t)nb)) ||
      (e = dalloc(&ctx->seg, (size_t)g.ncell + 1)) || (e = dalloc(&ctx->d_info, 8)) ||
      (e = dalloc(&ctx->cf.rhod, (size_t)g.ncell)) || (e = dalloc(&ctx->cf.eta, (size_t)g.ncell)) ||
      (e = dalloc(&ctx->cf.rho_a, (size_t)g.ncell)) || (e = dalloc(&ctx->outbuf, (size_t)g.ncell)) ||
      (e = dalloc(&ctx->th_dense, (size_t)g.ncell)) || (e = dalloc(&ctx->rv_dense, (size_t)g.ncell)) ||
      (e = dalloc(&ctx->cx, (size_t)(g.NX + 1) * g.NY * g.NZ)) || (e = dalloc(&ctx->cy, (size_t)g.NX * (g.NY + 1) * g.NZ)) ||
      (e = dalloc(&ctx->cz, (size_t)g.NX * g.NY * (g.NZ + 1))) || (e = dalloc(&ctx->flux_slots, NSLOT)) ||
      (e = dalloc(&ctx->flux_part, (size_t)g.ncell)) || (e = dalloc(&ctx->cf.mv, (size_t)6 * g.ncell)) ||
      (e = dalloc(&ctx->d_flux, 4)) || (e = dalloc(&ctx->cnt_mem, N_COUNTERS * NSLOT)))
    return bail(e, "scratch");
  ctx->cf.cx = ctx->cx; ctx->cf.cy = ctx->cy; ctx->cf.cz = ctx->cz;
  if ((e = cudaMallocHost((void**)&ctx->h_info, 8 * sizeof(u32)))) return bail(e, "pinned info");
  if ((e = cudaMemset(ctx->count, 0, sizeof(u32) * g.ncell)) || (e = cudaMemset(ctx->seg, 0, sizeof(u32) * ((size_t)g.ncell + 1))) ||
      (e = cudaMemset(ctx->d_info, 0, 8 * sizeof(u32))) ||
      (e = cudaMemset(ctx->cx, 0, sizeof(double) * (size_t)(g.NX + 1) * g.NY * g.NZ)) ||
      (e = cudaMemset(ctx->cy, 0, sizeof(double) * (size_t)g.NX * (g.NY + 1) * g.NZ)) ||
      (e = cudaMemset(ctx->cz, 0, sizeof(double) * (size_t)g.NX * g.NY * (g.NZ + 1))) ||
      (e = cudaMemset(ctx->flux_slots, 0, sizeof(double) * NSLOT)) || (e = cudaMemset(ctx->d_flux, 0, 4 * sizeof(double))) ||
      (e = cudaMemset(ctx->cnt_mem, 0, sizeof(unsigned long long) * N_COUNTERS * NSLOT)) ||
      (e = cudaMemset(ctx->outbuf, 0, sizeof(double) * g.ncell)))
    return bail(e, "memset");
  ctx->cnt.pairs = ctx->cnt_mem; ctx->cnt.collisions = ctx->cnt_mem + NSLOT; ctx->cnt.near_ties = ctx->cnt_mem + 2 * NSLOT;
  ctx->cnt.ill_posed = ctx->cnt_mem + 3 * NSLOT; ctx->cnt.f_evals = ctx->cnt_mem + 4 * NSLOT; ctx->cnt.sd_substeps = ctx->cnt_mem + 5 * NSLOT;
  ctx->cnt.cond_slow = ctx->cnt_mem + 6 * NSLOT;
  CoalParams& kp = ctx->kp;
  kp.kernel = o->kernel; kp.multi_coal = o->multi_coal; kp.golovin_b = o->golovin_b;
  kp.seed_lo = (u32)o->seed; kp.seed_hi = (u32)(o->seed >> 32);
  kp.n_eff_R = 0; kp.n_eff_q = 0;
  if (o->kernel == SDM_KERNEL_HYDRO_TAB) {
    kp.n_eff_R = o->n_eff_R; kp.n_eff_q = o->n_eff_q;
    for (int t = 1; t < o->n_eff_R; ++t) if (!(o->eff_R[t] > o->eff_R[t - 1])) { sdm_destroy(ctx); return fail(nullptr, SDM_ERR_INVALID, "sdm_create: eff_R must ascend"); }
    for (int t = 1; t < o->n_eff_q; ++t) if (!(o->eff_q[t] > o->eff_q[t - 1])) { sdm_destroy(ctx); return fail(nullptr, SDM_ERR_INVALID, "sdm_create: eff_q must ascend"); }
    if ((e = dalloc(&ctx->d_effR, o->n_eff_R)) || (e = dalloc(&ctx->d_effq, o->n_eff_q)) ||
        (e = dalloc(&ctx->d_efftab, (size_t)o->n_eff_R * o->n_eff_q)) ||
        (e = cudaMemcpy(ctx->d_effR, o->eff_R, sizeof(double) * o->n_eff_R, cudaMemcpyHostToDevice)) ||
        (e = cudaMemcpy(ctx->d_effq, o->eff_q, sizeof(double) * o->n_eff_q, cudaMemcpyHostToDevice)) ||
        (e = cudaMemcpy(ctx->d_efftab, o->eff_tab, sizeof(double) * (size_t)o->n_eff_R * o->n_eff_q, cudaMemcpyHostToDevice)))
      return bail(e, "efficiency table");
    kp.eff_R = ctx->d_effR; kp.eff_q = ctx->d_effq; kp.eff_tab = ctx->d_efftab;
  }
  ctx->o.eff_R = ctx->o.eff_q = ctx->o.eff_tab = nullptr;   // host pointers are not retained
  if (o->n_modes > 0) {
    if (!o->modes || !(o->sd_conc_mean > 0)) { sdm_destroy(ctx); return fail(nullptr, SDM_ERR_INVALID, "sdm_create: modes given without a modes array or sd_conc_mean"); }
    static_assert(sizeof(sdm_lognormal_mode) == sizeof(sdm_mode_view), "mode layout");
    const int rc = init_prepare(reinterpret_cast<const sdm_mode_view*>(o->modes), o->n_modes, o->sd_conc_mean, g.dV, ctx->ip);
    if (rc) { sdm_destroy(ctx); return fail(nullptr, SDM_ERR_INVALID, rc == -2 ? "sdm_create: the dry spectrum is too dilute for sd_conc_mean (no radius with multiplicity >= 1)" : "sdm_create: 1..8 modes with kappa, n_stp, r_mean > 0 and sigma_g > 1 required"); }
    const bool whole = o->x0 == 0 && o->x1 == 0 && o->y0 == 0 && o->y1 == 0 && o->z0 == 0 && o->z1 == 0;
    ctx->ip.x0 = whole ? 0.0 : o->x0; ctx->ip.x1 = whole ? g.X : o->x1;
    ctx->ip.y0 = whole ? 0.0 : o->y0; ctx->ip.y1 = whole ? g.Y : o->y1;
    ctx->ip.z0 = whole ? 0.0 : o->z0; ctx->ip.z1 = whole ? g.Z : o->z1;
    if ((g.hx && !(ctx->ip.x0 >= 0 && ctx->ip.x1 <= g.X && ctx->ip.x0 < ctx->ip.x1)) ||
        (g.hy && !(ctx->ip.y0 >= 0 && ctx->ip.y1 <= g.Y && ctx->ip.y0 < ctx->ip.y1)) ||
        (g.hz && !(ctx->ip.z0 >= 0 && ctx->ip.z1 <= g.Z && ctx->ip.z0 < ctx->ip.z1))) {
      sdm_destroy(ctx);
      return fail(nullptr, SDM_ERR_INVALID, "sdm_create: the Lagrangian domain x0..z1 must lie inside the grid");
    }
    ctx->ip.seed_lo = kp.seed_lo; ctx->ip.seed_hi = kp.seed_hi;
    ctx->have_modes = true;
  }
  ctx->o.modes = nullptr;
  if ((e = cudaEventCreateWithFlags(&ctx->ev_info, cudaEventDisableTiming)) ||
      (e = cudaEventCreateWithFlags(&ctx->ev_async, cudaEventDisableTiming)))
    return bail(e, "events");
  if ((e = cudaDeviceSynchronize())) return bail(e, "sync");
  *out = ctx;
  return SDM_OK;
}

void sdm_destroy(sdm_ctx* ctx) {
  if (!ctx) return;
  for (int b = 0; b < 2; ++b) {
    SdArrays& a = ctx->buf[b];
    cudaFree(a.n); cudaFree(a.rw2); cudaFree(a.rd3); cudaFree(a.kappa); cudaFree(a.x); cudaFree(a.y); cudaFree(a.z); cudaFree(a.id);
  }
  cudaFree(ctx->cell); cudaFree(ctx->off); cudaFree(ctx->rank); cudaFree(ctx->count); cudaFree(ctx->blocksum); cudaFree(ctx->seg);
  cudaFree(ctx->cf.mv);
  cudaFree(ctx->d_info); cudaFree(ctx->cf.rhod); cudaFree(ctx->cf.eta); cudaFree(ctx->cf.rho_a); cudaFree(ctx->outbuf);
  cudaFree(ctx->th_dense); cudaFree(ctx->rv_dense); cudaFree(ctx->cx); cudaFree(ctx->cy); cudaFree(ctx->cz);
  cudaFree(ctx->adv_tmp);
  cudaFree(ctx->flux_slots); cudaFree(ctx->flux_part); cudaFree(ctx->d_flux); cudaFree(ctx->cnt_mem);
  cudaFree(ctx->d_effR); cudaFree(ctx->d_effq); cudaFree(ctx->d_efftab);
  if (ctx->h_info) cudaFreeHost(ctx->h_info);
  if (ctx->h_rec) cudaFreeHost(ctx->h_rec);
  if (ctx->copy_stream) { cudaStreamDestroy(ctx->copy_stream); cudaEventDestroy(ctx->ev_copy_go); cudaEventDestroy(ctx->ev_h2d); cudaEventDestroy(ctx->ev_fields); }
  cudaFree(ctx->rec_dead); cudaFree(ctx->rec_cand); cudaFree(ctx->rec_hist); cudaFree(ctx->rec_info);
  if (ctx->ev_info) cudaEventDestroy(ctx->ev_info);
  if (ctx->ev_async) cudaEventDestroy(ctx->ev_async);
  for (int q = 0; q < SDM_N_STAGES; ++q) for (cudaEvent_t e : ctx->tev[q]) cudaEventDestroy(e);
  for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
  cudaGetLastError();
  delete ctx;
}

int sdm_init_range(const sdm_ctx* ctx, int g, double* lnr_lo, double* lnr_hi) {
  if (!ctx || !lnr_lo || !lnr_hi || !ctx->have_modes || g < 0 || g >= ctx->ip.n_spectra) return SDM_ERR_INVALID;
  *lnr_lo = ctx->ip.lnr_lo[g]; *lnr_hi = ctx->ip.lnr_hi[g];
  return SDM_OK;
}

int sdm_init(sdm_ctx* ctx, sdm_arrinfo th, sdm_arrinfo rv, sdm_arrinfo rhod, sdm_arrinfo c1, sdm_arrinfo c2, sdm_arrinfo c3,
             void* stream) {
  if (!ctx) return SDM_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  const Grid& g = ctx->g;
  if (!ctx->have_modes) return fail(ctx, SDM_ERR_INVALID, "sdm_init: the context was created without dry-aerosol modes");
  if (!th.data_zero || !rv.data_zero || !rhod.data_zero) return fail(ctx, SDM_ERR_INVALID, "sdm_init: th, rv and rhod are mandatory");
  const InitParams& ip = ctx->ip;
  double ncl = 1.0;
  if (g.hx) ncl *= (ip.x1 - ip.x0) / g.dx;
  if (g.hy) ncl *= (ip.y1 - ip.y0) / g.dy;
  if (g.hz) ncl *= (ip.z1 - ip.z0) / g.dz;
  const double Nd = std::floor(ctx->o.sd_conc_mean * ncl + 0.5);
  if (Nd > (double)ctx->cap_sd) return fail(ctx, SDM_ERR_CAPACITY, "sdm_init: sd_conc_mean x cells exceeds max_sd");
  const u64 N = (u64)Nd;
  launch_dense_copy(make_field(ctx, rhod), ctx->cf.rhod, g.NX, g.NY, g.NZ, st);
  ctx->launches++;
  ctx->mv_valid = false;
  const sdm_arrinfo comps[3] = {c1, c2, c3};
  if (int rc = copy_courants(ctx, comps, st)) return rc;
  ctx->cur = 0; ctx->cn = 0;
  // scratch per cell: RH to equilibrate with (outbuf) and the Kelvin length (eta, rewritten by every step_sync)
  if (ctx->o.real_bytes == 8) launch_init(view<double>(ctx->buf[0]), (u32)N, g, ip, make_field(ctx, th), make_field(ctx, rv), ctx->cf.rhod, ctx->outbuf, ctx->cf.eta, st);
  else launch_init(view<float>(ctx->buf[0]), (u32)N, g, ip, make_field(ctx, th), make_field(ctx, rv), ctx->cf.rhod, ctx->outbuf, ctx->cf.eta, st);
  ctx->launches += 1 + (N ? 1 : 0);
  CK(cudaGetLastError());
  const u32 info[8] = {(u32)N, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
  CK(cudaMemcpyAsync(ctx->d_info, info, sizeof(info), cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(ctx->count, 0, sizeof(u32) * g.ncell, st));
  CK(cudaMemsetAsync(ctx->cnt_mem, 0, sizeof(unsigned long long) * N_COUNTERS * NSLOT, st));
  CK(cudaMemsetAsync(ctx->flux_slots, 0, sizeof(double) * NSLOT, st));
  CK(cudaMemsetAsync(ctx->d_flux, 0, 4 * sizeof(double), st));
  CK(cudaMemsetAsync(ctx->outbuf, 0, sizeof(double) * g.ncell, st));
  CK(cudaStreamSynchronize(st));
  ctx->nslots = N; ctx->max_nc = 0; ctx->step = 0; ctx->synced = false; ctx->have_order = false; ctx->hist_valid = false;
  ctx->last_stream = st;
  return SDM_OK;
}

int sdm_init_from_arrays(sdm_ctx* ctx, sdm_arrinfo rhod, sdm_arrinfo c1, sdm_arrinfo c2, sdm_arrinfo c3, uint64_t N,
                         const uint64_t* n, const void* rw2, const void* rd3, const void* kappa, const void* x,
                         const void* y, const void* z, const uint32_t* id, void* stream) {
  if (!ctx) return SDM_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  const Grid& g = ctx->g;
  if (N > ctx->cap_sd) return fail(ctx, SDM_ERR_CAPACITY, "sdm_init_from_arrays: N exceeds max_sd");
  if (N && (!n || !rw2 || !rd3 || !kappa || !id || (g.hx && !x) || (g.hy && !y) || (g.hz && !z)))
    return fail(ctx, SDM_ERR_INVALID, "sdm_init_from_arrays: NULL attribute array");
  if (!rhod.data_zero) return fail(ctx, SDM_ERR_INVALID, "sdm_init_from_arrays: rhod is mandatory");
  launch_dense_copy(make_field(ctx, rhod), ctx->cf.rhod, g.NX, g.NY, g.NZ, st);
  ctx->launches++;
  ctx->mv_valid = false;
  const sdm_arrinfo comps[3] = {c1, c2, c3};
  if (int rc = copy_courants(ctx, comps, st)) return rc;
  ctx->cur = 0; ctx->cn = 0;
  SdArrays& a = ctx->buf[0];
  if (N) {
    CK(cudaMemcpyAsync(a.n, n, N * 8, cudaMemcpyDeviceToDevice, st));
    const size_t rb = (size_t)ctx->o.real_bytes;
    CK(cudaMemcpyAsync(a.rw2, rw2, N * rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(a.rd3, rd3, N * rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(a.kappa, kappa, N * rb, cudaMemcpyDeviceToDevice, st));
    if (g.hx) CK(cudaMemcpyAsync(a.x, x, N * rb, cudaMemcpyDeviceToDevice, st));
    if (g.hy) CK(cudaMemcpyAsync(a.y, y, N * rb, cudaMemcpyDeviceToDevice, st));
    if (g.hz) CK(cudaMemcpyAsync(a.z, z, N * rb, cudaMemcpyDeviceToDevice, st));
    CK(cudaMemcpyAsync(a.id, id, N * 4, cudaMemcpyDeviceToDevice, st));
  }
  const u32 info[8] = {(u32)N, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
  CK(cudaMemcpyAsync(ctx->d_info, info, sizeof(info), cudaMemcpyHostToDevice, st));
  CK(cudaMemsetAsync(ctx->count, 0, sizeof(u32) * g.ncell, st));
  CK(cudaMemsetAsync(ctx->cnt_mem, 0, sizeof(unsigned long long) * N_COUNTERS * NSLOT, st));
  CK(cudaMemsetAsync(ctx->flux_slots, 0, sizeof(double) * NSLOT, st));
  CK(cudaMemsetAsync(ctx->d_flux, 0, 4 * sizeof(double), st));
  CK(cudaStreamSynchronize(st));
  ctx->nslots = N; ctx->max_nc = 0; ctx->step = 0; ctx->synced = false; ctx->have_order = false; ctx->hist_valid = false;
  ctx->last_stream = st;
  return SDM_OK;
}

int sdm_step_sync(sdm_ctx* ctx, const sdm_opts* op, sdm_arrinfo th, sdm_arrinfo rv, sdm_arrinfo c1, sdm_arrinfo c2,
                  sdm_arrinfo c3, sdm_arrinfo rhod, void* stream) {
  if (!ctx || !op) return SDM_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  const Grid& g = ctx->g;
  if (!th.data_zero || !rv.data_zero) return fail(ctx, SDM_ERR_INVALID, "sdm_step_sync: th and rv are mandatory");
  if (op->cond && (op->sstp_cond < 1 || !(op->RH_max > 0))) return fail(ctx, SDM_ERR_INVALID, "sdm_step_sync: sstp_cond >= 1 and RH_max > 0 required");
  if (op->cond && op->cond_adapt_tol > 0.0 && ctx->cond_arith == 4)
    return fail(ctx, SDM_ERR_INVALID, "sdm_step_sync: cond_adapt_tol needs the fp64-arithmetic condensation (sdm_set_cond_arith 8)");
  if (ctx->synced) return fail(ctx, SDM_ERR_ORDER, "sdm_step_sync: called twice without step_async");
  ctx->last_stream = st;
  if (rhod.data_zero) { launch_dense_copy(make_field(ctx, rhod), ctx->cf.rhod, g.NX, g.NY, g.NZ, st); ctx->launches++; ctx->mv_valid = false; }
  const sdm_arrinfo comps[3] = {c1, c2, c3};
  if (int rc = copy_courants(ctx, comps, st)) return rc;

  // recycling of zero-multiplicity SDs, before they are compacted away (PAPER.md :641 "at the begining of each timestep")
  if (ctx->recycle && ctx->nslots) {
    t_begin(ctx, SDM_STAGE_RECYCLE, st);
    const SdArrays& b = ctx->buf[ctx->cur];
    launch_recycle_scan(b.n, b.id, (u32)ctx->nslots, ctx->rec_dead, ctx->rec_info, ctx->rec_hist, st);
    ctx->launches += 2;
    CK(cudaMemcpyAsync(ctx->h_rec, ctx->rec_info, 4 * sizeof(u32), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    ctx->host_syncs++;
    const u32 n_dead = ctx->h_rec[0], k = ctx->h_rec[1];
    if (k) {
      if (ctx->o.real_bytes == 8)
        ctx->launches += launch_recycle_apply(view<double>(b), g, (u32)ctx->nslots, n_dead, k, ctx->rec_dead, ctx->rec_cand, ctx->rec_info, ctx->h_rec + 4, st);
      else
        ctx->launches += launch_recycle_apply(view<float>(b), g, (u32)ctx->nslots, n_dead, k, ctx->rec_dead, ctx->rec_cand, ctx->rec_info, ctx->h_rec + 4, st);
      ctx->recycled += k;
    }
    CK(cudaGetLastError());
    t_end(ctx, SDM_STAGE_RECYCLE, st);
  }

  // a0-a3: compaction + cell index + counting sort by cell
  u32* d_cur = ctx->d_info + ctx->cn;
  u32* d_next = ctx->d_info + (ctx->cn ^ 1);
  CK(cudaMemsetAsync(ctx->d_info + 2, 0, sizeof(u32), st));
  CK(cudaMemsetAsync(ctx->d_info + 4, 0, 4 * sizeof(u32), st));
  // condensation tiles: about kCondTileTarget SDs per CTA at the occupancy seen before this step
  const bool arith32 = ctx->cond_arith == 4 && ctx->o.real_bytes == 4;
  const double tile_target = arith32 ? kCond32TileTarget : kCondTileTarget;
  const double mean_nc = (double)ctx->nslots / g.ncell;
  ctx->cond_cpb0 = (int)std::min<double>(kCondMaxCpb, std::max(1.0, tile_target / std::max(mean_nc, 1e-9)));
  {  // A population of a few waves of resident CTAs (5 per SM, 8 for the fp32 sweep) is bound by the latency of one tile
     // (10 substeps, each a sweep + a barrier + the cells' chain), not by throughput: the tiles of a launch then run in
     // k = 1, 2, 3 FULL waves (a launch of 1.1 waves takes as long as one of 2), with the smallest k whose tiles fit the
     // kernel's slots at mean + 5 sigma occupancy (configs[1], 180 000 SDs: 704 tiles of 8 cells on 740 slots;
     // configs[2], 720 000 SDs: 1407 tiles of 4 cells = two waves).  Beyond ~4 waves the fixed costs of smaller tiles lose
     // more than the balance gains.
    const double wave = (double)ctx->n_sm * (arith32 ? 8 : 5);
    const double cap = arith32 ? SDM_COND32_TILE_SLOTS : SDM_COND_TILE_SLOTS;
    if ((double)ctx->nslots / tile_target < 4.0 * wave && mean_nc > 0.0) {
      for (int k = 1; k <= 4; ++k) {
        const int cpb = (int)std::ceil((double)g.ncell / (k * wave));
        const double expect = cpb * mean_nc;
        if (cpb <= (int)kCondMaxCpb && expect + 5.0 * std::sqrt(expect) + 1.0 <= cap) { ctx->cond_cpb0 = std::max(cpb, 1); break; }
      }
    }
  }
  // sparse cells: the smallest candidate tile (a quarter of cond_cpb0) must fit the cell records of the small kernel, or the
  // launch would fall back to one cell per CTA
  ctx->cond_cpb0 = std::max(1, std::min(ctx->cond_cpb0, 4 * cond_max_cells(arith32)));
  // a0-a1: the last step_async left cell, off and the histogram behind (k_coal_move_tile), unless recycling moved SDs since
  const bool have_hist = ctx->hist_valid && !(ctx->recycle && ctx->nslots);
  if (ctx->hist_valid && !have_hist) CK(cudaMemsetAsync(ctx->count, 0, sizeof(u32) * g.ncell, st));
  ctx->hist_valid = false;
  if (!have_hist) {
    t_begin(ctx, SDM_STAGE_HIST, st);
    if (ctx->o.real_bytes == 8) launch_cellhist(view<double>(ctx->buf[ctx->cur]), d_cur, (u32)ctx->nslots, g, ctx->cell, ctx->off, ctx->count, st);
    else launch_cellhist(view<float>(ctx->buf[ctx->cur]), d_cur, (u32)ctx->nslots, g, ctx->cell, ctx->off, ctx->count, st);
    t_end(ctx, SDM_STAGE_HIST, st);
    ctx->launches += ctx->nslots ? 1 : 0;
  }
  t_begin(ctx, SDM_STAGE_SCAN, st);
  launch_scan(ctx->count, g.ncell, ctx->blocksum, ctx->seg, d_next, ctx->d_info + 2, st);
  t_end(ctx, SDM_STAGE_SCAN, st);
  launch_tile_max(ctx->seg, g.ncell, ctx->cond_cpb0, ctx->d_info + 4, st);
  ctx->launches++;
  ctx->launches += 3;
  CK(cudaMemcpyAsync(ctx->h_info, ctx->d_info, 8 * sizeof(u32), cudaMemcpyDeviceToHost, st));
  CK(cudaEventRecord(ctx->ev_info, st));
  t_begin(ctx, SDM_STAGE_SCATTER, st);
  if (ctx->o.real_bytes == 8) launch_scatter(view<double>(ctx->buf[ctx->cur]), view<double>(ctx->buf[ctx->cur ^ 1]), d_cur, (u32)ctx->nslots, g, ctx->cell, ctx->off, ctx->seg, st);
  else launch_scatter(view<float>(ctx->buf[ctx->cur]), view<float>(ctx->buf[ctx->cur ^ 1]), d_cur, (u32)ctx->nslots, g, ctx->cell, ctx->off, ctx->seg, st);
  t_end(ctx, SDM_STAGE_SCATTER, st);
  ctx->launches += ctx->nslots ? scatter_parts((u32)ctx->nslots) : 0;   // one launch, or two halves (sdm_sort.cu)
  CK(cudaGetLastError());
  CK(cudaEventSynchronize(ctx->ev_info));   // the scatter runs while the host sizes the next launches
  ctx->host_syncs++;
  ctx->cn ^= 1;
  ctx->cur ^= 1;
  ctx->nslots = ctx->h_info[ctx->cn];
  ctx->max_nc = ctx->h_info[2];
  for (int k = 0; k < 4; ++k) ctx->tile_max[k] = ctx->h_info[4 + k];
  if (ctx->h_info[3]) {   // raised by a rank kernel of the step before (reported here at the latest; cleared once reported)
    cudaMemsetAsync(ctx->d_info + 3, 0, sizeof(u32), st);
    return fail(ctx, SDM_ERR_CUDA, "sdm_step_sync: device-side error flag set (corrupted segment sizes)");
  }

  // launch sizing from the measured occupancy
  const double mean = (double)ctx->nslots / g.ncell;
  int G = pick_group(ctx, mean);
  const int P = std::max(next_pow2((int)ctx->max_nc), 2);
  if ((size_t)ng_of(G) * P * 10 > kSmemLimit) G = 256;
  if ((size_t)ng_of(G) * P * 10 > kSmemLimit || ctx->max_nc > 32768)
    return fail(ctx, SDM_ERR_CAPACITY, "sdm_step_sync: a cell holds more super-droplets than one CTA can sort (limit 16384)");
  ctx->G = G;
  const Field thf = make_field(ctx, th), rvf = make_field(ctx, rv);
  if (ctx->nslots) {
    t_begin(ctx, SDM_STAGE_RANK, st);
    CK(launch_rank(G, ctx->buf[ctx->cur].id, ctx->seg, g.ncell, (u32)ctx->step, ctx->kp.seed_lo, ctx->kp.seed_hi, P,
                   ctx->rank, (int*)(ctx->d_info + 3), st));
    t_end(ctx, SDM_STAGE_RANK, st);
    ctx->launches++;
  }
  ctx->have_order = true;
  if (ctx->wait_h2d) {   // sdm_step_host: th, rv arrive on the copy stream while the sort runs
    CK(cudaStreamWaitEvent(st, ctx->ev_h2d, 0));
    ctx->wait_h2d = false;
  }
  if (op->cond) {
    // the most preferred tile kernel (small, medium, large) any candidate tile size fits, with the largest such
    // tile; else one cell per CTA in place in global memory
    int cpb = 1, variant = arith32 ? cond_variant_f32(1, (int)ctx->max_nc) : cond_variant(1, (int)ctx->max_nc);
    for (int k = 3; k >= 0; --k) {
      const int cand = cond_tile_candidate(ctx->cond_cpb0, k);
      const int v = arith32 ? cond_variant_f32(cand, (int)ctx->tile_max[k]) : cond_variant(cand, (int)ctx->tile_max[k]);
      if (v && (variant == 0 || v <= variant)) { cpb = cand; variant = v; }
    }
    CondParams cp{g.dt / op->sstp_cond, op->sstp_cond, op->RH_max, ctx->kfast, op->cond_adapt_tol > 0.0 ? op->cond_adapt_tol : 0.0};
    ctx->last_cond_cpb = cpb;
    ctx->last_cond_variant = (ctx->o.real_bytes == 4 && arith32 && variant != 0 && op->sstp_cond <= 500) ? 100 + variant : variant;
    t_begin(ctx, SDM_STAGE_COND, st);
    if (ctx->o.real_bytes == 8)
      CK(launch_cond(cpb, variant, view<double>(ctx->buf[ctx->cur]), view<double>(ctx->buf[ctx->cur ^ 1]), ctx->rank, ctx->seg, g, thf,
                     rvf, ctx->cf, cp, ctx->cnt, st));
    else if (arith32 && variant != 0 && op->sstp_cond <= 500)   // (its packed per-lane counters hold 500 substeps)
      CK(launch_cond_f32(cpb, variant, view<float>(ctx->buf[ctx->cur]), ctx->rank, ctx->seg, g, thf, rvf, ctx->cf, cp, ctx->cnt, st));
    else
      CK(launch_cond(cpb, variant, view<float>(ctx->buf[ctx->cur]), view<float>(ctx->buf[ctx->cur ^ 1]), ctx->rank, ctx->seg, g, thf,
                     rvf, ctx->cf, cp, ctx->cnt, st));
    t_end(ctx, SDM_STAGE_COND, st);
  } else {
    launch_thermo(g, thf, rvf, ctx->cf, st);
    CK(cudaGetLastError());
  }
  ctx->launches++;
  ctx->synced = true;
  return SDM_OK;
}

int sdm_step_async(sdm_ctx* ctx, const sdm_opts* op, void* stream) {
  if (!ctx || !op) return SDM_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  const Grid& g = ctx->g;
  if (!ctx->synced) return fail(ctx, SDM_ERR_ORDER, "sdm_step_async: step_sync of this step has not been called");
  if (op->coal && op->sstp_coal < 1) return fail(ctx, SDM_ERR_INVALID, "sdm_step_async: sstp_coal >= 1 required");
  ctx->last_stream = st;
  if (ctx->nslots && (op->coal || op->adve || op->sedi)) {
    const int G = ctx->G;
    int cap = (int)((ctx->max_nc + 3) / 4 * 4);
    cap = std::max(cap, 4);
    const int sstp = op->coal ? op->sstp_coal : 1;
    const int adapt_max = (op->coal && op->coal_adapt_max > 1) ? op->coal_adapt_max : 0;
    const int multi = (sstp > 1 || adapt_max) ? 2 : 1;   // several groupings per step: the per-cell kernel with its sort buffers
    bool in_smem = coal_smem_bytes(G, cap, multi, true) <= kSmemLimit;
    if (!in_smem && coal_smem_bytes(G, cap, multi, false) > kSmemLimit)
      return fail(ctx, SDM_ERR_CAPACITY, "sdm_step_async: a cell holds more super-droplets than one CTA can pair");
    // (a slab hands SDs over after the step, recycling moves them before the next: the histogram is then built by k_cellhist)
    CoalMoveParams mp{op->coal, op->adve, op->sedi, sstp, (u32)ctx->step, (ctx->recycle || g.open_x) ? 0 : 1, adapt_max};
    int tile_cpb = 0, tile_need = 0;   // tile-resident kernel: largest candidate tile that fits (one set of pairs per step only)
    for (int k = 0; k < 4 && !tile_cpb && multi == 1 && !ctx->group_override; ++k) {
      const int cand = cond_tile_candidate(ctx->cond_cpb0, k);
      if (coal_tile_fits(cand, (int)ctx->tile_max[k], ctx->o.real_bytes)) { tile_cpb = cand; tile_need = (int)ctx->tile_max[k]; }
    }
    ctx->last_coal_cpb = tile_cpb;
    t_begin(ctx, SDM_STAGE_COAL_MOVE, st);
    const bool f64 = ctx->o.real_bytes == 8;
    ctx->n_flux_part = tile_cpb ? (g.ncell + tile_cpb - 1) / tile_cpb : 0;
    ctx->hist_valid = tile_cpb && mp.fold;
    if (tile_cpb && op->adve && !ctx->mv_valid) {   // eq. 16 per cell: once per set of Courant fields, not once per step
      launch_cell_move_consts(g, ctx->cf, st);
      ctx->mv_valid = true;
      ctx->launches++;
    }
    if (tile_cpb && f64)
      CK(launch_coal_move_tile(tile_cpb, tile_need, view<double>(ctx->buf[ctx->cur]), ctx->rank, ctx->seg, g, ctx->cf, ctx->kp, mp,
                               ctx->flux_part, ctx->cnt, ctx->cell, ctx->off, ctx->count, st));
    else if (tile_cpb)
      CK(launch_coal_move_tile(tile_cpb, tile_need, view<float>(ctx->buf[ctx->cur]), ctx->rank, ctx->seg, g, ctx->cf, ctx->kp, mp,
                               ctx->flux_part, ctx->cnt, ctx->cell, ctx->off, ctx->count, st));
    else if (f64)
      CK(launch_coal_move(G, cap, in_smem, view<double>(ctx->buf[ctx->cur]), ctx->rank, ctx->seg, g, ctx->cf, ctx->kp, mp,
                          ctx->flux_slots, ctx->cnt, st));
    else
      CK(launch_coal_move(G, cap, in_smem, view<float>(ctx->buf[ctx->cur]), ctx->rank, ctx->seg, g, ctx->cf, ctx->kp, mp,
                          ctx->flux_slots, ctx->cnt, st));
    t_end(ctx, SDM_STAGE_COAL_MOVE, st);
    ctx->launches++;
  }
  else ctx->n_flux_part = 0;
  launch_flux_sum(ctx->flux_slots, ctx->flux_part, ctx->n_flux_part, ctx->d_flux, ctx->d_flux + 1, ctx->d_info + 3, st);
  ctx->launches++;
  CK(cudaGetLastError());
  CK(cudaEventRecord(ctx->ev_async, st));
  ctx->step += 1;
  ctx->synced = false;
  ctx->have_order = false;
  return SDM_OK;
}

int sdm_step_async_result(sdm_ctx* ctx, double* rain_flux) {
  if (!ctx) return SDM_ERR_INVALID;
  CK(cudaEventSynchronize(ctx->ev_async));
  return check_device_flag(ctx, "sdm_step_async_result", rain_flux);
}

int sdm_step_host(sdm_ctx* ctx, const sdm_opts* op, double* th_host, double* rv_host, double* rain_flux, void* stream) {
  if (!ctx || !op || !th_host || !rv_host) return SDM_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  const Grid& g = ctx->g;
  const size_t bytes = sizeof(double) * g.ncell;
  if (!ctx->copy_stream) {
    CK(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    CK(cudaEventCreateWithFlags(&ctx->ev_copy_go, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&ctx->ev_h2d, cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&ctx->ev_fields, cudaEventDisableTiming));
  }
  cudaStream_t cs = ctx->copy_stream;
  // in: after whatever the caller's stream still does with the dense copies; the condensation kernel waits for ev_h2d
  CK(cudaEventRecord(ctx->ev_copy_go, st));
  CK(cudaStreamWaitEvent(cs, ctx->ev_copy_go, 0));
  CK(cudaMemcpyAsync(ctx->th_dense, th_host, bytes, cudaMemcpyHostToDevice, cs));
  CK(cudaMemcpyAsync(ctx->rv_dense, rv_host, bytes, cudaMemcpyHostToDevice, cs));
  CK(cudaEventRecord(ctx->ev_h2d, cs));
  ctx->wait_h2d = true;
  sdm_arrinfo th{ctx->th_dense, {0, 0, 0}}, rv{ctx->rv_dense, {0, 0, 0}}, none{nullptr, {0, 0, 0}};
  int idx = 0;   // dense C-order strides over the present dimensions
  const long long sx = (long long)g.NY * g.NZ, sy = g.NZ, sz = 1;
  if (g.hx) { th.strides[idx] = rv.strides[idx] = sx; ++idx; }
  if (g.hy) { th.strides[idx] = rv.strides[idx] = sy; ++idx; }
  if (g.hz) { th.strides[idx] = rv.strides[idx] = sz; ++idx; }
  if (int rc = sdm_step_sync(ctx, op, th, rv, none, none, none, none, stream)) { ctx->wait_h2d = false; return rc; }
  // out: th, rv are final once the work of step_sync is done (:816); they leave while coalescence and movement run
  CK(cudaEventRecord(ctx->ev_fields, st));
  CK(cudaStreamWaitEvent(cs, ctx->ev_fields, 0));
  CK(cudaMemcpyAsync(th_host, ctx->th_dense, bytes, cudaMemcpyDeviceToHost, cs));
  CK(cudaMemcpyAsync(rv_host, ctx->rv_dense, bytes, cudaMemcpyDeviceToHost, cs));
  if (int rc = sdm_step_async(ctx, op, stream)) return rc;
  CK(cudaStreamSynchronize(st));
  CK(cudaStreamSynchronize(cs));
  return check_device_flag(ctx, "sdm_step_host", rain_flux);
}

static int diag_launch(sdm_ctx* ctx, int wet, double lo, double hi, int k, int count_only, void* stream) {
  cudaStream_t st = (cudaStream_t)stream;
  ctx->last_stream = st;
  if (ctx->o.real_bytes == 8)
    launch_diag_mom(view<double>(ctx->buf[ctx->cur]), ctx->d_info + ctx->cn, (u32)ctx->nslots, ctx->g, wet, lo, hi, k, count_only,
                    ctx->cf.rhod, ctx->outbuf, st);
  else
    launch_diag_mom(view<float>(ctx->buf[ctx->cur]), ctx->d_info + ctx->cn, (u32)ctx->nslots, ctx->g, wet, lo, hi, k, count_only,
                    ctx->cf.rhod, ctx->outbuf, st);
  ctx->launches += (ctx->nslots ? 1 : 0) + (count_only ? 0 : 1);
  CK(cudaGetLastError());
  return SDM_OK;
}
int sdm_diag_sd_conc(sdm_ctx* ctx, void* stream) { return ctx ? diag_launch(ctx, 1, 0, 0, 0, 1, stream) : SDM_ERR_INVALID; }
int sdm_diag_dry_rng(sdm_ctx* ctx, double r_mi, double r_mx) {
  if (!ctx) return SDM_ERR_INVALID;
  ctx->dry_lo = r_mi; ctx->dry_hi = r_mx;
  return SDM_OK;
}
int sdm_diag_wet_rng(sdm_ctx* ctx, double r_mi, double r_mx) {
  if (!ctx) return SDM_ERR_INVALID;
  ctx->wet_lo = r_mi; ctx->wet_hi = r_mx;
  return SDM_OK;
}
int sdm_diag_dry_mom(sdm_ctx* ctx, int k, void* stream) { return ctx ? diag_launch(ctx, 0, ctx->dry_lo, ctx->dry_hi, k, 0, stream) : SDM_ERR_INVALID; }
int sdm_diag_wet_mom(sdm_ctx* ctx, int k, void* stream) { return ctx ? diag_launch(ctx, 1, ctx->wet_lo, ctx->wet_hi, k, 0, stream) : SDM_ERR_INVALID; }
const double* sdm_outbuf(sdm_ctx* ctx) { return ctx ? ctx->outbuf : nullptr; }

int sdm_n_sd(sdm_ctx* ctx, uint64_t* n_sd) {
  if (!ctx || !n_sd) return SDM_ERR_INVALID;
  *n_sd = ctx->nslots;
  return SDM_OK;
}

}  // extern "C"

namespace {
template <typename R>
SdArraysT<R> buffers_view(const sdm_sd_buffers& b) {
  return SdArraysT<R>{b.n, (R*)b.rw2, (R*)b.rd3, (R*)b.kappa, (R*)b.x, (R*)b.y, (R*)b.z, b.id};
}
bool buffers_ok(const sdm_ctx* c, const sdm_sd_buffers* b) {
  return b && b->n && b->rw2 && b->rd3 && b->kappa && b->x && b->id && (!c->g.hy || b->y) && (!c->g.hz || b->z);
}
}  // namespace

extern "C" {

int sdm_pack_leavers(sdm_ctx* ctx, uint64_t cap, const sdm_sd_buffers* left, const sdm_sd_buffers* right, uint64_t* n_left,
                     uint64_t* n_right, void* stream) {
  if (!ctx || !n_left || !n_right) return SDM_ERR_INVALID;
  if (!ctx->g.open_x) return fail(ctx, SDM_ERR_ORDER, "sdm_pack_leavers: the context was not created with open_x = 1");
  if (ctx->synced) return fail(ctx, SDM_ERR_ORDER, "sdm_pack_leavers: call it after step_async of the step");
  if (!buffers_ok(ctx, left) || !buffers_ok(ctx, right)) return fail(ctx, SDM_ERR_INVALID, "sdm_pack_leavers: NULL buffer array");
  cudaStream_t st = (cudaStream_t)stream;
  ctx->last_stream = st;
  CK(cudaStreamWaitEvent(st, ctx->ev_async, 0));
  u32* cnt2 = ctx->d_info + 6;   // two of the tile-maximum words: free between step_async and the next step_sync
  const bool f64 = ctx->o.real_bytes == 8;
  if (f64) launch_count_leavers(view<double>(ctx->buf[ctx->cur]), (u32)ctx->nslots, ctx->g, cnt2, st);
  else launch_count_leavers(view<float>(ctx->buf[ctx->cur]), (u32)ctx->nslots, ctx->g, cnt2, st);
  u32 h[2] = {0, 0};
  CK(cudaMemcpyAsync(h, cnt2, sizeof(h), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  ctx->launches += ctx->nslots ? 1 : 0;
  *n_left = h[0]; *n_right = h[1];
  if (h[0] > cap || h[1] > cap) return fail(ctx, SDM_ERR_CAPACITY, "sdm_pack_leavers: more leavers than the buffers hold");
  if (h[0] + h[1] == 0) return SDM_OK;
  if (f64) launch_pack_leavers(view<double>(ctx->buf[ctx->cur]), (u32)ctx->nslots, ctx->g, buffers_view<double>(*left), buffers_view<double>(*right), cnt2, st);
  else launch_pack_leavers(view<float>(ctx->buf[ctx->cur]), (u32)ctx->nslots, ctx->g, buffers_view<float>(*left), buffers_view<float>(*right), cnt2, st);
  ctx->launches++;
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(st));
  ctx->hist_valid = false;
  return SDM_OK;
}

int sdm_unpack_arrivals(sdm_ctx* ctx, uint64_t N, const sdm_sd_buffers* in, double x_shift, void* stream) {
  if (!ctx) return SDM_ERR_INVALID;
  if (!ctx->g.open_x) return fail(ctx, SDM_ERR_ORDER, "sdm_unpack_arrivals: the context was not created with open_x = 1");
  if (ctx->synced) return fail(ctx, SDM_ERR_ORDER, "sdm_unpack_arrivals: call it between step_async and the next step_sync");
  if (N == 0) return SDM_OK;
  if (!buffers_ok(ctx, in)) return fail(ctx, SDM_ERR_INVALID, "sdm_unpack_arrivals: NULL buffer array");
  if (ctx->nslots + N > ctx->cap_sd) return fail(ctx, SDM_ERR_CAPACITY, "sdm_unpack_arrivals: arrivals exceed max_sd");
  cudaStream_t st = (cudaStream_t)stream;
  ctx->last_stream = st;
  CK(cudaStreamWaitEvent(st, ctx->ev_async, 0));
  if (ctx->o.real_bytes == 8) launch_unpack_arrivals(view<double>(ctx->buf[ctx->cur]), (u32)ctx->nslots, (u32)N, ctx->g, buffers_view<double>(*in), x_shift, st);
  else launch_unpack_arrivals(view<float>(ctx->buf[ctx->cur]), (u32)ctx->nslots, (u32)N, ctx->g, buffers_view<float>(*in), x_shift, st);
  ctx->launches++;
  ctx->nslots += N;
  const u32 ns = (u32)ctx->nslots;
  CK(cudaMemcpyAsync(ctx->d_info + ctx->cn, &ns, sizeof(u32), cudaMemcpyHostToDevice, st));
  CK(cudaStreamSynchronize(st));   // &ns is a stack word
  CK(cudaGetLastError());
  ctx->hist_valid = false;
  return SDM_OK;
}

int sdm_upstream_advect(sdm_ctx* ctx, sdm_arrinfo psi, void* stream) {
  if (!ctx) return SDM_ERR_INVALID;
  if (!psi.data_zero) return fail(ctx, SDM_ERR_INVALID, "sdm_upstream_advect: psi is mandatory");
  if (!ctx->adv_tmp) CK(dalloc(&ctx->adv_tmp, (size_t)ctx->g.ncell));
  launch_upstream(make_field(ctx, psi), ctx->g, ctx->cf, ctx->adv_tmp, (cudaStream_t)stream);
  ctx->launches += 2;
  CK(cudaGetLastError());
  return SDM_OK;
}

int sdm_n_live(sdm_ctx* ctx, uint64_t* n_live) { return sdm_n_sd(ctx, n_live); }

int sdm_export_state(sdm_ctx* ctx, uint64_t* n, void* rw2, void* rd3, void* kappa, void* x, void* y, void* z,
                     uint32_t* id, void* stream) {
  if (!ctx) return SDM_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  const SdArrays& a = ctx->buf[ctx->cur];
  const size_t N = ctx->nslots;
  if (!N) return SDM_OK;
  if (n) CK(cudaMemcpyAsync(n, a.n, N * 8, cudaMemcpyDeviceToDevice, st));
  const size_t rb = (size_t)ctx->o.real_bytes;
  if (rw2) CK(cudaMemcpyAsync(rw2, a.rw2, N * rb, cudaMemcpyDeviceToDevice, st));
  if (rd3) CK(cudaMemcpyAsync(rd3, a.rd3, N * rb, cudaMemcpyDeviceToDevice, st));
  if (kappa) CK(cudaMemcpyAsync(kappa, a.kappa, N * rb, cudaMemcpyDeviceToDevice, st));
  if (x && ctx->g.hx) CK(cudaMemcpyAsync(x, a.x, N * rb, cudaMemcpyDeviceToDevice, st));
  if (y && ctx->g.hy) CK(cudaMemcpyAsync(y, a.y, N * rb, cudaMemcpyDeviceToDevice, st));
  if (z && ctx->g.hz) CK(cudaMemcpyAsync(z, a.z, N * rb, cudaMemcpyDeviceToDevice, st));
  if (id) CK(cudaMemcpyAsync(id, a.id, N * 4, cudaMemcpyDeviceToDevice, st));
  return SDM_OK;
}

int sdm_export_order(sdm_ctx* ctx, uint32_t* ids_sorted, uint32_t* seg_start, void* stream) {
  if (!ctx || !ids_sorted || !seg_start) return SDM_ERR_INVALID;
  if (!ctx->have_order) return fail(ctx, SDM_ERR_ORDER, "sdm_export_order: valid only between step_sync and step_async");
  cudaStream_t st = (cudaStream_t)stream;
  if (ctx->nslots) { launch_export_order(ctx->buf[ctx->cur].id, ctx->rank, ctx->seg, ctx->g.ncell, ids_sorted, st); ctx->launches++; }
  CK(cudaMemcpyAsync(seg_start, ctx->seg, sizeof(u32) * ((size_t)ctx->g.ncell + 1), cudaMemcpyDeviceToDevice, st));
  CK(cudaGetLastError());
  return SDM_OK;
}

int sdm_stats(sdm_ctx* ctx, sdm_stats_t* out) {
  if (!ctx || !out) return SDM_ERR_INVALID;
  CK(cudaStreamSynchronize(ctx->last_stream));
  std::vector<unsigned long long> h(N_COUNTERS * NSLOT);
  CK(cudaMemcpy(h.data(), ctx->cnt_mem, sizeof(unsigned long long) * N_COUNTERS * NSLOT, cudaMemcpyDeviceToHost));
  unsigned long long s[N_COUNTERS] = {0, 0, 0, 0, 0, 0, 0};
  for (int q = 0; q < N_COUNTERS; ++q) for (int t = 0; t < NSLOT; ++t) s[q] += h[(size_t)q * NSLOT + t];
  out->n_sd = ctx->nslots; out->max_cell_count = ctx->max_nc; out->step = ctx->step; out->kernel_launches = ctx->launches;
  out->pairs = s[0]; out->collisions = s[1]; out->near_ties = s[2]; out->ill_posed = s[3]; out->newton_iters = s[4];
  out->sd_substeps = s[5]; out->cond_slow = s[6];
  out->recycled = ctx->recycled;
  out->cond_variant = (u64)ctx->last_cond_variant; out->cond_tile_cells = (u64)ctx->last_cond_cpb;
  out->coal_tile_cells = (u64)ctx->last_coal_cpb; out->host_syncs = ctx->host_syncs;
  return SDM_OK;
}

int sdm_set_step(sdm_ctx* ctx, uint64_t step) {
  if (!ctx) return SDM_ERR_INVALID;
  if (ctx->synced) return fail(ctx, SDM_ERR_ORDER, "sdm_set_step: not between step_sync and step_async");
  ctx->step = step;
  return SDM_OK;
}

int sdm_set_timing(sdm_ctx* ctx, int enable) {
  if (!ctx) return SDM_ERR_INVALID;
  ctx->timing = enable != 0;
  return SDM_OK;
}

int sdm_stage_times(sdm_ctx* ctx, double* ms, uint64_t* launches, int reset) {
  if (!ctx || !ms) return SDM_ERR_INVALID;
  CK(cudaStreamSynchronize(ctx->last_stream));
  t_fold(ctx);
  for (int q = 0; q < SDM_N_STAGES; ++q) {
    ms[q] = ctx->t_ms[q];
    if (launches) launches[q] = ctx->t_cnt[q];
    if (reset) { ctx->t_ms[q] = 0; ctx->t_cnt[q] = 0; }
  }
  return SDM_OK;
}

int sdm_set_recycle(sdm_ctx* ctx, int on) {
  if (!ctx) return SDM_ERR_INVALID;
  if (on && !ctx->rec_dead) {
    const size_t cap = recycle_items_capacity(ctx->cap_sd);
    CK(dalloc(&ctx->rec_dead, cap));
    CK(dalloc(&ctx->rec_cand, cap));
    CK(dalloc(&ctx->rec_hist, 2048));
    CK(dalloc(&ctx->rec_info, 8));
    CK(cudaMallocHost((void**)&ctx->h_rec, 8 * sizeof(u32)));
  }
  ctx->recycle = on != 0;
  return SDM_OK;
}

int sdm_set_cond_arith(sdm_ctx* ctx, int bytes) {
  if (!ctx) return SDM_ERR_INVALID;
  if (bytes != 8 && bytes != 4) return fail(ctx, SDM_ERR_INVALID, "sdm_set_cond_arith: 8 or 4");
  if (bytes == 4 && ctx->o.real_bytes != 4) return fail(ctx, SDM_ERR_INVALID, "sdm_set_cond_arith: fp32 arithmetic needs real_bytes = 4");
  ctx->cond_arith = bytes;
  return SDM_OK;
}

int sdm_set_cond_kfast(sdm_ctx* ctx, int kfast) {
  if (!ctx) return SDM_ERR_INVALID;
  if (kfast < 1 || kfast > 200) return fail(ctx, SDM_ERR_INVALID, "sdm_set_cond_kfast: 1..200");
  ctx->kfast = kfast;
  return SDM_OK;
}

int sdm_set_group_size(sdm_ctx* ctx, int group) {
  if (!ctx) return SDM_ERR_INVALID;
  if (!(group == 0 || group == 4 || group == 8 || group == 16 || group == 32 || group == 256))
    return fail(ctx, SDM_ERR_INVALID, "sdm_set_group_size: 0, 4, 8, 16, 32 or 256");
  ctx->group_override = group;
  return SDM_OK;
}

}  // extern "C"
