// Host-side launch interface between sdm_api.cu and the kernel translation units.
#pragma once
#include "sdm_common.cuh"

namespace sdm {

// CTA shape of the cell-resident kernels: sub-warp / warp groups share a 128-thread CTA, a CTA-wide
// group is the CTA.
template <int G>
struct CtaOf { static constexpr int threads = (G <= 32) ? 128 : G; };

struct CondParams {
  double dtp;        // dt / sstp_cond
  int sstp;
  double RH_max;
  int kfast;         // growth-rate evaluations per SD in the dense sweep before an SD is deferred to the second pass
  double adapt_tol;  // > 0: per-cell substep counts (DESIGN.md R-adapt); fp64-arithmetic kernels only
};
struct CoalMoveParams {
  int coal, adve, sedi, sstp_coal;
  u32 step;
  int fold;          // k_coal_move_tile also writes next step's cell index, offset and histogram (a0-a1 folded into a6)
  int coal_adapt_max;   // > 1: per-cell coalescence substeps from P_ij (DESIGN.md R-adapt-coal); per-cell kernel only
  double inv_dx, inv_dy, inv_dz;   // 1/dx .. (IEEE), filled in by launch_coal_move_tile
};
struct CellFields {  // library-owned dense per-cell arrays
  double* rhod;      // copy of the caller's rhod
  double* eta;       // viscosity after the condensation feedback (for v_term)
  double* rho_a;     // air density rhod (1 + rv)
  const double *cx, *cy, *cz;   // rho_d * Courant on the Arakawa-C grid, dense C order
  double* mv;        // eq. 16 per cell, 6 doubles: ax, bx, ay, by, az, bz (k_cell_move_consts; rebuilt when rhod or a Courant field changes)
};

// sdm_sort.cu
template <typename R>
void launch_cellhist(const SdArraysT<R>& a, const u32* d_nslots, u32 nslots_bound, const Grid& g, u32* cell, u32* off,
                     u32* count, cudaStream_t st);
int scan_num_blocks(int ncell);
int scatter_parts(u32 nslots_bound);   // launches of the reorder (1 or 2)
void launch_scan(u32* count, int ncell, u32* blocksum, u32* seg, u32* d_nslots_next, u32* d_maxcount, cudaStream_t st);
void launch_tile_max(const u32* seg, int ncell, int cpb0, u32* d_tilemax4, cudaStream_t st);
template <typename R>
void launch_scatter(const SdArraysT<R>& src, const SdArraysT<R>& dst, const u32* d_nslots, u32 nslots_bound, const Grid& g,
                    const u32* cell, const u32* off, const u32* seg, cudaStream_t st);
cudaError_t launch_rank(int G, const u32* id, const u32* seg, int ncell, u32 step, u32 seed_lo, u32 seed_hi, int P,
                        u16* rank, int* d_error, cudaStream_t st);
void launch_export_order(const u32* id, const u16* rank, const u32* seg, int ncell, u32* ids_sorted, cudaStream_t st);

// sdm_cond.cu
// cpb: cells per CTA; variant = cond_variant(cpb, most populated tile): 1, 2, 3 = shared-memory tile kernels for
// up to 800 / 1280 / 4096 SDs per tile (in order of preference), 0 = fits none: work in place in global memory
// (cpb == 1, `alt` = idle ping-pong copy used as scratch)
int cond_variant(int cpb, int need);
int cond_max_cells(bool arith32);   // most cells per tile the small tile kernel has room for (sparse cells)
int cond_tile_candidate(int cpb0, int k);   // k-th candidate tile size (cells) tried by k_tile_max, k = 0..3
template <typename R>
cudaError_t launch_cond(int cpb, int variant, const SdArraysT<R>& a, const SdArraysT<R>& alt, const u16* rank, const u32* seg,
                        const Grid& g, Field th, Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt,
                        cudaStream_t st);
size_t cond_smem_bytes(int cpb, int cap);
// the tile kernels (variant 1..3 of cond_variant_f32) with the sweep in fp32 arithmetic (sdm_set_cond_arith; fp32 state only)
int cond_variant_f32(int cpb, int need);
cudaError_t launch_cond_f32(int cpb, int variant, const SdArraysT<float>& a, const u16* rank, const u32* seg, const Grid& g,
                            Field th, Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt, cudaStream_t st);
void launch_thermo(const Grid& g, Field th, Field rv, const CellFields& cf, cudaStream_t st);

// sdm_coal_move.cu
template <typename R>
cudaError_t launch_coal_move(int G, int cap, bool in_smem, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g,
                             const CellFields& cf, const CoalParams& kp, const CoalMoveParams& mp, double* flux_slots,
                             const Counters& cnt, cudaStream_t st);
size_t coal_smem_bytes(int G, int cap, int sstp_coal, bool in_smem);
// tile-resident variant for sstp_coal == 1 (cpb cells per CTA, most populated tile `need` SDs)
bool coal_tile_fits(int cpb, int need, int real_bytes);
// flux_part: one double per CTA (ncell of them suffice); cell_out, off_out, count: next step's a0-a1 when mp.fold
template <typename R>
cudaError_t launch_coal_move_tile(int cpb, int need, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g,
                                  const CellFields& cf, const CoalParams& kp, const CoalMoveParams& mp, double* flux_part,
                                  const Counters& cnt, u32* cell_out, u32* off_out, u32* count, cudaStream_t st);
// the table cf.mv from cf.rhod and the Courant fields
void launch_cell_move_consts(const Grid& g, const CellFields& cf, cudaStream_t st);
// also copies the step's device error flag into flux_out[2], so that one read-back serves both
void launch_flux_sum(double* flux_slots, const double* flux_part, int n_part, double* flux_out, double* flux_total, const u32* d_flag,
                     cudaStream_t st);

// sdm_recycle.cu: recycling of zero-multiplicity SDs (PAPER.md :641, :651; reading R-recycle)
struct __align__(16) RecItem { u64 key; u32 id; u32 slot; };   // ordered by (key, id); key = ~N for donors, 0 for dead SDs
size_t recycle_items_capacity(u64 cap_sd);   // items each of the two lists must hold
// counts the dead SDs (list `dead`, unordered), builds the histogram of multiplicities and picks the threshold bin;
// info (8 u32, device): [0] dead SDs, [1] k = SDs that will be recycled, [2] candidates, [3] threshold bin
void launch_recycle_scan(const u64* n, const u32* id, u32 nslots, RecItem* dead, u32* info, u32* hist, cudaStream_t st);
// collects and orders the donors, orders the dead SDs by id and applies the recycling; synchronises the stream once
// (h_ncand: pinned host word); returns the number of kernels launched
template <typename R>
int launch_recycle_apply(const SdArraysT<R>& a, const Grid& g, u32 nslots, u32 n_dead, u32 k, RecItem* dead, RecItem* cand,
                         u32* info, u32* h_ncand, cudaStream_t st);

// sdm_init.cu
constexpr int INIT_MAX_MODES = 8;
struct sdm_mode_view { double kappa, n_stp, r_mean, sigma_g; };   // same layout as sdm_lognormal_mode (sdm.h)
struct InitParams {
  int n_modes, n_spectra;
  int mode_spectrum[INIT_MAX_MODES];
  double mode_lnr[INIT_MAX_MODES], mode_amp[INIT_MAX_MODES], mode_2ls2[INIT_MAX_MODES];   // ln r_m, N/(sqrt(2 pi) ln s), 2 ln^2 s
  double kappa[INIT_MAX_MODES], lnr_lo[INIT_MAX_MODES], lnr_hi[INIT_MAX_MODES];          // per spectrum
  double sd_conc_spectrum, rho_stp;
  double x0, y0, z0, x1, y1, z1;
  u32 seed_lo, seed_hi;
};
int init_prepare(const sdm_mode_view* modes, int n_modes, double sd_conc_mean, double dV, InitParams& ip);
template <typename R>
void launch_init(const SdArraysT<R>& a, u32 N, const Grid& g, const InitParams& ip, Field th, Field rv, const double* rhod,
                 double* RHeq, double* Akel, cudaStream_t st);

// sdm_diag.cu
template <typename R>
void launch_diag_mom(const SdArraysT<R>& a, const u32* d_nslots, u32 nslots_bound, const Grid& g, int wet, double r_mi,
                     double r_mx, int k, int count_only, const double* rhod, double* out, cudaStream_t st);
void launch_dense_copy(Field src, double* dst, int n0, int n1, int n2, cudaStream_t st);

// sdm_slab.cu: exchange of SDs between slabs of a domain decomposed along x
template <typename R>
void launch_count_leavers(const SdArraysT<R>& a, u32 nslots, const Grid& g, u32* cnt2, cudaStream_t st);
template <typename R>
void launch_pack_leavers(const SdArraysT<R>& a, u32 nslots, const Grid& g, const SdArraysT<R>& left, const SdArraysT<R>& right, u32* cnt2,
                         cudaStream_t st);
template <typename R>
void launch_unpack_arrivals(const SdArraysT<R>& a, u32 first, u32 count, const Grid& g, const SdArraysT<R>& in, double x_shift,
                            cudaStream_t st);

// sdm_euler.cu: one upstream step of a scalar field with the context's rho_d x Courant arrays (tmp: ncell doubles); 2 launches
void launch_upstream(Field psi, const Grid& g, const CellFields& cf, double* tmp, cudaStream_t st);

}  // namespace sdm
