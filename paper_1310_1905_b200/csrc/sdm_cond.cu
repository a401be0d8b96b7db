// Stage a4: condensational growth, all sstp_cond substeps fused in one
// tile-resident kernel.  A CTA of 256 threads owns a TILE of consecutive grid cells (about 1800
// super-droplets): the SDs are staged once in shared memory in sorted order and stay there for all
// substeps.  Per substep
//   A. one thread per cell applies the feedback of the previous substep (eq. 25-26) and
//      diagnoses T, p, rho_vs, RH.. from theta, r_v, rho_d (eq. 43-44, Table 2),
//   B. all threads sweep the tile's SDs DENSELY (lane utilisation does not depend on the cell
//      populations) and solve eq. 17 by a bracketed Newton iteration on r_w^2 inside the interval of
//      eq. 18-19 (the paper bisects, :579, and names a faster root finder as the first optimisation,
//      :912); the sweep spends at most `kfast` growth-rate evaluations per SD,
//   C. the few SDs that did not converge in B are collected in a list and solved to the end in a second,
//      again densely packed, pass (so one slow SD does not hold 31 lanes for its whole iteration),
//   D. one warp per cell sums N (r_w^3' - r_w^3) in sorted order (deterministic) for the next feedback.
// The solver is a small state machine around ONE inlined growth-rate evaluation, so that lanes of a
// warp differ only in their trip count.  fp64 throughout; this kernel is fp64-ALU bound.
#include "sdm_kernels.cuh"

namespace sdm {

constexpr int COND_THREADS = 256;
constexpr int COND_WARPS = COND_THREADS / 32;

struct CellK {   // per-cell constants of one substep (shared memory, SoA over the tile's cells)
  double RH, A, c0, lD, lK, heat, kE, Sc, Pr;
};
constexpr int CELLK_N = 9;

// [L] Sherwood / Nusselt number (Clift et al.): 1 + (1 + Re X)^(1/3) max(1, Re^0.077)
__device__ __forceinline__ double vent(double Re, double X) {
  const double x = Re * X;
  double cb;
  if (x < 2.5e-4) {   // (1+x)^(1/3) by its series, truncation < 2e-16
    cb = 1.0 + x * (1.0 / 3.0 + x * (-1.0 / 9.0 + x * (5.0 / 81.0)));
  } else {
    cb = cbrt(1.0 + x);
  }
  const double m = (Re > 1.0) ? pow(Re, 0.077) : 1.0;
  return 1.0 + cb * m;
}

struct SdK {   // per-SD constants of one substep
  double rd3, krd3;   // r_d^3, kappa r_d^3
  double Kc, hDc;     // K_0 Nu/2 (eq. 24 without beta_T), heat * D_0 Sh/2
  double cDK;         // c0 * Dc * Kc
};

// Growth rate f(y) = d r_w^2/dt (eq. 20-24) and df/dy at y = r_w^2, written with one reciprocal:
//   beta_M = N_M/D_M, beta_T = N_T/D_T (Fuchs-Sutugin multiplied through by r^2),
//   D_eff = Dc Kc N_M N_T / Q,  Q = Kc N_T D_M + heat Dc N_M D_T,
//   a_w = P/W, P = r^3 - r_d^3, W = P + kappa r_d^3,  f = c0 D_eff (RH - a_w exp(A/r)).
__device__ __forceinline__ void growth_fd(double y, const SdK& s, const CellK& c, double& f, double& df) {
  const double invr = rsqrt(y);
  const double r = y * invr;
  const double lDr = c.lD * r, lKr = c.lK * r;
  const double NM = y + lDr, DM = fma(1.71, lDr, y) + 1.33 * (c.lD * c.lD);
  const double NT = y + lKr, DT = fma(1.71, lKr, y) + 1.33 * (c.lK * c.lK);
  const double KN = s.Kc * NT, HN = s.hDc * NM;
  const double Q = fma(KN, DM, HN * DT);
  const double r3 = y * r;
  const double P = r3 - s.rd3, W = P + s.krd3;
  const double ex = exp(c.A * invr);
  const double invQW = 1.0 / (Q * W);
  const double invQ = invQW * W, invW = invQW * Q;
  const double NN = NM * NT;
  const double aw = P * invW;
  const double S = c.RH - aw * ex;
  const double cD = s.cDK * invQ;
  f = cD * NN * S;
  // derivative
  const double hr = 0.5 * invr;   // dr/dy
  const double NMp = fma(c.lD, hr, 1.0), DMp = fma(1.71 * c.lD, hr, 1.0);
  const double NTp = fma(c.lK, hr, 1.0), DTp = fma(1.71 * c.lK, hr, 1.0);
  const double NNp = fma(NMp, NT, NM * NTp);
  const double Qp = s.Kc * fma(NTp, DM, NT * DMp) + s.hDc * fma(NMp, DT, NM * DTp);
  const double awp = 1.5 * r * s.krd3 * (invW * invW);
  const double Sp = -ex * (awp - aw * (c.A * hr) * (invr * invr));
  df = cD * fma(NNp - NN * (Qp * invQ), S, NN * Sp);
}

// ---- fast path (k_cond3): the same equations written in r = sqrt(y), which stays resident in shared
// memory over the substeps (no sqrt per substep), with one reciprocal per evaluation.
// 1/a from the hardware seed (MUFU.RCP64H, ~2^-20) and NR Newton-Raphson refinements (2 -> < 1 ulp)
template <int NR>
__device__ __forceinline__ double rcp_nr(double a) {
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(a));
#pragma unroll
  for (int k = 0; k < NR; ++k) {
    const double e = fma(-a, x, 1.0);
    x = fma(x, e, x);
  }
  return x;
}

struct CellR {   // per-cell constants of one substep used by the fast path
  double RH, A, lD, lK, qD, qK, lD171, lK171;
  float kE, Sc, Pr;
};

// f(r) = d r_w^2/dt (eq. 20-24) and df/dr; also returns y = r^2.  Notation as growth_fd.
__device__ __forceinline__ void growth_r(double r, const SdK& s, const CellR& c, double& y, double& f, double& dfr) {
  y = r * r;
  const double lDr = c.lD * r, lKr = c.lK * r;
  const double NM = y + lDr, DM = fma(1.71, lDr, y) + c.qD;
  const double NT = y + lKr, DT = fma(1.71, lKr, y) + c.qK;
  const double KN = s.Kc * NT, HN = s.hDc * NM;
  const double Q = fma(KN, DM, HN * DT);
  const double r3 = y * r;
  const double P = r3 - s.rd3, W = P + s.krd3;
  const double QW = Q * W;
  const double inv = rcp_nr<2>(r * QW);
  const double invr = inv * QW, invQ = inv * (r * W), invW = inv * (r * Q);
  const double t = c.A * invr;
  const double ex = exp(t);
  const double NN = NM * NT;
  const double aw = P * invW;
  const double S = fma(-aw, ex, c.RH);
  const double cD = s.cDK * invQ;
  f = cD * NN * S;
  const double r2 = r + r;
  const double NMp = r2 + c.lD, DMp = r2 + c.lD171;
  const double NTp = r2 + c.lK, DTp = r2 + c.lK171;
  const double NNp = fma(NMp, NT, NM * NTp);
  const double Qp = s.Kc * fma(NTp, DM, NT * DMp) + s.hDc * fma(NMp, DT, NM * DTp);
  const double awp = 3.0 * y * s.krd3 * (invW * invW);
  const double Sp = ex * fma(aw, t * invr, -awp);
  dfr = cD * fma(NNp - NN * (Qp * invQ), S, NN * Sp);
}

// (1+x)^(1/3) - 1 by the binomial series, truncation < 1e-17 for 0 <= x < 0.02
__device__ __forceinline__ double cbrt1pm1_small(double x) {
  double p = -935.0 / 59049.0;
  p = fma(p, x, 374.0 / 19683.0);
  p = fma(p, x, -154.0 / 6561.0);
  p = fma(p, x, 22.0 / 729.0);
  p = fma(p, x, -10.0 / 243.0);
  p = fma(p, x, 5.0 / 81.0);
  p = fma(p, x, -1.0 / 9.0);
  p = fma(p, x, 1.0 / 3.0);
  return p * x;
}

// [L] ventilation at the substep's starting radius r0 (reading R-vent) -> per-SD constants.
// Re·Sc below 2.5e-4 (r0 below ~3 um): Sh - 2 < 1e-4 enters D only through 2 + (Sh - 2), so Re and the
// series are evaluated in fp32 (relative error 3e-7 of a 1e-4 term: < 3e-11 of D).  Above: fp64.
__device__ __forceinline__ void sd_setup(double r0, double c0, double heat, double kE, double Sc, double Pr,
                                         const CellR& c, SdK& s) {
  const float rf = (float)r0;
  const float ef = c.kE * rf * sqrtf(rf);
  const float qf = ef / (sqrtf(1.0f + ef) + 1.0f);
  const float Ref = (float)(cst::kc_delta0 * cst::kc_delta0 / 4.0) * (qf * qf);
  const float xs = Ref * c.Sc, xp = Ref * c.Pr;
  double shm, num;   // Sh - 2, Nu - 2
  if (fmaxf(xs, xp) < 2.5e-4f) {
    shm = (double)(xs * (1.0f / 3.0f + xs * (-1.0f / 9.0f + xs * (5.0f / 81.0f))));
    num = (double)(xp * (1.0f / 3.0f + xp * (-1.0f / 9.0f + xp * (5.0f / 81.0f))));
  } else {
    const double e = kE * (r0 * sqrt(r0));
    const double q = e / (sqrt(1.0 + e) + 1.0);
    const double Re = (cst::kc_delta0 * cst::kc_delta0 / 4.0) * (q * q);
    const double x1 = Re * Sc, x2 = Re * Pr;
    if (Re <= 1.0 && fmax(x1, x2) < 0.02) {
      shm = cbrt1pm1_small(x1);
      num = cbrt1pm1_small(x2);
    } else {
      shm = vent(Re, Sc) - 2.0;
      num = vent(Re, Pr) - 2.0;
    }
  }
  const double Dc = fma(0.5 * cst::D_0, shm, cst::D_0);   // eq. 23 without beta_M: D_0 Sh / 2
  s.Kc = fma(0.5 * cst::K_0, num, cst::K_0);              // eq. 24 without beta_T: K_0 Nu / 2
  s.hDc = heat * Dc;
  s.cDK = c0 * Dc * s.Kc;
}

// One condensation substep of one SD: root of g(y) = y - y0 - dt' f(y) in [a, b] of eq. 18-19
// (reading R-bracket), with the ill-posed-bracket rule of :579.  Newton steps are kept
// inside the shrinking bracket [lo, hi]; a step that leaves it is replaced by a bisection, and before
// the first departure through an end that has never been evaluated the sign of g there decides whether
// the bracket is well-posed at all.  Returns false when `max_evals` evaluations did not suffice.
//
// Stopping rule for a Newton step of size d_k from an iterate whose previous step was d_(k-1):
// the error left after the step is C d_k^2 with C = |g''/(2g')|, estimated by d_k/d_(k-1)^2 and
// bounded below by 1/y (first step: 100/y); stop when that is below 1e-11 y.
enum { M_FIRST = 0, M_MAIN = 1, M_CHK_A = 2, M_CHK_B = 3 };

__device__ __forceinline__ bool cond_solve(double y0, double rd2, double rd3, double krd3, const CellK& c, double dtp,
                                           int max_evals, double& y_out, unsigned& n_ill, unsigned& n_eval) {
  SdK s;
  s.rd3 = rd3; s.krd3 = krd3;
  {
    // [L] ventilation at the substep's starting radius (reading R-vent); Re from the terminal
    // velocity of Khvorostyanov & Curry 2002: e = c1 sqrt(X) = kE r^(3/2)
    const double r0 = sqrt(y0);
    const double e = c.kE * (r0 * sqrt(r0));
    const double q = e / (sqrt(1.0 + e) + 1.0);
    const double Re = (cst::kc_delta0 * cst::kc_delta0 / 4.0) * (q * q);
    const double Dc = cst::D_0 * vent(Re, c.Sc) * 0.5;   // eq. 23 without beta_M
    s.Kc = cst::K_0 * vent(Re, c.Pr) * 0.5;              // eq. 24 without beta_T
    s.hDc = c.heat * Dc;
    s.cDK = c.c0 * Dc * s.Kc;
  }
  int mode = M_FIRST;
  double yE = y0, y = y0, g = 0.0, gp = 1.0, a = 0.0, b = 0.0, lo = 0.0, hi = 0.0, dprev = 0.0;
  bool lo_unv = false, hi_unv = false;
  for (int it = 0; it < max_evals; ++it) {
    double f, df;
    growth_fd(yE, s, c, f, df);   // the only evaluation site
    ++n_eval;
    bool bisect = false;
    if (mode == M_FIRST) {
      const double two = 2.0 * dtp * f;
      a = fmax(rd2, y0 + fmin(two, 0.0));   // eq. 18
      b = y0 + fmax(two, 0.0);              // eq. 19
      if (!(a < b)) { y_out = a; return true; }
      // g(lo) < 0 < g(hi) is what a well-posed bracket means; the end that is not y0 is unverified
      lo = a; hi = b;
      lo_unv = !(f > 0.0); hi_unv = (f > 0.0);
      g = -dtp * f; gp = fma(-dtp, df, 1.0);
    } else if (mode == M_CHK_B) {
      const double gb = b - y0 - dtp * f;
      if (gb == 0.0) { y_out = b; return true; }
      if (gb < 0.0) { n_ill += (b - a > 1e-9 * b); y_out = 0.5 * (a + b); return true; }   // :579
      hi_unv = false; bisect = true;
    } else if (mode == M_CHK_A) {
      const double ga = a - y0 - dtp * f;
      if (ga == 0.0) { y_out = a; return true; }
      if (ga > 0.0) { n_ill += (b - a > 1e-9 * b); y_out = 0.5 * (a + b); return true; }
      lo_unv = false; bisect = true;
    } else {
      y = yE;
      g = y - y0 - dtp * f; gp = fma(-dtp, df, 1.0);
      if (g == 0.0) { y_out = y; return true; }
      if (g < 0.0) { lo = y; lo_unv = false; } else { hi = y; hi_unv = false; }
    }
    // next point
    double yn;
    bool newton = !bisect;
    if (newton) {
      yn = (gp > 0.0) ? y - g / gp : (g < 0.0 ? hi : lo);
      if (!(yn > lo && yn < hi)) {
        newton = false;
        if (g < 0.0 && hi_unv) { mode = M_CHK_B; yE = b; continue; }
        if (g > 0.0 && lo_unv) { mode = M_CHK_A; yE = a; continue; }
      }
    }
    if (!newton) yn = 0.5 * (lo + hi);
    const double d = fabs(yn - y);
    y = yn;
    bool conv;
    if (newton) {
      const double tol = 1e-11 * y;
      const double d2 = d * d;
      conv = (dprev > 0.0) ? (d2 <= tol * y && d2 * d <= tol * (dprev * dprev)) : (100.0 * d2 <= tol * y);
      dprev = d;
    } else {
      conv = d <= 2e-16 * y;   // a bisection step bounds the error directly
      dprev = 0.0;
    }
    if (conv || !(hi - lo > 1e-15 * hi)) { y_out = y; return true; }
    mode = M_MAIN; yE = y;
  }
  return false;
}

// per-cell constants of one substep from theta, r_v, rho_d; returns T and l_v for the feedback of eq. 26
__device__ __forceinline__ void cell_consts(double th, double rv, double rhod, double c_exn, double RH_max, CellK& c,
                                            double& T_out, double& lv_out) {
  // eq. 43: T = [theta (rhod R_d/p_1000)^(R_d/c_pd)]^(c_pd/(c_pd-R_d)); c_exn is the inner power (rhod is fixed)
  const double T = pow(th * c_exn, cst::c_pd / (cst::c_pd - cst::R_d));
  const double p = rhod * (cst::R_d + rv * cst::R_v) * T;                 // eq. 44
  const double lv = cst::l_v0 + (cst::c_pv - cst::c_l) * (T - cst::T_0);  // Table 2 :1087
  // [L] Clausius-Clapeyron integral for the linear l_v(T)
  const double ca = (cst::l_v0 + (cst::c_l - cst::c_pv) * cst::T_0) / cst::R_v;
  const double cb = (cst::c_l - cst::c_pv) / cst::R_v;
  const double pvs = cst::p_vs0 * exp(ca * (1.0 / cst::T_0 - 1.0 / T) - cb * log(T / cst::T_0));
  const double rho_vs = pvs / (cst::R_v * T);
  T_out = T; lv_out = lv;
  c.RH = fmin(rv * rhod / rho_vs, RH_max);                                // eq. 30, :685
  c.A = 2.0 * cst::sigma_w / (cst::R_v * T * cst::rho_w);                 // Table 2 :1056
  c.c0 = 2.0 * rho_vs / cst::rho_w;
  c.lD = 2.0 * cst::D_0 / sqrt(2.0 * cst::R_v * T);                       // [L] Fuchs-Sutugin lengths
  c.lK = (4.0 / 5.0) * cst::K_0 * T / (p * sqrt(2.0 * cst::R_d * T));
  c.heat = (rho_vs * lv / T) * (lv / (cst::R_v * T) - 1.0);               // eq. 21
  const double eta = eta_air(T);
  const double rho_a = rhod * (1.0 + rv);
  // e = c1 sqrt(X), X = (32/3) r^3 (rho_w - rho_a) g rho_a / eta^2  ->  e = kE r^(3/2)
  const double c1 = 4.0 / (cst::kc_delta0 * cst::kc_delta0 * sqrt(cst::kc_C0));
  c.kE = c1 * sqrt((32.0 / 3.0) * (cst::rho_w - rho_a) * cst::g * rho_a) / eta;
  c.Sc = eta / (rho_a * cst::D_0);
  c.Pr = eta * cst::c_pd / cst::K_0;
}

// Shared memory of one CTA (SMEM variant), cap = SD slots, cpb = cells per tile:
//   double cell[(CELLK_N + 1) * cpb]   constants of the substep + the cell's sum of N d(r_w^3)
//   double sd[6 * cap]                 y = r_w^2, r_d^3, kappa r_d^3, N, r_d^2, N d(r_w^3)  (sorted order)
//   u32 segl[cpb + 2]                  tile-local segment offsets, list counter
//   u16 cidx[cap], list[cap]           local cell of each slot; slots left for the second pass
// GMEM variant (a cell too crowded for shared memory; cpb = 1): the state stays in HBM/L2 in storage
// order, contributions go to alt.rw2 in sorted order, the list to alt.id.
size_t cond_smem_bytes(int cpb, int cap) {
  return (size_t)(CELLK_N + 1) * cpb * 8 + (size_t)6 * cap * 8 + (size_t)(cpb + 2) * 4 + (size_t)cap * 4 + 16;
}

template <bool SMEM>
__global__ void __launch_bounds__(COND_THREADS, 2)
k_cond(SdArrays a, SdArrays alt, const u16* __restrict__ rank, const u32* __restrict__ seg, Grid g, Field th_f, Field rv_f,
       CellFields cf, CondParams cp, Counters cnt, int cpb, int cap) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c_first = blockIdx.x * cpb;
  const int nc = min(cpb, g.ncell - c_first);
  double* s_cell = reinterpret_cast<double*>(smem_raw);
  double* s_sum = s_cell + CELLK_N * cpb;
  double* s_sd = s_cell + (CELLK_N + 1) * cpb;
  const int capd = SMEM ? cap : 0;
  double *s_y = s_sd, *s_rd3 = s_sd + capd, *s_krd3 = s_sd + 2 * capd, *s_dn = s_sd + 3 * capd, *s_rd2 = s_sd + 4 * capd;
  double* s_con = s_sd + 5 * capd;
  u32* segl = reinterpret_cast<u32*>(s_sd + 6 * capd);
  u32* list_n = segl + cpb + 1;
  u16* cidx = reinterpret_cast<u16*>(segl + cpb + 2);
  u16* list16 = cidx + capd;
  const u32 s0 = seg[c_first];
  const int M = (int)(seg[c_first + nc] - s0);
  u32* list32 = alt.id + s0;
  if constexpr (!SMEM) s_con = alt.rw2 + s0;

  // thread `tid` owns cell c_first + tid for the whole kernel: theta, r_v and the feedback live in its registers
  double th = 0, rv = 0, rhod = 1, c_exn = 0, fbk = 0, T = 0, lv = 0;
  int ci = 0, cj = 0, ck = 0;
  if (tid < nc) {
    const int c = c_first + tid;
    ck = c % g.NZ; cj = (c / g.NZ) % g.NY; ci = c / (g.NZ * g.NY);
    th = th_f.at(ci, cj, ck); rv = rv_f.at(ci, cj, ck);
    rhod = cf.rhod[c];
    c_exn = pow(rhod * cst::R_d / cst::p_1000, cst::R_d / cst::c_pd);
    fbk = -(4.0 * cst::pi * cst::rho_w / 3.0) / (rhod * g.dV);   // eq. 25 prefactor
    segl[tid] = seg[c] - s0;
    s_sum[tid] = 0.0;
  }
  if (tid == 0) segl[nc] = (u32)M;
  __syncthreads();

  // stage the tile in sorted order (coalesced reads; the cell of a slot by binary search in segl)
  if constexpr (SMEM) {
    for (int t = tid; t < M; t += COND_THREADS) {
      int lo = 0, hi = nc;   // segl[lo] <= t < segl[hi]
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)t) lo = mid; else hi = mid; }
      const u32 s = s0 + t;
      const int e = (int)segl[lo] + rank[s];
      const double rd3 = a.rd3[s];
      const double q = cbrt(rd3);
      s_y[e] = a.rw2[s];
      s_rd3[e] = rd3;
      s_krd3[e] = a.kappa[s] * rd3;
      s_dn[e] = (double)a.n[s];
      s_rd2[e] = q * q;
      cidx[e] = (u16)lo;
    }
  }

  unsigned n_ill = 0, n_eval = 0, n_sub = 0, n_slow = 0;
  for (int sub = 0; sub < cp.sstp && M > 0; ++sub) {
    // A. feedback of the previous substep (eq. 25-26, old theta and T) and the new cell constants
    if (tid < nc) {
      if (sub > 0) {
        const double drv = fbk * s_sum[tid];
        th += drv * (-th * lv / (cst::c_pd * T));
        rv += drv;
      }
      CellK c;
      cell_consts(th, rv, rhod, c_exn, cp.RH_max, c, T, lv);
      s_cell[0 * cpb + tid] = c.RH; s_cell[1 * cpb + tid] = c.A; s_cell[2 * cpb + tid] = c.c0;
      s_cell[3 * cpb + tid] = c.lD; s_cell[4 * cpb + tid] = c.lK; s_cell[5 * cpb + tid] = c.heat;
      s_cell[6 * cpb + tid] = c.kE; s_cell[7 * cpb + tid] = c.Sc; s_cell[8 * cpb + tid] = c.Pr;
    }
    if (tid == 0) *list_n = 0u;
    __syncthreads();

    // B/C. pass 0: dense sweep with at most kfast evaluations per SD; pass 1: the listed rest, to the end
    for (int pass = 0; pass < 2; ++pass) {
      const int count = pass == 0 ? M : (int)*list_n;
      const int max_evals = pass == 0 ? cp.kfast : 200;
      for (int q0 = warp * 32; q0 < count; q0 += COND_THREADS) {
        const int q = q0 + lane;
        const bool valid = q < count;
        bool done = true;
        int e = 0;
        if (valid) {
          if (pass == 0) e = q; else e = SMEM ? (int)list16[q] : (int)list32[q];
          double y0, rd3, krd3, rd2, dn;
          int cl = 0, econ = e;
          if constexpr (SMEM) {
            y0 = s_y[e]; rd3 = s_rd3[e]; krd3 = s_krd3[e]; rd2 = s_rd2[e]; dn = s_dn[e];
            cl = cidx[e];
          } else {
            const u32 s = s0 + e;
            y0 = a.rw2[s]; rd3 = a.rd3[s]; krd3 = a.kappa[s] * rd3; dn = (double)a.n[s];
            const double qq = cbrt(rd3);
            rd2 = qq * qq;
            econ = rank[s];
          }
          CellK c;
          c.RH = s_cell[0 * cpb + cl]; c.A = s_cell[1 * cpb + cl]; c.c0 = s_cell[2 * cpb + cl];
          c.lD = s_cell[3 * cpb + cl]; c.lK = s_cell[4 * cpb + cl]; c.heat = s_cell[5 * cpb + cl];
          c.kE = s_cell[6 * cpb + cl]; c.Sc = s_cell[7 * cpb + cl]; c.Pr = s_cell[8 * cpb + cl];
          double y1 = y0;
          unsigned ill = 0;
          done = cond_solve(y0, rd2, rd3, krd3, c, cp.dtp, max_evals, y1, ill, n_eval);
          if (done) {
            n_ill += ill;
            ++n_sub;
            s_con[econ] = dn * (y1 * sqrt(y1) - y0 * sqrt(y0));
            if constexpr (SMEM) s_y[e] = y1; else a.rw2[s0 + e] = y1;
          }
        }
        if (pass == 0) {   // warp-aggregated append of the unfinished slots
          const unsigned need = __ballot_sync(0xffffffffu, !done);
          if (need) {
            u32 base = 0;
            if (lane == 0) base = atomicAdd(list_n, (u32)__popc(need));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (!done) {
              const u32 pos = base + __popc(need & ((1u << lane) - 1u));
              if constexpr (SMEM) list16[pos] = (u16)e; else list32[pos] = (u32)e;
              ++n_slow;
            }
          }
        }
      }
      __syncthreads();
    }

    // D. per-cell sum of N d(r_w^3) in sorted order: lane-strided partial sums, xor butterfly
    for (int cl = warp; cl < nc; cl += COND_WARPS) {
      const int b0 = (int)segl[cl], b1 = (int)segl[cl + 1];
      double acc = 0.0;
      for (int e = b0 + lane; e < b1; e += 32) acc += s_con[e];
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
      if (lane == 0) s_sum[cl] = acc;
    }
    __syncthreads();
  }

  if (tid < nc) {
    if (M > 0) {   // feedback of the last substep
      const double drv = fbk * s_sum[tid];
      th += drv * (-th * lv / (cst::c_pd * T));
      rv += drv;
    }
    th_f.at(ci, cj, ck) = th;
    rv_f.at(ci, cj, ck) = rv;
    // air properties after the feedback, used by coalescence and sedimentation (v_term)
    const double Tn = pow(th * c_exn, cst::c_pd / (cst::c_pd - cst::R_d));
    cf.eta[c_first + tid] = eta_air(Tn);
    cf.rho_a[c_first + tid] = rhod * (1.0 + rv);
  }
  if constexpr (SMEM) {
    for (int t = tid; t < M; t += COND_THREADS) {
      int lo = 0, hi = nc;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)t) lo = mid; else hi = mid; }
      const u32 s = s0 + t;
      a.rw2[s] = s_y[(int)segl[lo] + rank[s]];
    }
  }
  // counters: one atomic per warp and counter, spread over NSLOT addresses
  unsigned v0 = n_ill, v1 = n_eval, v2 = n_sub, v3 = n_slow;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    v0 += __shfl_xor_sync(0xffffffffu, v0, d);
    v1 += __shfl_xor_sync(0xffffffffu, v1, d);
    v2 += __shfl_xor_sync(0xffffffffu, v2, d);
    v3 += __shfl_xor_sync(0xffffffffu, v3, d);
  }
  if (lane == 0) {
    const int slot = (blockIdx.x * COND_WARPS + warp) & (NSLOT - 1);
    if (v0) atomicAdd(&cnt.ill_posed[slot], (unsigned long long)v0);
    if (v1) atomicAdd(&cnt.f_evals[slot], (unsigned long long)v1);
    if (v2) atomicAdd(&cnt.sd_substeps[slot], (unsigned long long)v2);
    if (v3) atomicAdd(&cnt.cond_slow[slot], (unsigned long long)v3);
  }
}

// ---- k_cond3: the shared-memory tile kernel, third version ---------------------------------------
// Differences from k_cond<true> (kept above for cells too crowded for shared memory):
//  * r_w (not r_w^2) is resident in shared memory: no sqrt per substep, N d(r_w^3) by two products;
//  * the sweep is straight-line code around growth_r with a warp-uniform iteration loop; anything
//    irregular (Newton leaving the bracket of eq. 18-19, an end to verify, slow convergence) is
//    put on a WARP-private list and solved afterwards by cond_solve, the robust state machine;
//  * small CTAs (T3 threads, several per SM) so that the serial phases of one tile (cell constants,
//    slow list, barriers) overlap the sweeps of the others.
// Shared memory: double cell[C3_N * cpb]; double sd[6 * cap] = r, r_d^3, kappa r_d^3, N, r_d^2,
// N d(r_w^3); float cellf[3 * cpb]; u32 segl[cpb + 1]; u16 cidx[cap]; u16 list[lstride * warps].
constexpr int C3_N = 12;   // RH, A, c0, lD, lK, heat, kE, Sc, Pr, qD, qK, sum
constexpr int T3 = 128;
static int c3_lstride(int cap) { return ((cap + T3 - 1) / T3) * 32; }
size_t cond3_smem_bytes(int cpb, int cap) {
  return (size_t)C3_N * cpb * 8 + (size_t)6 * cap * 8 + (size_t)3 * cpb * 4 + (size_t)(cpb + 1) * 4 + (size_t)cap * 2 +
         (size_t)c3_lstride(cap) * (T3 / 32) * 2 + 32;
}

__global__ void __launch_bounds__(T3, 5)
k_cond3(SdArrays a, const u16* __restrict__ rank, const u32* __restrict__ seg, Grid g, Field th_f, Field rv_f,
        CellFields cf, CondParams cp, Counters cnt, int cpb, int cap, int lstride) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NW = T3 / 32;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c_first = blockIdx.x * cpb;
  const int nc = min(cpb, g.ncell - c_first);
  double* s_cell = reinterpret_cast<double*>(smem_raw);
  double* s_sum = s_cell + 11 * cpb;
  double* s_r = s_cell + C3_N * cpb;
  double *s_rd3 = s_r + cap, *s_krd3 = s_r + 2 * cap, *s_dn = s_r + 3 * cap, *s_rd2 = s_r + 4 * cap, *s_con = s_r + 5 * cap;
  float* s_cf = reinterpret_cast<float*>(s_r + 6 * cap);
  u32* segl = reinterpret_cast<u32*>(s_cf + 3 * cpb);
  u16* cidx = reinterpret_cast<u16*>(segl + cpb + 1);
  u16* mylist = cidx + ((cap + 1) & ~1) + warp * lstride;
  const u32 s0 = seg[c_first];
  const int M = (int)(seg[c_first + nc] - s0);

  // thread `tid` owns cell c_first + tid: theta, r_v and the feedback live in its registers
  double th = 0, rv = 0, rhod = 1, c_exn = 0, fbk = 0, T = 0, lv = 0;
  int ci = 0, cj = 0, ck = 0;
  if (tid < nc) {
    const int c = c_first + tid;
    ck = c % g.NZ; cj = (c / g.NZ) % g.NY; ci = c / (g.NZ * g.NY);
    th = th_f.at(ci, cj, ck); rv = rv_f.at(ci, cj, ck);
    rhod = cf.rhod[c];
    c_exn = pow(rhod * cst::R_d / cst::p_1000, cst::R_d / cst::c_pd);
    fbk = -(4.0 * cst::pi * cst::rho_w / 3.0) / (rhod * g.dV);   // eq. 25 prefactor
    segl[tid] = seg[c] - s0;
    s_sum[tid] = 0.0;
  }
  if (tid == 0) segl[nc] = (u32)M;
  __syncthreads();
  for (int t = tid; t < M; t += T3) {   // stage the tile in sorted order
    int lo = 0, hi = nc;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)t) lo = mid; else hi = mid; }
    const u32 s = s0 + t;
    const int e = (int)segl[lo] + rank[s];
    const double rd3 = a.rd3[s];
    const double q = cbrt(rd3);
    s_r[e] = sqrt(a.rw2[s]);
    s_rd3[e] = rd3;
    s_krd3[e] = a.kappa[s] * rd3;
    s_dn[e] = (double)a.n[s];
    s_rd2[e] = q * q;
    cidx[e] = (u16)lo;
  }
  unsigned n_ill = 0, n_eval = 0, n_sub = 0, n_slow = 0;
  for (int sub = 0; sub < cp.sstp && M > 0; ++sub) {
    // A. feedback of the previous substep (eq. 25-26, old theta and T) and the new cell constants
    if (tid < nc) {
      if (sub > 0) {
        const double drv = fbk * s_sum[tid];
        th += drv * (-th * lv / (cst::c_pd * T));
        rv += drv;
      }
      CellK c;
      cell_consts(th, rv, rhod, c_exn, cp.RH_max, c, T, lv);
      s_cell[0 * cpb + tid] = c.RH; s_cell[1 * cpb + tid] = c.A; s_cell[2 * cpb + tid] = c.c0;
      s_cell[3 * cpb + tid] = c.lD; s_cell[4 * cpb + tid] = c.lK; s_cell[5 * cpb + tid] = c.heat;
      s_cell[6 * cpb + tid] = c.kE; s_cell[7 * cpb + tid] = c.Sc; s_cell[8 * cpb + tid] = c.Pr;
      s_cell[9 * cpb + tid] = 1.33 * (c.lD * c.lD); s_cell[10 * cpb + tid] = 1.33 * (c.lK * c.lK);
      s_cf[0 * cpb + tid] = (float)c.kE; s_cf[1 * cpb + tid] = (float)c.Sc; s_cf[2 * cpb + tid] = (float)c.Pr;
    }
    __syncthreads();
    // B. dense sweep.  st: 0 = iterating, 1 = solved, 2 = left to cond_solve (warp-private list)
    int nslow = 0;
    const double dtp = cp.dtp;
    for (int q0 = warp * 32; q0 < M; q0 += T3) {
      const int e = q0 + lane;
      const bool valid = e < M;
      const int cl = valid ? (int)cidx[e] : 0;
      const double r0 = valid ? s_r[e] : 1e-6;
      const double rd2 = valid ? s_rd2[e] : 1e-14;
      SdK s;
      s.rd3 = valid ? s_rd3[e] : 1e-21;
      s.krd3 = valid ? s_krd3[e] : 1e-21;
      CellR c;
      c.RH = s_cell[0 * cpb + cl]; c.A = s_cell[1 * cpb + cl]; c.lD = s_cell[3 * cpb + cl]; c.lK = s_cell[4 * cpb + cl];
      c.qD = s_cell[9 * cpb + cl]; c.qK = s_cell[10 * cpb + cl];
      c.lD171 = 1.71 * c.lD; c.lK171 = 1.71 * c.lK;
      c.kE = s_cf[0 * cpb + cl]; c.Sc = s_cf[1 * cpb + cl]; c.Pr = s_cf[2 * cpb + cl];
      sd_setup(r0, s_cell[2 * cpb + cl], s_cell[5 * cpb + cl], s_cell[6 * cpb + cl], s_cell[7 * cpb + cl],
               s_cell[8 * cpb + cl], c, s);
      double y0, f, dfr;
      growth_r(r0, s, c, y0, f, dfr);
      n_eval += valid;
      const double two = 2.0 * dtp * f;
      double lo = fmax(rd2, y0 + fmin(two, 0.0));   // eq. 18
      double hi = y0 + fmax(two, 0.0);              // eq. 19
      double r = r0, dprev = 0.0;
      int st;
      if (!(lo < hi)) {
        st = (lo == y0) ? 1 : 2;                    // a = b: the result is a
      } else {
        const double gp = fma(-dtp, dfr, r0 + r0);
        const double rn = fma(dtp * f, rcp_nr<1>(gp), r0);
        const double yn = rn * rn;
        if (!(gp > 0.0 && yn >= lo && yn <= hi)) {   // a step that rounds to nothing stays on the end it started from
          st = 2;
        } else {
          dprev = fabs(rn - r0);
          r = rn;
          st = (400.0 * (dprev * dprev) <= 1e-11 * (rn * rn)) ? 1 : 0;
        }
      }
      if (!valid) st = 1;
      for (int it = 1; it < cp.kfast; ++it) {
        if (!__any_sync(0xffffffffu, st == 0)) break;
        if (st == 0) {
          double y;
          growth_r(r, s, c, y, f, dfr);
          ++n_eval;
          const double gv = y - y0 - dtp * f;
          const double gp = fma(-dtp, dfr, r + r);
          if (gv < 0.0) lo = y; else hi = y;
          const double rn = fma(-gv, rcp_nr<1>(gp), r);
          const double yn = rn * rn;
          if (!(gp > 0.0 && yn >= lo && yn <= hi)) {   // a step that rounds to nothing stays on the end it started from
            st = 2;
          } else {
            const double d = fabs(rn - r);
            const double tol = 1e-11 * rn, d2 = d * d;
            const bool conv = (4.0 * d2 <= tol * rn) && (2.0 * d2 * d <= tol * (dprev * dprev));
            r = rn; dprev = d;
            if (conv || !(hi - lo > 1e-15 * hi)) st = 1;
          }
        }
      }
      if (st == 0) st = 2;
      if (valid && st == 1) {
        s_con[e] = s_dn[e] * (r * r * r - r0 * y0);
        s_r[e] = r;
        ++n_sub;
      }
      const unsigned need = __ballot_sync(0xffffffffu, st == 2);
      if (st == 2) mylist[nslow + __popc(need & ((1u << lane) - 1u))] = (u16)e;
      nslow += __popc(need);
    }
    __syncwarp();
    // C. the listed rest: the bracketed state machine, from the start of the substep
    for (int k0 = 0; k0 < nslow; k0 += 32) {
      const int k = k0 + lane;
      if (k < nslow) {
        const int e = (int)mylist[k];
        const int cl = (int)cidx[e];
        CellK c;
        c.RH = s_cell[0 * cpb + cl]; c.A = s_cell[1 * cpb + cl]; c.c0 = s_cell[2 * cpb + cl];
        c.lD = s_cell[3 * cpb + cl]; c.lK = s_cell[4 * cpb + cl]; c.heat = s_cell[5 * cpb + cl];
        c.kE = s_cell[6 * cpb + cl]; c.Sc = s_cell[7 * cpb + cl]; c.Pr = s_cell[8 * cpb + cl];
        const double r0 = s_r[e], y0 = r0 * r0;
        double y1 = y0;
        unsigned ill = 0;
        cond_solve(y0, s_rd2[e], s_rd3[e], s_krd3[e], c, dtp, 200, y1, ill, n_eval);
        const double r1 = sqrt(y1);
        n_ill += ill;
        ++n_sub; ++n_slow;
        s_con[e] = s_dn[e] * (r1 * r1 * r1 - r0 * y0);
        s_r[e] = r1;
      }
    }
    __syncthreads();
    // D. per-cell sum of N d(r_w^3) in sorted order: lane-strided partial sums, xor butterfly
    for (int cl = warp; cl < nc; cl += NW) {
      const int b0 = (int)segl[cl], b1 = (int)segl[cl + 1];
      double acc = 0.0;
      for (int e = b0 + lane; e < b1; e += 32) acc += s_con[e];
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
      if (lane == 0) s_sum[cl] = acc;
    }
    __syncthreads();
  }

  if (tid < nc) {
    if (M > 0) {   // feedback of the last substep
      const double drv = fbk * s_sum[tid];
      th += drv * (-th * lv / (cst::c_pd * T));
      rv += drv;
    }
    th_f.at(ci, cj, ck) = th;
    rv_f.at(ci, cj, ck) = rv;
    // air properties after the feedback, used by coalescence and sedimentation (v_term)
    const double Tn = pow(th * c_exn, cst::c_pd / (cst::c_pd - cst::R_d));
    cf.eta[c_first + tid] = eta_air(Tn);
    cf.rho_a[c_first + tid] = rhod * (1.0 + rv);
  }
  for (int t = tid; t < M; t += T3) {
    int lo = 0, hi = nc;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)t) lo = mid; else hi = mid; }
    const u32 s = s0 + t;
    const double r = s_r[(int)segl[lo] + rank[s]];
    a.rw2[s] = r * r;
  }
  unsigned v0 = n_ill, v1 = n_eval, v2 = n_sub, v3 = n_slow;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    v0 += __shfl_xor_sync(0xffffffffu, v0, d);
    v1 += __shfl_xor_sync(0xffffffffu, v1, d);
    v2 += __shfl_xor_sync(0xffffffffu, v2, d);
    v3 += __shfl_xor_sync(0xffffffffu, v3, d);
  }
  if (lane == 0) {
    const int slot = (blockIdx.x * NW + warp) & (NSLOT - 1);
    if (v0) atomicAdd(&cnt.ill_posed[slot], (unsigned long long)v0);
    if (v1) atomicAdd(&cnt.f_evals[slot], (unsigned long long)v1);
    if (v2) atomicAdd(&cnt.sd_substeps[slot], (unsigned long long)v2);
    if (v3) atomicAdd(&cnt.cond_slow[slot], (unsigned long long)v3);
  }
}

// eta, rho_a per cell when condensation is switched off
__global__ void k_thermo(Grid g, Field th_f, Field rv_f, CellFields cf) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.ncell) return;
  const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
  const double th = th_f.at(i, j, k), rv = rv_f.at(i, j, k), rhod = cf.rhod[c];
  const double T = T_of(th, rhod);
  cf.eta[c] = eta_air(T);
  cf.rho_a[c] = rhod * (1.0 + rv);
}

// cpb cells per CTA; cap > 0: shared-memory slots per CTA (>= the most populated tile); cap == 0: GMEM
// variant (cpb must be 1), `alt` = the idle ping-pong copy of the state used as scratch.
cudaError_t launch_cond(int cpb, int cap, const SdArrays& a, const SdArrays& alt, const u16* rank, const u32* seg,
                        const Grid& g, Field th, Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt,
                        cudaStream_t st) {
  const int grid = (g.ncell + cpb - 1) / cpb;
  if (cap > 0) {
    const size_t smem = cond3_smem_bytes(cpb, cap);
    cudaError_t e = cudaFuncSetAttribute(k_cond3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_cond3<<<grid, T3, smem, st>>>(a, rank, seg, g, th, rv, cf, cp, cnt, cpb, cap, c3_lstride(cap));
  } else {
    const size_t smem = cond_smem_bytes(cpb, 0);
    k_cond<false><<<grid, COND_THREADS, smem, st>>>(a, alt, rank, seg, g, th, rv, cf, cp, cnt, cpb, 0);
  }
  return cudaGetLastError();
}

void launch_thermo(const Grid& g, Field th, Field rv, const CellFields& cf, cudaStream_t st) {
  k_thermo<<<(g.ncell + 127) / 128, 128, 0, st>>>(g, th, rv, cf);
}

}  // namespace sdm
