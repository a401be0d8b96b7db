// Stage a4: condensational growth (eq. 17-26), all sstp_cond substeps fused in one
// tile-resident kernel.  Kernels of this file:
//   k_cond4   the fp64 kernel of the step: a CTA of 128 threads owns a tile of ~10 consecutive cells (<= 800 SDs, 5 CTAs per
//             SM; 256 / 1280 and 512 / 4096 variants for crowded cells); r_w, r_d^3, kappa r_d^3, N of the tile stay in shared
//             memory in sorted order for all substeps.  Per substep: (D) 8-lane groups sum N d(r_w^3) of the cells in a fixed
//             order; (A) one lane per cell on the first warp applies the feedback (eq. 25-26) and advances T, p_vs .. by short
//             series; (B) the warps sweep the tile's SDs in 32-SD chunks and solve eq. 17 by a Newton iteration in r = sqrt(y)
//             bracketed by eq. 18-19 (the paper bisects, :579, and names a faster root finder as the first optimisation, :912);
//             (C) whatever is irregular - an iterate leaving the bracket, a bracket that may hold several roots, a Kelvin
//             exponent out of range - was put on a list and is solved by cond_solve (bracketed Newton / bisection state
//             machine) or by the paper's literal bisection, which hands over to Newton once its bracket holds one root.
//             With cp.adapt_tol > 0 every cell takes its own number of substeps (reading R-adapt).
//   k_cond4f  the same design with the sweep in fp32 arithmetic for the fp32 state (sdm_set_cond_arith 4).
//   k_cond    one crowded cell (beyond 4096 SDs) per CTA, in place in global memory, cond_solve only.
//   k_thermo  eta, rho_a per cell when condensation is switched off.
// fp64 throughout unless stated; k_cond4 is bound by latency in front of the fp64 pipe.
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
  double c0Dc;        // c0 * D_0 Sh/2 (bounds c0 D_eff in single_root_bracket)
  double cDK;         // c0 * Dc * Kc
};

// Growth rate f(y) = d r_w^2/dt (eq. 20-24) and df/dy at y = r_w^2, written with one reciprocal:
//   beta_M = N_M/D_M, beta_T = N_T/D_T (Fuchs-Sutugin multiplied through by r^2),
//   D_eff = Dc Kc N_M N_T / Q,  Q = Kc N_T D_M + heat Dc N_M D_T,
//   a_w = P/W, P = r^3 - r_d^3, W = P + kappa r_d^3,  f = c0 D_eff (RH - a_w exp(A/r)).
__device__ __forceinline__ void growth_fd(double y, const SdK& s, const CellK& c, double& f, double& df, double& cDN_out) {
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
  const double cDN = cD * NN;   // c0 D_eff(y)
  cDN_out = cDN;
  f = cDN * S;
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
__device__ __forceinline__ void growth_fd(double y, const SdK& s, const CellK& c, double& f, double& df) {
  double cDN;
  growth_fd(y, s, c, f, df, cDN);
}

// ---- fast path (k_cond4): the same equations written in r = sqrt(y), which stays resident in shared
// memory over the substeps (no sqrt per substep), with one reciprocal per evaluation.
// fp64 literals cost two UMOV/MOV issue slots each on sm_100 (64-bit immediates do not exist), which in
// a polynomial doubles the instruction count; constants that the hot loop needs therefore live in
// constant memory, where one LDCU.128 fetches two of them into uniform registers.
enum {
  KC_LOG2E = 0, KC_MAGIC, KC_LN2_HI, KC_LN2_LO,   // exp: range reduction
  KC_E13, KC_E12, KC_E11, KC_E10, KC_E9, KC_E8, KC_E7, KC_E6, KC_E5, KC_E4, KC_E3, KC_E2,   // 1/n!
  KC_TOL, KC_TOL400, KC_EPSW, KC_D0, KC_HALF_D0, KC_K0, KC_HALF_K0, KC_171,
  KC_D2Q, KC_B1, KC_B2, KC_B3, KC_B4, KC_B5,   // delta0^2/4; binomial series of (1+x)^(1/3) - 1
  KC_N
};
#ifndef SDM_COND_TOL
#define SDM_COND_TOL 1e-11   // bound on the relative error left in r by a Newton step of the sweep
#endif
#ifndef SDM_COND_TOL1
#define SDM_COND_TOL1 (1e-11 / 400.0)   // the same for the first step, whose curvature is bounded, not estimated
#endif
__constant__ double KC[KC_N] = {
    1.4426950408889634074, 6755399441055744.0 /* 1.5 * 2^52 */, 6.93147180369123816490e-01, 1.90821492927058770002e-10,
    1.0 / 6227020800.0, 1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0, 1.0 / 362880.0, 1.0 / 40320.0, 1.0 / 5040.0,
    1.0 / 720.0, 1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0, 0.5,
    SDM_COND_TOL, SDM_COND_TOL1, 1e-15, cst::D_0, 0.5 * cst::D_0, cst::K_0, 0.5 * cst::K_0, 1.71,
    cst::kc_delta0 * cst::kc_delta0 / 4.0, 1.0 / 3.0, -1.0 / 9.0, 5.0 / 81.0, -10.0 / 243.0, 22.0 / 729.0};

// exp(t) for 0 <= t < 8 (t = A/r, the Kelvin exponent): n = rint(t log2 e) by the 1.5*2^52 trick,
// s = t - n ln 2 in two parts (|s| <= 0.347), Taylor polynomial of degree 13 (remainder
// 0.347^14/14! = 4e-18), result scaled by 2^n through the exponent field.  No overflow, underflow
// or NaN handling: the caller keeps t in range and sends everything else to cond_solve.
__device__ __forceinline__ double exp_kelvin(double t) {
  const double z = fma(t, KC[KC_LOG2E], KC[KC_MAGIC]);
  const int n = __double2loint(z);
  const double fn = z - KC[KC_MAGIC];
  double s = fma(-fn, KC[KC_LN2_HI], t);
  s = fma(-fn, KC[KC_LN2_LO], s);
  // even and odd part as two Horner chains in s^2 (same 14 operations as one chain of 13, half the depth:
  // a dependent DFMA issues every ~9 cycles on sm_100; measured)
  const double s2 = s * s;
  double pe = KC[KC_E12], po = KC[KC_E13];
  pe = fma(pe, s2, KC[KC_E10]); po = fma(po, s2, KC[KC_E11]);
  pe = fma(pe, s2, KC[KC_E8]); po = fma(po, s2, KC[KC_E9]);
  pe = fma(pe, s2, KC[KC_E6]); po = fma(po, s2, KC[KC_E7]);
  pe = fma(pe, s2, KC[KC_E4]); po = fma(po, s2, KC[KC_E5]);
  pe = fma(pe, s2, KC[KC_E2]); po = fma(po, s2, KC[KC_E3]);
  pe = fma(pe, s2, 1.0); po = fma(po, s2, 1.0);
  const double p = fma(po, s, pe);
  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));
}

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
};

// f(r) = d r_w^2/dt (eq. 20-24) and df/dr; also returns y = r^2 and t = A/r.  Notation as growth_fd.
__device__ __forceinline__ void growth_r(double r, const SdK& s, const CellR& c, double& y, double& f, double& dfr,
                                         double& t_out) {
  y = r * r;
  const double lDr = c.lD * r, lKr = c.lK * r;
  const double NM = y + lDr, DM = fma(KC[KC_171], lDr, y) + c.qD;
  const double NT = y + lKr, DT = fma(KC[KC_171], lKr, y) + c.qK;
  const double KN = s.Kc * NT, HN = s.hDc * NM;
  const double Q = fma(KN, DM, HN * DT);
  const double r3 = y * r;
  const double P = r3 - s.rd3, W = P + s.krd3;
  // two reciprocals, 1/r and 1/(Q W), instead of one of r Q W: the Kelvin exponent and its exp then depend on r alone and run
  // beside the chain that leads to Q (the kernel is bound by dependent-instruction latency)
  const double invr = rcp_nr<2>(r);
  const double t = c.A * invr;
  t_out = t;
  const double ex = exp_kelvin(t);
  const double inv = rcp_nr<2>(Q * W);
  const double invQ = inv * W, invW = inv * Q;
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

// max / min without the NaN handling of fmax / fmin (DSETP + 2 SEL instead of DSETP + 2 FSEL + LOP3 + moves); the
// sweep sends anything that is not a finite, ordered bracket to the slow list anyway
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }

// sqrt(a) and 1/a from the fp32 hardware seeds and ONE fp64 Newton step (relative error ~1e-14, which is
// ample for the ventilation coefficients: they enter D and K through 1 + (Sh-2)/2)
__device__ __forceinline__ double sqrt_seeded(double a) {
  const float af = (float)a;
  const float is = rsqrtf(af);
  const double s = (double)(af * is);
  return fma(fma(-s, s, a), (double)(0.5f * is), s);
}
__device__ __forceinline__ double rcp_seeded(double a) {
  float xf;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(xf) : "f"((float)a));   // MUFU.RCP, 1 ulp: one instruction where __frcp_rn takes eight
  const double x = (double)xf;
  return fma(fma(-a, x, 1.0), x, x);
}

// (1 + x)^(1/3) - 1 for x >= 0.02 from the fp32 cube root and one fp64 Newton step (relative error ~1e-14)
__device__ __forceinline__ double cbrt1pm1_seeded(double x) {
  const double w = 1.0 + x;
  const double c = (double)cbrtf((float)w);
  const double c2 = c * c;
  return (c - 1.0) - fma(c2, c, -w) * rcp_seeded(3.0 * c2);
}

// [L] ventilation at the substep's starting radius r0 (reading R-vent) -> per-SD constants.
// Re from the terminal velocity of Khvorostyanov & Curry 2002: e = c1 sqrt(X) = kE r^(3/2),
// Re = (delta0^2/4) (sqrt(1+e) - 1)^2.  fp64 throughout, with roots and reciprocals from fp32 seeds and one
// Newton step (~1e-14).  Up to Re Sc = 0.02 (r ~ 20 um) the binomial series of (1+x)^(1/3) - 1 to x^5 (next
// term 2e-10 of the first); beyond, the seeded cube root; Re > 1 (drizzle and rain) takes the library pow.
// Haze and small droplets (e < 0.01, r below ~3 um) take a short cut that needs no fp64 root: with q = sqrt(1+e) - 1,
// q^2 = (e^2/4)(1 - e/2 + 5 e^2/16 - 7 e^3/32 + O(e^4)), e^2 = kE^2 r^3 exactly and e itself only inside the bracket (an fp32 root
// is ample there: the bracket differs from 1 by < 5e-3); Re Sc < 4e-4 then, so three terms of the binomial series suffice.
// Error of D_0 Sh/2: < 1e-13 relative.
__device__ __forceinline__ void sd_setup(double r0, double c0, double heat, double kE, double Sc, double Pr, SdK& s) {
  const double e2 = (kE * kE) * (r0 * (r0 * r0));
  double shm, num;   // Sh - 2, Nu - 2
  if (e2 < 1e-4) {
    float ef;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(ef) : "f"((float)e2));
    const float corr = fmaf(ef, fmaf(ef, fmaf(ef, -0.21875f, 0.3125f), -0.5f), 1.0f);
    const double Re = (0.25 * KC[KC_D2Q]) * (e2 * (double)corr);
    const double xs = Re * Sc, xp = Re * Pr;
    shm = xs * fma(xs, fma(xs, KC[KC_B3], KC[KC_B2]), KC[KC_B1]);
    num = xp * fma(xp, fma(xp, KC[KC_B3], KC[KC_B2]), KC[KC_B1]);
    const double Dc = fma(KC[KC_HALF_D0], shm, KC[KC_D0]);
    s.Kc = fma(KC[KC_HALF_K0], num, KC[KC_K0]);
    s.hDc = heat * Dc;
    s.c0Dc = c0 * Dc;
    s.cDK = s.c0Dc * s.Kc;
    return;
  }
  const double e = kE * (r0 * sqrt_seeded(r0));
  const double q = e * rcp_seeded(sqrt_seeded(1.0 + e) + 1.0);   // sqrt(1+e) - 1 without cancellation
  const double Re = KC[KC_D2Q] * (q * q);
  const double xs = Re * Sc, xp = Re * Pr;
  if (dmax(xs, xp) < 0.02) {
    double a = KC[KC_B5], b = KC[KC_B5];
    a = fma(a, xs, KC[KC_B4]); b = fma(b, xp, KC[KC_B4]);
    a = fma(a, xs, KC[KC_B3]); b = fma(b, xp, KC[KC_B3]);
    a = fma(a, xs, KC[KC_B2]); b = fma(b, xp, KC[KC_B2]);
    a = fma(a, xs, KC[KC_B1]); b = fma(b, xp, KC[KC_B1]);
    shm = a * xs; num = b * xp;
  } else {
    shm = cbrt1pm1_seeded(xs); num = cbrt1pm1_seeded(xp);
    if (Re > 1.0) {   // (1 + c)(1 + m) - 1, m = Re^0.077 - 1
      const double m = pow(Re, 0.077) - 1.0;
      shm = shm + m + shm * m;
      num = num + m + num * m;
    }
  }
  const double Dc = fma(KC[KC_HALF_D0], shm, KC[KC_D0]);   // eq. 23 without beta_M: D_0 Sh / 2
  s.Kc = fma(KC[KC_HALF_K0], num, KC[KC_K0]);              // eq. 24 without beta_T: K_0 Nu / 2
  s.hDc = heat * Dc;
  s.c0Dc = c0 * Dc;
  s.cDK = s.c0Dc * s.Kc;
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
// Root selection.  eq. 17 can have SEVERAL roots inside the bracket of eq. 18-19 (a haze particle far from
// equilibrium in supersaturated air: the implicit-Euler haze root, one at the unstable Koehler equilibrium and an
// "activated" one), or two, in which case the paper's rule (:579) calls the bracket ill-posed.  The paper's
// bisection then defines the result, and a Newton iteration started at y0 would land elsewhere.  Newton is
// therefore used only where the bracket [lo, hi] provably or structurally holds at most one root:
//  (1) it lies on the solute-dominated side of the Koehler curve, hi <= y_c = 3 kappa r_d^3 / A (for
//      kappa <= 2 the activity term then outweighs the Kelvin term everywhere in it: a_w e^(A/r) rises with r, f
//      has one zero and g = y - y0 - dt' f one sign change), or
//  (2) it is narrow, hi - lo <= lo/2, and from max(lo, y_c) on the Kelvin term is too weak to bend g back:
//      dt' c0 D 1.3 A / (2 r^3) <= 1/2 and e^(A/r) <= 1.3, or
//  (3) the particle grows (lo = y0) in subsaturated air: a_w e^(A/r) = RH < 1 has one solution y_eq, on the
//      rising side of the Koehler curve, f > 0 below it and f < 0 above, so g > 0 from y_eq on and changes sign
//      once between y0 and y_eq (haze catching up with a moister cell: by far the most frequent wide bracket), or
//  (4) the particle evaporates (f(y0) < 0, hi = y0) and the Kelvin term is as weak as in (2), however wide the bracket.
//      A root below y0 needs f < 0 there (g = y - y0 - dt' f), i.e. S = RH - a_w e^(A/r) < 0, and the set S < 0 is an
//      interval that holds y0 (the Koehler curve a_w e^(A/r) rises to r_c, then falls towards 1).  On it D_eff' S <= 0
//      (D_eff rises with r), so g' >= 1 - dt' c0 D_eff S', and S' > 0 only on the falling branch y >= y_c, where
//      S' <= e^(A/r) A / (2 r^3): with e^(A/r) <= 1.3 and r^3 >= ym^(3/2), g' >= 1 - K3 / (2 ym^(3/2)) > 0: g rises
//      through the whole set, one root at most (a droplet of ~1 um shrinking by 10 % per substep under cloud base: its
//      bracket [0.6 y0, y0] is too wide for (2), and the literal bisection took 36 to 315 evaluations for it).
//      Below y0, c0 D_eff(y) <= c0 D_eff(y0), which the evaluation at y0 has as f / S: dtcDe = dt' c0 D_eff(y0) takes
//      the place of dtcD in this rule (a third of it at 0.5 um), and the rule asks for g' > 0 only:
//      K3 / (2 ym^(3/2)) <= 0.92.  Applied on the slow list only (RULE4; its SDs then need one round of the warp
//      bisection and ~3 Newton evaluations): in the sweeps every instruction of this test is paid by every SD-substep,
//      and the two it takes there cost the 67M-SD step 0.8 % while its list is 5e-5 of the SD-substeps either way
//      (profiles/r2_k_cond4_ncu_full.md).
// Everything else is solved by the paper's own procedure, literally (bisect_paper).  dtcD = dt' c0 D_0 Sh/2.
template <bool RULE4 = true>
__device__ __forceinline__ bool single_root_bracket(double lo, double hi, double y0, double RH, double rd3, double krd3, double A,
                                                    double invA, double dtcD, double dtcDe) {
  const double yc = 3.0 * krd3 * invA;
  if ((hi <= yc && krd3 <= 2.0 * rd3) || (RH < 1.0 && lo == y0)) return true;   // (1), (3)
  const double ym = dmax(lo, yc);
  const bool evap = RULE4 && hi <= y0;   // a bracket below y0: only an evaporating particle has one (a growing one has lo = y0 < hi)
  const double K3 = 1.3 * A * (evap ? dtcDe : dtcD);
  const double K32 = evap ? 0.3 * (K3 * K3) : K3 * K3;
  return (evap || hi - lo <= 0.5 * lo) && (ym * ym * ym >= K32) && (A * A <= 0.0625 * ym);   // (4), (2)
}

// per-SD constants of one substep in plain fp64 (cond_solve and the literal bisection)
__device__ __forceinline__ void slow_setup(double y0, double rd3, double krd3, const CellK& c, SdK& s, double& Dc) {
  s.rd3 = rd3; s.krd3 = krd3;
  // [L] ventilation at the substep's starting radius (reading R-vent); Re from the terminal
  // velocity of Khvorostyanov & Curry 2002: e = c1 sqrt(X) = kE r^(3/2)
  const double r0 = sqrt(y0);
  const double e = c.kE * (r0 * sqrt(r0));
  const double q = e / (sqrt(1.0 + e) + 1.0);
  const double Re = (cst::kc_delta0 * cst::kc_delta0 / 4.0) * (q * q);
  Dc = cst::D_0 * vent(Re, c.Sc) * 0.5;     // eq. 23 without beta_M
  s.Kc = cst::K_0 * vent(Re, c.Pr) * 0.5;   // eq. 24 without beta_T
  s.hDc = c.heat * Dc;
  s.c0Dc = c.c0 * Dc;
  s.cDK = s.c0Dc * s.Kc;
}

// Root of g(y) = y - y0 - dt' f(y) in a bracket [a, b] with g(a) g(b) < 0 that holds exactly one root (single_root_bracket):
// Newton steps kept inside the shrinking bracket, bisection where a step leaves it.  ga_pos: g(a) > 0.  The literal
// bisection of the paper's procedure hands over to this as soon as its bracket is certified: what it would go on to
// compute is this root to 1e-15 b, 40 evaluations later.
__device__ __forceinline__ double newton_in_bracket(double a, double b, bool ga_pos, double y0, const SdK& s, const CellK& c, double dtp,
                                                    unsigned& n_eval) {
  double y = 0.5 * (a + b);
  for (int it = 0; it < 100; ++it) {
    double f, df;
    growth_fd(y, s, c, f, df);
    ++n_eval;
    const double g = y - y0 - dtp * f, gp = fma(-dtp, df, 1.0);
    if (g == 0.0) return y;
    if ((g > 0.0) == ga_pos) a = y; else b = y;
    double yn = y - g / gp;
    const bool newton = yn > a && yn < b;
    if (!newton) yn = 0.5 * (a + b);
    const double d = fabs(yn - y);
    y = yn;
    // a Newton step of size d leaves ~d^2 |g''/2g'| <= d^2 (100/y): stop below 1e-13 y; a bisection step bounds the error directly
    if (newton ? (100.0 * d * d <= 1e-13 * (y * y)) : (d <= 2e-16 * y)) return y;
    if (!(b - a > 1e-15 * b)) return 0.5 * (a + b);
  }
  return y;
}

// The paper's procedure (:573-579) for one SD by a whole WARP: signs of g at both ends, (a+b)/2 if they agree,
// else bisection - five levels per round: lane l = 1..31 is node l of the binary tree of midpoints below the
// current interval (heap order), computes its midpoint with the very operations the serial bisection would use on
// the way there, evaluates g, and the ballot of the signs lets every lane walk the five levels.  Same result
// as the serial loop of the oracle, a fifth of its latency.  All lanes pass the same arguments.
__device__ __forceinline__ double bisect_paper_warp(double a, double b, double f0, double y0, const SdK& s, const CellK& c,
                                                    double dtp, int lane, unsigned& n_ill, unsigned& n_eval, double rd3, double krd3,
                                                    double invA, double dtcD, double dtcDe) {
  double f, df;
  double ga, gb;
  if (a == y0) ga = -dtp * f0; else { growth_fd(a, s, c, f, df); n_eval += (lane == 0); ga = a - y0 - dtp * f; }
  if (b == y0) gb = -dtp * f0; else { growth_fd(b, s, c, f, df); n_eval += (lane == 0); gb = b - y0 - dtp * f; }
  if (ga == 0.0) return a;
  if (gb == 0.0) return b;
  if ((ga > 0.0) == (gb > 0.0)) { n_ill += (lane == 0 && b - a > 1e-9 * b); return 0.5 * (a + b); }
  const bool ga_pos = ga > 0.0;
  const int depth = 31 - __clz(max(lane, 1));   // level of this lane's node (root = 0)
  for (;;) {
    // this lane's node: follow the bits of `lane` below its leading one from the current interval
    double lo = a, hi = b;
    bool alive = lane >= 1;
    for (int j = depth - 1; j >= 0 && alive; --j) {
      if (!(hi - lo > 1e-15 * hi)) { alive = false; break; }
      const double m = 0.5 * (lo + hi);
      if (m <= lo || m >= hi) { alive = false; break; }
      if ((lane >> j) & 1) lo = m; else hi = m;
    }
    double m = 0.5 * (lo + hi);
    alive = alive && (hi - lo > 1e-15 * hi) && m > lo && m < hi;
    double gm = 1.0;
    if (alive) { growth_fd(m, s, c, f, df); ++n_eval; gm = m - y0 - dtp * f; }
    const unsigned right = __ballot_sync(0xffffffffu, alive && ((gm > 0.0) == ga_pos));
    const unsigned zero = __ballot_sync(0xffffffffu, alive && gm == 0.0);
    // walk five levels with the signs
    int node = 1;
    bool done = false;
    for (int lev = 0; lev < 5; ++lev) {
      if (!(b - a > 1e-15 * b)) { done = true; break; }
      const double mm = 0.5 * (a + b);
      if (mm <= a || mm >= b) { done = true; break; }
      if ((zero >> node) & 1u) return mm;
      if ((right >> node) & 1u) { a = mm; node = 2 * node + 1; } else { b = mm; node = 2 * node; }
    }
    if (done) break;
    // five levels narrower: once the bracket provably holds one root, Newton finishes (the same on every lane)
    if (single_root_bracket(a, b, y0, c.RH, rd3, krd3, c.A, invA, dtcD, dtcDe)) {
      unsigned ev = 0;
      const double y = newton_in_bracket(a, b, ga_pos, y0, s, c, dtp, ev);
      n_eval += (lane == 0) ? ev : 0u;
      return y;
    }
  }
  return 0.5 * (a + b);
}

enum { M_FIRST = 0, M_MAIN = 1, M_CHK_A = 2, M_CHK_B = 3 };

__device__ __forceinline__ bool cond_solve(double y0, double rd2, double rd3, double krd3, const CellK& c, double dtp,
                                           int max_evals, double& y_out, unsigned& n_ill, unsigned& n_eval) {
  SdK s;
  double Dc;
  slow_setup(y0, rd3, krd3, c, s, Dc);
  int mode = M_FIRST;
  double yE = y0, y = y0, g = 0.0, gp = 1.0, a = 0.0, b = 0.0, lo = 0.0, hi = 0.0, dprev = 0.0, dtcDe = 0.0;
  bool lo_unv = false, hi_unv = false;
  for (int it = 0; it < max_evals; ++it) {
    double f, df, cDN;
    growth_fd(yE, s, c, f, df, cDN);   // the only evaluation site
    ++n_eval;
    bool bisect = false;
    if (mode == M_FIRST) {
      const double two = 2.0 * dtp * f;
      a = fmax(rd2, y0 + fmin(two, 0.0));   // eq. 18
      b = y0 + fmax(two, 0.0);              // eq. 19
      if (!(a < b)) { y_out = a; return true; }
      dtcDe = dtp * cDN;                    // dt' c0 D_eff(y0): rule (4) of single_root_bracket
      if (!single_root_bracket(a, b, y0, c.RH, rd3, krd3, c.A, 1.0 / c.A, dtp * c.c0 * Dc, dtcDe)) {
        // the paper's procedure, literally (:573-579): signs at both ends, (a+b)/2 if they agree, else bisection
        if (max_evals < 100) return false;   // not in a budgeted sweep: leave it to the pass that may finish
        const double f0 = f;
        double ga, gb;
        if (a == y0) ga = -dtp * f0; else { growth_fd(a, s, c, f, df); ++n_eval; ga = a - y0 - dtp * f; }
        if (b == y0) gb = -dtp * f0; else { growth_fd(b, s, c, f, df); ++n_eval; gb = b - y0 - dtp * f; }
        if (ga == 0.0) { y_out = a; return true; }
        if (gb == 0.0) { y_out = b; return true; }
        if ((ga > 0.0) == (gb > 0.0)) { n_ill += (b - a > 1e-9 * b); y_out = 0.5 * (a + b); return true; }
        int level = 0;
        while (b - a > 1e-15 * b) {
          const double m = 0.5 * (a + b);
          if (m <= a || m >= b) break;
          growth_fd(m, s, c, f, df);
          ++n_eval;
          const double gm = m - y0 - dtp * f;
          if (gm == 0.0) { y_out = m; return true; }
          if ((gm > 0.0) == (ga > 0.0)) { a = m; ga = gm; } else { b = m; gb = gm; }
          if (++level % 5 == 0 && single_root_bracket(a, b, y0, c.RH, rd3, krd3, c.A, 1.0 / c.A, dtp * c.c0 * Dc, dtcDe)) {
            y_out = newton_in_bracket(a, b, ga > 0.0, y0, s, c, dtp, n_eval);   // one root left in the bracket: Newton finishes
            return true;
          }
        }
        y_out = 0.5 * (a + b);
        return true;
      }
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
      const double tol = SDM_COND_TOL * y;
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
// order, contributions go to alt.n (8 bytes per SD, used as doubles) in sorted order, the list to alt.id.
size_t cond_smem_bytes(int cpb, int cap) {
  return (size_t)(CELLK_N + 1) * cpb * 8 + (size_t)6 * cap * 8 + (size_t)(cpb + 2) * 4 + (size_t)cap * 4 + 16;
}

template <bool SMEM, typename R>
__global__ void __launch_bounds__(COND_THREADS, 2)
k_cond(SdArraysT<R> a, SdArraysT<R> alt, const u16* __restrict__ rank, const u32* __restrict__ seg, Grid g, Field th_f, Field rv_f,
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
  if constexpr (!SMEM) s_con = reinterpret_cast<double*>(alt.n) + s0;

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
  int nsub = cp.sstp;
  double dtp = cp.dtp;
  if (cp.adapt_tol > 0.0 && M > 0 && cpb == 1) {   // R-adapt (see k_cond4): the cell's number of substeps in this step
    __shared__ double s_red[COND_WARPS];
    __shared__ int s_nsub;
    if (tid == 0) {
      CellK c;
      cell_consts(th, rv, rhod, c_exn, cp.RH_max, c, T, lv);
      s_cell[0] = c.RH; s_cell[1] = c.A; s_cell[2] = c.c0; s_cell[3] = c.lD; s_cell[4] = c.lK; s_cell[5] = c.heat;
      s_cell[6] = c.kE; s_cell[7] = c.Sc; s_cell[8] = c.Pr;
    }
    __syncthreads();
    CellK c;
    c.RH = s_cell[0]; c.A = s_cell[1]; c.c0 = s_cell[2]; c.lD = s_cell[3]; c.lK = s_cell[4]; c.heat = s_cell[5];
    c.kE = s_cell[6]; c.Sc = s_cell[7]; c.Pr = s_cell[8];
    const double dt_full = cp.dtp * cp.sstp;
    double acc = 0.0;
    for (int t = tid; t < M; t += COND_THREADS) {
      double y0, rd3, krd3, dn;
      if constexpr (SMEM) { y0 = s_y[t]; rd3 = s_rd3[t]; krd3 = s_krd3[t]; dn = s_dn[t]; }
      else { const u32 sl = s0 + t; y0 = a.rw2[sl]; rd3 = a.rd3[sl]; krd3 = a.kappa[sl] * rd3; dn = (double)a.n[sl]; }
      SdK sk;
      double Dc, f, df;
      slow_setup(y0, rd3, krd3, c, sk, Dc);
      growth_fd(y0, sk, c, f, df);
      acc += dn * (1.5 * sqrt(y0) * (dt_full * f));
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if (lane == 0) s_red[warp] = acc;
    __syncthreads();
    if (tid == 0) {
      double est = 0.0;
      for (int w = 0; w < COND_WARPS; ++w) est += s_red[w];
      const double eps = fabs(fbk * est) / (rv * fmax(fabs(c.RH - 1.0), 1e-3));
      const double want = cp.sstp * eps / cp.adapt_tol;
      int d = cp.sstp;
      for (int k = cp.sstp - 1; k >= 1; --k)
        if (cp.sstp % k == 0 && (double)k >= want) d = k;
      s_nsub = d;
    }
    __syncthreads();
    nsub = s_nsub;
    dtp = dt_full / nsub;
  }
  for (int sub = 0; sub < nsub && M > 0; ++sub) {
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
          done = cond_solve(y0, rd2, rd3, krd3, c, dtp, max_evals, y1, ill, n_eval);
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

// ---- k_cond4: the shared-memory tile kernel ----------------------------------------------------------
// A CTA of T threads owns a tile of `cpb` consecutive cells holding at most CAP super-droplets.
//  * r_w (not r_w^2) is resident in shared memory: no sqrt per substep, N d(r_w^3) by two products;
//  * the sweep is straight-line code around growth_r with a warp-uniform iteration loop; anything
//    irregular (Newton leaving the bracket of eq. 18-19, an end to verify, slow convergence, a Kelvin
//    exponent out of range, a bracket that may hold several roots) is put on a list and solved afterwards by
//    cond_solve, the robust state machine;
//  * warps take 32-SD chunks of the tile from a shared counter, so a warp that met slow SDs does not
//    hold the others at the barrier;
//  * CAP is a compile-time constant, so every shared array sits at a fixed offset from one index
//    register, and the per-cell constants are one record per cell fetched with LDS.128;
//  * the state of a cell (theta, r_v, T, p_vs ..) lives in that record between substeps, not in
//    registers, and is advanced INCREMENTALLY: the feedback of eq. 25-26 changes theta by a relative
//    d ~ 1e-5 per substep, so T (eq. 43) and p_vs follow from short series in d instead of pow, exp
//    and log; each warp sums and advances the cells it owns, which takes the serial chain from ~560
//    instructions on one warp (with three waiting at a barrier) to ~150 on all of them;
//  * small CTAs (128 threads, 5 per SM) so that the serial phases of one tile overlap the sweeps of
//    the others; a 512-thread variant with CAP 4096 serves cells of hundreds to thousands of SDs.
// Shared memory: double sd[6][CAP] = r, r_d^3, kappa r_d^3, N, r_d^2, N d(r_w^3); u16 cidx[CAP];
// u16 list[CAP]; CellRec cell[cpb]; u32 segl[cpb + 1]; u32 ctr[2].
struct __align__(16) CellRec {
  double RH, A, lD, lK, qD, qK, lD171, lK171;   // fast path (CellR)
  double c0, heat, kE, Sc, Pr;                  // cond_solve and the per-SD set-up
  double eta;                                   // [L] viscosity, for the cell fields written at the end
  double th, rv, rhod, fbk;                     // theta, r_v (advanced every substep), rho_d, eq. 25 prefactor
  double T, invT, lv, pvs;                      // eq. 43, Table 2, [L] Clausius-Clapeyron
  double invA, pad;
  double dtp;                                   // dt' of the cell in the current substep; 0: the cell sits this substep out (R-adapt)
  double stride;                                // the cell takes every stride-th of the sstp_cond substeps (1 without R-adapt)
};
static_assert(sizeof(CellRec) == 208, "CellRec");

// everything the substep needs from (T, 1/T, p_vs, r_v, rho_d); square roots and reciprocals from fp32
// seeds (sqrt_seeded, rcp_nr: relative error < 1e-14, they feed correction factors and RH to 1e-15)
__device__ __forceinline__ void cell_derive(CellRec& R, double RH_max) {
  const double T = R.T, invT = R.invT, rv = R.rv, rhod = R.rhod;
  const double p = rhod * (cst::R_d + rv * cst::R_v) * T;                          // eq. 44
  const double lv = cst::l_v0 + (cst::c_pv - cst::c_l) * (T - cst::T_0);           // Table 2 :1087
  const double rho_vs = R.pvs * invT * (1.0 / cst::R_v);
  R.lv = lv;
  R.RH = fmin(rv * rhod * rcp_nr<2>(rho_vs), RH_max);                              // eq. 30, :685
  R.A = (2.0 * cst::sigma_w / (cst::R_v * cst::rho_w)) * invT;                     // Table 2 :1056
  R.invA = (cst::R_v * cst::rho_w / (2.0 * cst::sigma_w)) * T;
  R.c0 = (2.0 / cst::rho_w) * rho_vs;
  const double sqT = sqrt_seeded(T);
  const double lD = (2.0 * cst::D_0 * 0.03291540093383166 /* 1/sqrt(2 R_v) */) * (sqT * invT);   // [L] Fuchs-Sutugin lengths
  const double lK = ((4.0 / 5.0) * cst::K_0 * 0.04173919355648411 /* 1/sqrt(2 R_d) */) * (sqT * rcp_nr<2>(p));
  R.lD = lD; R.lK = lK;
  R.qD = 1.33 * (lD * lD); R.qK = 1.33 * (lK * lK); R.lD171 = 1.71 * lD; R.lK171 = 1.71 * lK;
  const double lvT = lv * invT;
  R.heat = (rho_vs * lvT) * (lvT * (1.0 / cst::R_v) - 1.0);                        // eq. 21
  // eta = 1.72e-5 (393/(T+120)) (T/273)^1.5
  const double eta = (1.72e-5 * 393.0 * 2.2169506691164923e-4 /* 273^-1.5 */) * (T * sqT) * rcp_nr<2>(T + 120.0);
  const double rho_a = rhod * (1.0 + rv);
  const double inv_eta = rcp_nr<2>(eta);
  // e = c1 sqrt(X), X = (32/3) r^3 (rho_w - rho_a) g rho_a / eta^2  ->  e = kE r^(3/2)
  const double c1 = 4.0 / (cst::kc_delta0 * cst::kc_delta0 * 0.5403702434442518 /* sqrt(C0) */);
  R.kE = c1 * sqrt_seeded((32.0 / 3.0 * cst::g) * ((cst::rho_w - rho_a) * rho_a)) * inv_eta;
  R.Sc = eta * rcp_nr<2>(rho_a * cst::D_0);
  R.Pr = eta * (cst::c_pd / cst::K_0);
  R.eta = eta;
}

// first substep: T from eq. 43 and p_vs from the Clausius-Clapeyron integral, as cell_consts
__device__ __forceinline__ void cell_init(CellRec& R, double RH_max) {
  const double c_exn = pow(R.rhod * cst::R_d / cst::p_1000, cst::R_d / cst::c_pd);
  const double T = pow(R.th * c_exn, cst::c_pd / (cst::c_pd - cst::R_d));
  const double ca = (cst::l_v0 + (cst::c_l - cst::c_pv) * cst::T_0) / cst::R_v;
  const double cb = (cst::c_l - cst::c_pv) / cst::R_v;
  R.T = T; R.invT = 1.0 / T;
  R.pvs = cst::p_vs0 * exp(ca * (1.0 / cst::T_0 - 1.0 / T) - cb * log(T / cst::T_0));
  cell_derive(R, RH_max);
}

// Feedback of one substep (eq. 25-26 with the old theta and T, :195) and the new T, p_vs.
// theta' = theta (1 + d), d = -drv l_v/(c_pd T);  T' = T (1+d)^g, g = c_pd/(c_pd - R_d) (eq. 43, rho_d fixed):
// u = g log1p(d) and T'/T - 1 = expm1(u) by their series (|d| <= 1e-3: truncation < 1e-18);
// p_vs'/p_vs = exp(v), v = ca (1/T - 1/T') - cb log(T'/T) = ca expm1(u)/T' - cb u.
// `full` (first substep of a step, or an implausibly large d) recomputes from theta.
__device__ __forceinline__ void cell_advance(CellRec& R, double sum, double RH_max, bool apply) {
  if (apply) {
    const double drv = R.fbk * sum;
    const double d = -drv * R.lv * R.invT * (1.0 / cst::c_pd);
    R.th = fma(R.th, d, R.th);
    R.rv += drv;
    if (fabs(d) > 1e-3) { cell_init(R, RH_max); return; }
    const double l = d * fma(d, fma(d, fma(d, fma(d, 0.2, -0.25), 1.0 / 3.0), -0.5), 1.0);   // log1p(d)
    const double u = (cst::c_pd / (cst::c_pd - cst::R_d)) * l;
    const double em = u * fma(u, fma(u, fma(u, fma(u, 1.0 / 120.0, 1.0 / 24.0), 1.0 / 6.0), 0.5), 1.0);   // expm1(u)
    const double T = fma(R.T, em, R.T);
    const double invT = rcp_nr<2>(T);
    const double ca = (cst::l_v0 + (cst::c_l - cst::c_pv) * cst::T_0) / cst::R_v;
    const double cb = (cst::c_l - cst::c_pv) / cst::R_v;
    const double v = fma(ca * em, invT, -cb * u);
    R.pvs *= exp_kelvin(v);
    R.T = T; R.invT = invT;
  }
  cell_derive(R, RH_max);
}

template <int CAP, int T>
struct Cond4 {
  static constexpr int NW = T / 32;
  static constexpr size_t fixed_bytes = (size_t)6 * CAP * 8 + (size_t)CAP * 2 + (size_t)CAP * 2;
  static size_t smem(int cpb) { return fixed_bytes + (size_t)cpb * sizeof(CellRec) + (size_t)(cpb + 1) * 4 + 16; }
};

// ADAPT: per-cell substep counts (cp.adapt_tol > 0, DESIGN.md R-adapt); the fixed-substep instantiation carries none of it.
// KF: evaluations per SD-substep in the sweep as a compile-time constant (0: cp.kfast, sdm_set_cond_kfast)
template <int CAP, int T, int MINB, typename R, bool ADAPT, int KF = 0>
__global__ void __launch_bounds__(T, MINB)
k_cond4(SdArraysT<R> a, const u16* __restrict__ rank, const u32* __restrict__ seg, Grid g, Field th_f, Field rv_f,
        CellFields cf, CondParams cp, Counters cnt, int cpb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using L = Cond4<CAP, T>;
  constexpr int NW = L::NW;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c_first = blockIdx.x * cpb;
  const int nc = min(cpb, g.ncell - c_first);
  double* s_r = reinterpret_cast<double*>(smem_raw);
  double *s_rd3 = s_r + CAP, *s_krd3 = s_r + 2 * CAP, *s_dn = s_r + 3 * CAP, *s_rd2 = s_r + 4 * CAP, *s_con = s_r + 5 * CAP;
  u16* cidx = reinterpret_cast<u16*>(s_r + 6 * CAP);
  u16* list = cidx + CAP;
  CellRec* s_cell = reinterpret_cast<CellRec*>(smem_raw + L::fixed_bytes);
  u32* segl = reinterpret_cast<u32*>(s_cell + cpb);
  u32* ctr = segl + cpb + 1;   // [0] next chunk of the sweep, [1] length of the slow list
  const u32 s0 = seg[c_first];
  const int M = (int)(seg[c_first + nc] - s0);

  for (int cl = tid; cl < nc; cl += T) {   // thread cl owns cell cl of the tile (cpb <= T)
    const int c = c_first + cl;
    const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
    CellRec& R = s_cell[cl];
    R.th = th_f.at(i, j, k); R.rv = rv_f.at(i, j, k);
    const double rhod = cf.rhod[c];
    R.rhod = rhod;
    R.fbk = -(4.0 * cst::pi * cst::rho_w / 3.0) / (rhod * g.dV);   // eq. 25 prefactor
    segl[cl] = seg[c] - s0;
  }
  if (tid == 0) { segl[nc] = (u32)M; ctr[0] = 0u; ctr[1] = 0u; }
  __syncthreads();
  const bool by_cell = M >= 24 * nc;   // populated cells: a warp stages a cell at a time (no search for the cell of a slot)
  for (int q = by_cell ? warp : tid; q < (by_cell ? nc : M); q += by_cell ? NW : T) {   // stage the tile in sorted order
    int cl, t0, t1;
    if (by_cell) {
      cl = q; t0 = (int)segl[cl] + lane; t1 = (int)segl[cl + 1];
    } else {
      int lo = 0, hi = nc;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)q) lo = mid; else hi = mid; }
      cl = lo; t0 = q; t1 = q + 1;
    }
    const int b0 = (int)segl[cl];
    for (int t = t0; t < t1; t += 32) {
      const u32 s = s0 + t;
      const int e = b0 + rank[s];
      const double rd3 = a.rd3[s];
      // r_d = cbrt(r_d^3) from the fp32 cube root and one fp64 Newton step (1e-14: r_d^2 only bounds eq. 18 from below)
      const double c = (double)cbrtf((float)rd3);
      const double c2 = c * c;
      const double rd = c - fma(c2, c, -rd3) * rcp_seeded(3.0 * c2);
      s_r[e] = sqrt((double)a.rw2[s]);
      s_rd3[e] = rd3;
      s_krd3[e] = a.kappa[s] * rd3;
      s_dn[e] = (double)a.n[s];
      s_rd2[e] = rd * rd;
      cidx[e] = (u16)cl;
    }
  }
  unsigned n_ill = 0, n_eval = 0, n_sub = 0, n_slow = 0;
  const int nsub = M > 0 ? cp.sstp : 0;
  constexpr bool adapt = ADAPT;
  if (ADAPT && M > 0) {
    // R-adapt (PAPER.md :566; oracle: adaptive_substeps): substeps of each cell from the vapour its SDs would take up in one
    // explicit step, eps = |d r_v| / (r_v max(|RH - 1|, 1e-3)); the smallest divisor d of sstp_cond with d >= sstp_cond eps / tol
    __syncthreads();
    if (tid < ((nc + 31) & ~31))
      for (int cl = tid; cl < nc; cl += T) cell_init(s_cell[cl], cp.RH_max);
    __syncthreads();
    const double dt_full = cp.dtp * cp.sstp;
    for (int q0 = warp * 32; q0 < M; q0 += NW * 32) {
      const int e = q0 + lane;
      if (e < M) {
        const CellRec& R = s_cell[(int)cidx[e]];
        const double r0 = s_r[e];
        SdK s;
        s.rd3 = s_rd3[e]; s.krd3 = s_krd3[e];
        CellR c;
        c.RH = R.RH; c.A = R.A; c.lD = R.lD; c.lK = R.lK; c.qD = R.qD; c.qK = R.qK; c.lD171 = R.lD171; c.lK171 = R.lK171;
        sd_setup(r0, R.c0, R.heat, R.kE, R.Sc, R.Pr, s);
        double y0, f, dfr, t;
        growth_r(r0, s, c, y0, f, dfr, t);
        if (!(t < 4.0)) {   // beyond the range of exp_kelvin: the plain evaluation
          CellK ck;
          ck.RH = R.RH; ck.A = R.A; ck.c0 = R.c0; ck.lD = R.lD; ck.lK = R.lK; ck.heat = R.heat; ck.kE = R.kE; ck.Sc = R.Sc; ck.Pr = R.Pr;
          SdK ss;
          double Dc, df;
          slow_setup(y0, s.rd3, s.krd3, ck, ss, Dc);
          growth_fd(y0, ss, ck, f, df);
        }
        s_con[e] = s_dn[e] * (1.5 * r0 * (dt_full * f));
      }
    }
    __syncthreads();
    {
      const int l8 = lane & 7, grp = lane >> 3;
      for (int cl = warp * 4 + grp; cl < ((nc + 3) & ~3); cl += NW * 4) {
        double acc = 0.0;
        if (cl < nc) {
          const int b1 = (int)segl[cl + 1];
          for (int e = (int)segl[cl] + l8; e < b1; e += 8) acc += s_con[e];
        }
        acc += __shfl_xor_sync(0xffffffffu, acc, 4);
        acc += __shfl_xor_sync(0xffffffffu, acc, 2);
        acc += __shfl_xor_sync(0xffffffffu, acc, 1);
        if (cl < nc && l8 == 0) {
          CellRec& R = s_cell[cl];
          const double drv = fabs(R.fbk * acc);
          const double eps = drv / (R.rv * fmax(fabs(R.RH - 1.0), 1e-3));
          const double want = cp.sstp * eps / cp.adapt_tol;
          int d = cp.sstp;
          for (int k = cp.sstp - 1; k >= 1; --k)
            if (cp.sstp % k == 0 && (double)k >= want) d = k;
          R.stride = (double)(cp.sstp / d);
        }
      }
    }
    __syncthreads();
  }
  for (int sub = 0; sub <= nsub; ++sub) {
    // D. per-cell sums of N d(r_w^3): 8 lanes per cell, fixed order (deterministic); R.pad carries the sum.
    // A. feedback (eq. 25-26) and the constants of the next substep, one lane per cell on the FIRST warp(s): the chain
    // is as long for 3 lanes as for 30, and four warps issuing it cost four times the issue and fp64 slots.  The pass
    // after the last substep only applies the feedback.
    if (sub > 0) {
      const int l8 = lane & 7, grp = lane >> 3;
      for (int cl = warp * 4 + grp; cl < ((nc + 3) & ~3); cl += NW * 4) {   // warp-uniform trip count
        double acc = 0.0;
        const bool was_active = cl < nc && (!ADAPT || s_cell[cl].dtp > 0.0);   // the cell took part in the substep just done
        if (was_active) {
          const int b1 = (int)segl[cl + 1];
          for (int e = (int)segl[cl] + l8; e < b1; e += 8) acc += s_con[e];
        }
        acc += __shfl_xor_sync(0xffffffffu, acc, 4);
        acc += __shfl_xor_sync(0xffffffffu, acc, 2);
        acc += __shfl_xor_sync(0xffffffffu, acc, 1);
        if (was_active && l8 == 0) s_cell[cl].pad = acc;
      }
      __syncthreads();
    }
    if (tid < ((nc + 31) & ~31)) {
      for (int cl = tid; cl < nc; cl += T) {
        CellRec& R = s_cell[cl];
        if constexpr (ADAPT) {
          const int stride = (int)R.stride;
          const bool now = sub < nsub && sub % stride == 0;   // the cell takes part in this substep
          if (sub > 0 && (now || sub == nsub)) cell_advance(R, R.pad, cp.RH_max, true);   // the feedback of its last substep is pending
          R.dtp = now ? cp.dtp * stride : 0.0;
        } else {
          if (sub == 0) cell_init(R, cp.RH_max); else cell_advance(R, R.pad, cp.RH_max, true);
        }
      }
    }
    if (tid == 0) { ctr[0] = 0u; ctr[1] = 0u; }
    if (sub == nsub) break;
    __syncthreads();
    // B. dense sweep.  st: 0 = iterating, 1 = solved, 2 = left to cond_solve (list)
    for (int q0 = warp * 32; q0 < M; q0 += NW * 32) {   // static chunks (a shared counter costs an atomic, a shuffle and two S2R per chunk)
      const int e = q0 + lane;
      const int ec = min(e, M - 1);   // lanes past the end of the tile redo its last SD and discard the result
      const CellRec& R = s_cell[(int)cidx[ec]];
      const double dtp = ADAPT ? R.dtp : cp.dtp;
      const bool valid = e < M && (!ADAPT || dtp > 0.0);
      if (ADAPT && !__any_sync(0xffffffffu, valid)) continue;   // every cell of the chunk sits this substep out
      const double r0 = s_r[ec];
      const double rd2 = s_rd2[ec];
      SdK s;
      s.rd3 = s_rd3[ec];
      s.krd3 = s_krd3[ec];
      CellR c;
      c.RH = R.RH; c.A = R.A; c.lD = R.lD; c.lK = R.lK; c.qD = R.qD; c.qK = R.qK; c.lD171 = R.lD171; c.lK171 = R.lK171;
      sd_setup(r0, R.c0, R.heat, R.kE, R.Sc, R.Pr, s);
      double y0, f, dfr, t;
      growth_r(r0, s, c, y0, f, dfr, t);
      n_eval += valid;
      const double two = 2.0 * dtp * f;
      double lo = dmax(rd2, y0 + dmin(two, 0.0));   // eq. 18
      double hi = y0 + dmax(two, 0.0);              // eq. 19
      double r = r0, dprev = 0.0;
      double rq = r0, gq = 0.0, gpq = 1.0;   // previous iterate, g and dg/dr there (for the curvature estimate)
      int st;
      // guards: the range of exp_kelvin, and the bracket must hold at most one root
      const bool guard = !(t < 4.0) ||
                         !single_root_bracket<false>(lo, hi, y0, c.RH, s.rd3, s.krd3, c.A, R.invA, dtp * s.c0Dc, 0.0);
      if (!(lo < hi)) {
        st = (lo == y0) ? 1 : 2;                    // a = b: the result is a
      } else {
        const double gp = fma(-dtp, dfr, r0 + r0);
        const double rn = fma(dtp * f, rcp_nr<1>(gp), r0);
        const double yn = rn * rn;
        gq = -dtp * f; gpq = gp;
        if (!(gp > 0.0 && yn >= lo && yn <= hi)) {   // a step that rounds to nothing stays on the end it started from
          st = 2;
        } else {
          dprev = fabs(rn - r0);
          r = rn;
          st = (dprev * dprev <= KC[KC_TOL400] * (rn * rn)) ? 1 : 0;
        }
      }
#ifdef SDM_DEBUG_REASON
      if (valid && st == 2) atomicAdd(&cnt.collisions[tid], 1ull);                 // first Newton step left the bracket / a = b off y0
      if (valid && guard) atomicAdd(&cnt.pairs[tid], 1ull);                        // guard (certificate, eps, t)
#endif
      if (guard) st = 2;
      if (!valid) st = 1;
#pragma unroll 1
      for (int it = 1; it < (KF ? KF : cp.kfast); ++it) {   // KF: the bound as an immediate (0.6 % of the kernel); unrolling costs 4 %
        if (!__any_sync(0xffffffffu, st == 0)) break;
        if (st == 0) {
          double y;
          growth_r(r, s, c, y, f, dfr, t);
          ++n_eval;
          const double gv = y - y0 - dtp * f;
          const double gp = fma(-dtp, dfr, r + r);
          if (gv < 0.0) lo = y; else hi = y;
          // Newton step dN = -g/g', corrected to third order with g'' at r from the cubic through the last two
          // iterates (values and slopes): g''(r) = [6 (g_q - g)/s + 2 g'_q + 4 g']/s, s = r - r_q;
          // step = dN (1 + c), c = -dN g''/(2 g').  One reciprocal, of g' s.
          const double sq = r - rq;
          const double inv = rcp_nr<1>(gp * sq);
          const double dN = -gv * (inv * sq);
          const double h = fma(6.0 * (gq - gv), inv * gp, fma(2.0, gpq, 4.0 * gp));
          double cc = -0.5 * dN * (h * inv);
          const bool third = fabs(cc) <= 0.1;
          if (!third) cc = 0.0;
          const double rn = fma(dN, cc, dN) + r;
          const double yn = rn * rn;
          if (!(gp > 0.0 && yn >= lo && yn <= hi && t < 4.0)) {
            st = 2;
          } else {
            const double d = fabs(dN);
            const double tol = KC[KC_TOL] * rn, d2 = d * d;
            // Newton alone leaves C d^2 (C from the last two steps, at least 1/r); with the correction what is left
            // is d cm (16 (s/r)^2 + cm), cm = max(|c|, d/r): the error of the curvature estimate and the next order
            bool conv = (4.0 * d2 <= tol * rn) && (2.0 * d2 * d <= tol * (dprev * dprev));
            if (third) {
              const double cmr = dmax(fabs(cc) * rn, d);
              conv = conv || (d * cmr * fma(cmr, rn, 16.0 * (sq * sq)) <= 0.5 * tol * (yn * rn));
            }
            rq = r; gq = gv; gpq = gp;
            r = rn; dprev = d;
            if (conv || !(hi - lo > KC[KC_EPSW] * hi)) st = 1;
          }
        }
      }
#ifdef SDM_DEBUG_REASON
      if (valid && st == 0) atomicAdd(&cnt.near_ties[tid], 1ull);                  // no convergence within kfast evaluations
#endif
      if (st == 0) st = 2;
      if (valid && st == 1) {
        s_con[e] = s_dn[e] * (r * r * r - r0 * y0);
        s_r[e] = r;
        ++n_sub;
      }
      // append to the tile's slow list: one shared atomic per listed SD.  Listed SDs are rare (5e-5 of the SD-substeps), a vote
      // that aggregates them per warp is paid by every chunk (0.65 % of the kernel); the order of the list does not matter
      if (st == 2) list[atomicAdd(&ctr[1], 1u)] = (u16)e;
    }
    __syncthreads();
    // C. the listed rest, from the start of the substep: cond_solve (bracketed Newton) or the paper's literal
    // bisection.  A long list (a shock, e.g. the first step) is worked off one SD per thread; a short one
    // (steady state: usually one SD holding the whole tile at the barrier) one SD per WARP, for latency.
    const int nlist = (int)ctr[1];
    if (nlist > 0) {
      const bool per_warp = nlist <= 2 * NW;
      for (int k = per_warp ? warp : tid; k < nlist; k += per_warp ? NW : T) {
        const int e = (int)list[k];
        const CellRec& R = s_cell[(int)cidx[e]];
        const double dtp = ADAPT ? R.dtp : cp.dtp;
        CellK c;
        c.RH = R.RH; c.A = R.A; c.c0 = R.c0; c.lD = R.lD; c.lK = R.lK; c.heat = R.heat; c.kE = R.kE; c.Sc = R.Sc; c.Pr = R.Pr;
        const double r0 = s_r[e], y0 = r0 * r0;
        const double rd2 = s_rd2[e], rd3 = s_rd3[e], krd3 = s_krd3[e];
        double y1 = y0;
        unsigned ill = 0, ev = 0;
        bool solved = false;
        if (per_warp) {   // all lanes hold the same SD
          SdK s;
          double Dc, f, df, cDN;
          slow_setup(y0, rd3, krd3, c, s, Dc);
          growth_fd(y0, s, c, f, df, cDN);
          const double two = 2.0 * dtp * f;
          const double a = fmax(rd2, y0 + fmin(two, 0.0)), b = y0 + fmax(two, 0.0);   // eq. 18-19
          if (a < b) {   // the paper's procedure on the whole warp, whatever the bracket: it hands over to Newton once certified
            ev = (lane == 0);
            y1 = bisect_paper_warp(a, b, f, y0, s, c, dtp, lane, ill, ev, rd3, krd3, R.invA, dtp * s.c0Dc, dtp * cDN);
            solved = true;
          }
        }
        if (!solved) {
          cond_solve(y0, rd2, rd3, krd3, c, dtp, 200, y1, ill, ev);
          if (per_warp && lane != 0) { ill = 0; ev = 0; }   // the lanes of the warp did the same work: count it once
        }
        n_ill += ill; n_eval += ev;
        if (!per_warp || lane == 0) {
          const double r1 = sqrt(y1);
          ++n_sub; ++n_slow;
          s_con[e] = s_dn[e] * (r1 * r1 * r1 - r0 * y0);
          s_r[e] = r1;
        }
      }
      __syncthreads();
    }
  }

  for (int cl = tid; cl < nc; cl += T) {
    const int c = c_first + cl;
    const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
    const CellRec& R = s_cell[cl];
    th_f.at(i, j, k) = R.th;
    rv_f.at(i, j, k) = R.rv;
    // air properties after the feedback, used by coalescence and sedimentation (v_term)
    cf.eta[c] = R.eta;
    cf.rho_a[c] = R.rhod * (1.0 + R.rv);
  }
  for (int q = by_cell ? warp : tid; q < (by_cell ? nc : M); q += by_cell ? NW : T) {
    int cl, t0, t1;
    if (by_cell) {
      cl = q; t0 = (int)segl[cl] + lane; t1 = (int)segl[cl + 1];
    } else {
      int lo = 0, hi = nc;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)q) lo = mid; else hi = mid; }
      cl = lo; t0 = q; t1 = q + 1;
    }
    const int b0 = (int)segl[cl];
    for (int t = t0; t < t1; t += 32) {
      const u32 s = s0 + t;
      const double r = s_r[b0 + rank[s]];
      a.rw2[s] = r * r;
    }
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


// =====================================================================================================================
// fp32 arithmetic (real_t = float of the paper's templates, :747, :908; north_star: radii to 1e-4 in fp32; selected by
// sdm_set_cond_arith(ctx, 4) with real_bytes = 4).  The sweep of k_cond4 in single precision; everything that decides
// a branch of the method (root selection, ill-posed brackets, iterates leaving the bracket) still goes to the fp64
// slow list, and the cells' thermodynamics and the feedback stay fp64.  What makes single precision sufficient:
//  * lengths in micrometres (r ~ 1e-3 .. 3e3, r^3 ~ 1e-9 .. 1e10, D_0 and K_0 scaled by 1e12): every intermediate of
//    eq. 20-24 stays inside the fp32 range, and no product of three large factors is formed (three reciprocals
//    instead of the one of the fp64 path; MUFU.RCP is cheap in fp32);
//  * the unknown is the increment d = r - r0, g(d) = d (2 r0 + d) - dt' f(r0 + d): the growth per substep (1e-3 r and
//    less) is resolved to its own 1e-7, and N d(r^3) = N d (3 r0^2 + 3 r0 d + d^2) has no cancellation;
//  * the driving force without cancellation: RH - a_w e^(A/r) = (RH - 1) + kappa r_d^3 / W - a_w expm1(A/r), with RH - 1
//    taken from the fp64 cell record: three terms of size 1e-1 .. 1e-4 each known to 1e-7 of itself, where the plain
//    form subtracts two numbers near 1;
//  * the first step solves d^2 + g' d - dt' f0 = 0 exactly (Newton in r^2 with f linearised in r), so that what is
//    left is dt' f'' d^2 / (2 g'), and |f''| is bounded from quantities the evaluation has anyway:
//    |f''| <= (8/r) (|f'| + |f|/r + c (a_w' + a_w t / r) e^t), c = f / S (power-law factors of degree <= 4 and the
//    Koehler terms).  An SD is done when that bound is below 1e-6 r: a cloud droplet growing by 0.3 % per substep
//    (bound 4 (d/r)^3) and haze following its cell (bound 8 (d/r)^2, d/r < 3.5e-4) take ONE evaluation.
// MUFU approximations (1-2 ulp, no special-case branches): ample for the 1e-6 the sweep is solved to
__device__ __forceinline__ float frcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fsqrt(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float fex2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

struct CellF {   // per-cell constants of one substep, lengths in micrometres
  float S0, RH, A, invA, lD, lK, qD, qK, lD171, lK171, c0, heat, kE, Sc, Pr, pad;
};
static_assert(sizeof(CellF) == 64, "CellF");
struct SdF { float rd3, krd3, Kc, hDc, c0Dc, cDK; };

__device__ __forceinline__ void cell_to_float(const CellRec& R, CellF& F) {
  F.S0 = (float)(R.RH - 1.0); F.RH = (float)R.RH;
  F.A = (float)(R.A * 1e6); F.invA = (float)(R.invA * 1e-6);
  F.lD = (float)(R.lD * 1e6); F.lK = (float)(R.lK * 1e6);
  F.qD = (float)(R.qD * 1e12); F.qK = (float)(R.qK * 1e12);
  F.lD171 = (float)(R.lD171 * 1e6); F.lK171 = (float)(R.lK171 * 1e6);
  F.c0 = (float)R.c0; F.heat = (float)R.heat;
  F.kE = (float)(R.kE * 1e-9);   // e = kE r^(3/2), r in micrometres
  F.Sc = (float)R.Sc; F.Pr = (float)R.Pr; F.pad = 0.f;
}

// [L] ventilation at the substep's starting radius (reading R-vent), as sd_setup; D_0, K_0 in um^2/s units
__device__ __forceinline__ void sd_setup_f(float r0, const CellF& c, SdF& s) {
  const float e = c.kE * (r0 * fsqrt(r0));
  const float q = e * frcp(fsqrt(1.0f + e) + 1.0f);
  const float Re = (float)(cst::kc_delta0 * cst::kc_delta0 / 4.0) * (q * q);
  const float xs = Re * c.Sc, xp = Re * c.Pr;
  float shm, num;
  if (fmaxf(xs, xp) < 0.02f) {
    float a = 22.0f / 729.0f, b = 22.0f / 729.0f;
    a = fmaf(a, xs, -10.0f / 243.0f); b = fmaf(b, xp, -10.0f / 243.0f);
    a = fmaf(a, xs, 5.0f / 81.0f); b = fmaf(b, xp, 5.0f / 81.0f);
    a = fmaf(a, xs, -1.0f / 9.0f); b = fmaf(b, xp, -1.0f / 9.0f);
    a = fmaf(a, xs, 1.0f / 3.0f); b = fmaf(b, xp, 1.0f / 3.0f);
    shm = a * xs; num = b * xp;
  } else {
    shm = cbrtf(1.0f + xs) - 1.0f; num = cbrtf(1.0f + xp) - 1.0f;
    if (Re > 1.0f) {
      const float m = powf(Re, 0.077f) - 1.0f;
      shm = shm + m + shm * m;
      num = num + m + num * m;
    }
  }
  const float Dc = fmaf((float)(0.5e12 * cst::D_0), shm, (float)(1e12 * cst::D_0));
  s.Kc = fmaf((float)(0.5e12 * cst::K_0), num, (float)(1e12 * cst::K_0));
  s.hDc = c.heat * Dc;
  s.c0Dc = c.c0 * Dc;
  s.cDK = s.c0Dc * s.Kc;
}

// e^t - 1 for 0 <= t < 4 with relative error ~1e-7: Taylor to t^7 below 0.25 (next term 0.25^7/8! = 1.5e-9 of t),
// exp2 of the hardware otherwise
__device__ __forceinline__ float expm1_kelvin_f(float t) {
  if (t < 0.25f) {
    float p = 1.0f / 5040.0f;
    p = fmaf(p, t, 1.0f / 720.0f); p = fmaf(p, t, 1.0f / 120.0f); p = fmaf(p, t, 1.0f / 24.0f);
    p = fmaf(p, t, 1.0f / 6.0f); p = fmaf(p, t, 0.5f); p = fmaf(p, t, 1.0f);
    return p * t;
  }
  return fex2(t * 1.4426950408889634f) - 1.0f;
}

// f(r) = d r_w^2/dt [um^2/s], df/dr and B >= |d2f/dr2| (see above); r, lengths in micrometres
__device__ __forceinline__ void growth_f32(float r, const SdF& s, const CellF& c, float& f, float& dfr, float& B, float& t_out) {
  const float y = r * r;
  const float lDr = c.lD * r, lKr = c.lK * r;
  const float NM = y + lDr, DM = fmaf(1.71f, lDr, y) + c.qD;
  const float NT = y + lKr, DT = fmaf(1.71f, lKr, y) + c.qK;
  const float KN = s.Kc * NT, HN = s.hDc * NM;
  const float Q = fmaf(KN, DM, HN * DT);
  const float P = fmaf(y, r, -s.rd3), W = P + s.krd3;
  const float invQ = frcp(Q), invW = frcp(W), invr = frcp(r);
  const float t = c.A * invr;
  t_out = t;
  const float em1 = expm1_kelvin_f(t), ex = 1.0f + em1;
  const float aw = P * invW;
  const float S = c.S0 + fmaf(-aw, em1, s.krd3 * invW);
  const float NN = NM * NT;
  const float cN = s.cDK * invQ * NN;
  f = cN * S;
  const float r2 = r + r;
  const float NMp = r2 + c.lD, DMp = r2 + c.lD171, NTp = r2 + c.lK, DTp = r2 + c.lK171;
  const float NNp = fmaf(NMp, NT, NM * NTp);
  const float Qp = s.Kc * fmaf(NTp, DM, NT * DMp) + s.hDc * fmaf(NMp, DT, NM * DTp);
  const float awp = 3.0f * y * s.krd3 * (invW * invW);
  const float kel = aw * t * invr;
  const float Sp = ex * (kel - awp);
  const float lnp = NNp * frcp(NN) - Qp * invQ;   // d ln(NN/Q) / dr
  dfr = fmaf(f, lnp, cN * Sp);
  B = 8.0f * invr * (fabsf(dfr) + fabsf(f) * invr + cN * ex * (awp + kel));
}

__device__ __forceinline__ bool single_root_bracket_f(float Dlo, float Dhi, float y0, float two, float S0, float rd3, float krd3,
                                                      float A, float invA, float dtcD) {
  const float lo = y0 + Dlo, hi = y0 + Dhi;
  const float yc = 3.0f * krd3 * invA;
  if ((hi <= 0.999f * yc && krd3 <= 2.0f * rd3) || (S0 < 0.0f && Dlo == 0.0f && two > 0.0f)) return true;   // (1), (3)
  const float ym = fmaxf(lo, yc);
  const float K3 = 1.3f * A * dtcD;
  return (Dhi - Dlo <= 0.49f * lo) && (ym * ym * ym >= 1.01f * K3 * K3) && (A * A <= 0.06f * ym);             // (2)
}

constexpr float COND_TOLF = 1e-6f;   // bound on the error left in r, relative (north_star: 1e-4 on radii in fp32)

template <int CAP, int T>
struct Cond4F {
  static constexpr int NW = T / 32;
  static constexpr size_t fixed_bytes = (size_t)6 * CAP * 4 + (size_t)2 * CAP * 2;
  static size_t smem(int cpb) { return fixed_bytes + (size_t)cpb * (sizeof(CellRec) + sizeof(CellF)) + (size_t)(cpb + 1) * 4 + 16; }
};

template <int CAP, int T, int MINB>
__global__ void __launch_bounds__(T, MINB)
k_cond4f(SdArraysT<float> a, const u16* __restrict__ rank, const u32* __restrict__ seg, Grid g, Field th_f, Field rv_f,
         CellFields cf, CondParams cp, Counters cnt, int cpb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using L = Cond4F<CAP, T>;
  constexpr int NW = L::NW;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c_first = blockIdx.x * cpb;
  const int nc = min(cpb, g.ncell - c_first);
  float* s_r = reinterpret_cast<float*>(smem_raw);   // micrometres
  float *s_rd3 = s_r + CAP, *s_krd3 = s_r + 2 * CAP, *s_dn = s_r + 3 * CAP, *s_rd2 = s_r + 4 * CAP, *s_con = s_r + 5 * CAP;
  u16* cidx = reinterpret_cast<u16*>(s_r + 6 * CAP);
  u16* list = cidx + CAP;
  CellRec* s_cell = reinterpret_cast<CellRec*>(smem_raw + L::fixed_bytes);
  CellF* s_cf = reinterpret_cast<CellF*>(s_cell + cpb);
  u32* segl = reinterpret_cast<u32*>(s_cf + cpb);
  u32* ctr = segl + cpb + 1;   // [0] next chunk of the sweep, [1] length of the slow list
  const u32 s0 = seg[c_first];
  const int M = (int)(seg[c_first + nc] - s0);

  // The fp32 sweep costs ~8 instructions per SD-substep, so what surrounds it is organised for instruction count:
  // the cells' fp64 thermodynamics run on the lanes of ONE warp (the chain is as long for 3 lanes as for 30, and four
  // warps issuing it cost four times the slots), staging and the per-cell sums go cell by cell without searches.
  for (int cl = tid; cl < nc; cl += T) {
    const int c = c_first + cl;
    const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
    CellRec& R = s_cell[cl];
    R.th = th_f.at(i, j, k); R.rv = rv_f.at(i, j, k);
    const double rhod = cf.rhod[c];
    R.rhod = rhod;
    R.fbk = -(4.0 * cst::pi * cst::rho_w / 3.0) / (rhod * g.dV);   // eq. 25 prefactor
    segl[cl] = seg[c] - s0;
  }
  if (tid == 0) { segl[nc] = (u32)M; ctr[0] = 0u; ctr[1] = 0u; }
  __syncthreads();
  const bool by_cell = M >= 24 * nc;   // populated cells: a warp stages a cell at a time
  for (int q = by_cell ? warp : tid; q < (by_cell ? nc : M); q += by_cell ? NW : T) {   // stage the tile in sorted order, lengths in micrometres
    int cl, t0, t1;
    if (by_cell) {
      cl = q; t0 = (int)segl[cl] + lane; t1 = (int)segl[cl + 1];
    } else {
      int lo = 0, hi = nc;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)q) lo = mid; else hi = mid; }
      cl = lo; t0 = q; t1 = q + 1;
    }
    const int b0 = (int)segl[cl];
    for (int t = t0; t < t1; t += 32) {
      const u32 s = s0 + t;
      const int e = b0 + rank[s];
      const float rd3 = a.rd3[s] * 1e18f;
      const float q3 = cbrtf(rd3);
      s_r[e] = fsqrt(a.rw2[s] * 1e12f);
      s_rd3[e] = rd3;
      s_krd3[e] = a.kappa[s] * rd3;
      s_dn[e] = (float)a.n[s];
      s_rd2[e] = q3 * q3;
      cidx[e] = (u16)cl;
    }
  }
  // per-lane counters, packed so that the sweep holds one register: evaluations (low 20 bits: a lane stays far below 2^20 per
  // launch) and solved SD-substeps (high 12: at most ~7 per substep and lane, sstp_cond <= 500); the slow list's counters are touched only there
  unsigned n_es = 0, n_ill = 0, n_slow = 0;
  const float dtp = (float)cp.dtp;
  const int nsub = M > 0 ? cp.sstp : 0;
  for (int sub = 0; sub <= nsub; ++sub) {
    // D. per-cell sums of N d(r_w^3) [um^3]: 8 lanes per cell, fixed order (deterministic); R.pad carries the sum
    if (sub > 0) {
      const int l8 = lane & 7, grp = lane >> 3;
      for (int cl = warp * 4 + grp; cl < ((nc + 3) & ~3); cl += NW * 4) {   // warp-uniform trip count
        float acc = 0.0f;   // fp32 sum of ~64 terms: 1e-6 of the substep's change of r_v
        if (cl < nc) {
          const int b1 = (int)segl[cl + 1];
          for (int e = (int)segl[cl] + l8; e < b1; e += 8) acc += s_con[e];
        }
        acc += __shfl_xor_sync(0xffffffffu, acc, 4);
        acc += __shfl_xor_sync(0xffffffffu, acc, 2);
        acc += __shfl_xor_sync(0xffffffffu, acc, 1);
        if (cl < nc && l8 == 0) s_cell[cl].pad = (double)acc * 1e-18;
      }
      __syncthreads();
    }
    // A. feedback (eq. 25-26) and the constants of the next substep, fp64, one lane per cell on the first warp(s)
    if (tid < ((nc + 31) & ~31)) {
      for (int cl = tid; cl < nc; cl += T) {
        CellRec& R = s_cell[cl];
        if (sub == 0) cell_init(R, cp.RH_max); else cell_advance(R, R.pad, cp.RH_max, true);
        cell_to_float(R, s_cf[cl]);
      }
    }
    if (tid == 0) { ctr[0] = 0u; ctr[1] = 0u; }
    if (sub == nsub) break;
    __syncthreads();
    // B. dense sweep in fp32.  st: 0 = iterating, 1 = solved, 2 = left to the fp64 list
    for (int q0 = warp * 32; q0 < M; q0 += NW * 32) {   // static chunks: with ~1 evaluation per SD the warps stay balanced
      const bool valid = q0 + lane < M;
      const int e = min(q0 + lane, M - 1);   // lanes past the end of the tile redo its last SD and discard the result
      const CellF c = s_cf[(int)cidx[e]];
      const float r0 = s_r[e], rd2 = s_rd2[e];
      SdF s;
      s.rd3 = s_rd3[e]; s.krd3 = s_krd3[e];
      sd_setup_f(r0, c, s);
      float f, dfr, B, t;
      growth_f32(r0, s, c, f, dfr, B, t);
      n_es += valid;
      const float y0 = r0 * r0, r02 = r0 + r0;
      const float dtf = dtp * f, two = dtf + dtf;
      // eq. 18-19 in D = y - y0
      float Dlo = fmaxf(rd2 - y0, fminf(two, 0.0f)), Dhi = fmaxf(two, 0.0f);
      const bool guard = !(t < 4.0f) || !single_root_bracket_f(Dlo, Dhi, y0, two, c.S0, s.rd3, s.krd3, c.A, c.invA, dtp * s.c0Dc);
      Dlo *= 0.99f; Dhi *= 0.99f;   // an iterate this close to an end of the bracket is left to the fp64 list
      float d = 0.0f;
      int st;
      if (!(Dlo < Dhi)) {
        st = (two == 0.0f) ? 1 : 2;   // a = b = y0: the result is a
      } else {
        const float gp = fmaf(-dtp, dfr, r02);
        const float disc = fmaf(gp, gp, 4.0f * dtf);
        if (!(gp > 0.0f && disc > 0.0f)) {
          st = 2;
        } else {
          d = two * frcp(gp + fsqrt(disc));   // d^2 + g' d - dt' f0 = 0, the root that vanishes with f0
          const float D = d * (r02 + d);
          if (!(D >= Dlo && D <= Dhi)) st = 2;
          else st = (dtp * B * d * d <= 2.0f * COND_TOLF * gp * (r0 + d)) ? 1 : 0;
        }
      }
      if (guard) st = 2;
      if (!valid) st = 1;
      for (int it = 1; it < cp.kfast; ++it) {
        if (!__any_sync(0xffffffffu, st == 0)) break;
        if (st == 0) {
          const float r = r0 + d;
          growth_f32(r, s, c, f, dfr, B, t);
          ++n_es;
          const float D = d * (r02 + d);
          const float gv = fmaf(-dtp, f, D);
          const float gp = fmaf(-dtp, dfr, r + r);
          if (gv < 0.0f) Dlo = D; else Dhi = D;
          const float dN = -gv * frcp(gp);
          const float dn = d + dN;
          const float Dn = dn * (r02 + dn);
          if (!(gp > 0.0f && Dn >= Dlo && Dn <= Dhi && t < 4.0f)) {
            st = 2;
          } else {
            d = dn;
            st = (fmaf(dtp, B, 2.0f) * dN * dN <= 2.0f * COND_TOLF * gp * (r0 + dn)) ? 1 : 0;
          }
        }
      }
      if (st == 0) st = 2;
      if (valid && st == 1) {
        s_con[e] = s_dn[e] * (d * fmaf(3.0f * r0, r0 + d, d * d));   // N (r^3 - r0^3) without cancellation
        s_r[e] = r0 + d;
        n_es += 0x100000u;
      }
      if (st == 2) list[atomicAdd(&ctr[1], 1u)] = (u16)e;   // as in k_cond4: no vote per chunk for the rare listed SD
    }
    __syncthreads();
    // C. the listed rest in fp64 (SI units), exactly as k_cond4 does: cond_solve or the paper's literal bisection
    const int nlist = (int)ctr[1];
    if (nlist > 0) {
      const bool per_warp = nlist <= 2 * NW;
      for (int k = per_warp ? warp : tid; k < nlist; k += per_warp ? NW : T) {
        const int e = (int)list[k];
        const CellRec& R = s_cell[(int)cidx[e]];
        CellK c;
        c.RH = R.RH; c.A = R.A; c.c0 = R.c0; c.lD = R.lD; c.lK = R.lK; c.heat = R.heat; c.kE = R.kE; c.Sc = R.Sc; c.Pr = R.Pr;
        const double r0 = (double)s_r[e] * 1e-6, y0 = r0 * r0;
        const double rd3 = (double)s_rd3[e] * 1e-18, krd3 = (double)s_krd3[e] * 1e-18;
        const double rd2 = fmin((double)s_rd2[e] * 1e-12, y0);
        double y1 = y0;
        unsigned ill = 0, ev = 0;
        bool solved = false;
        if (per_warp) {   // all lanes hold the same SD
          SdK s;
          double Dc, f, df, cDN;
          slow_setup(y0, rd3, krd3, c, s, Dc);
          growth_fd(y0, s, c, f, df, cDN);
          const double two = 2.0 * cp.dtp * f;
          const double a_ = fmax(rd2, y0 + fmin(two, 0.0)), b_ = y0 + fmax(two, 0.0);   // eq. 18-19
          if (a_ < b_) {   // the paper's procedure on the whole warp, whatever the bracket: it hands over to Newton once certified
            ev = (lane == 0);
            y1 = bisect_paper_warp(a_, b_, f, y0, s, c, cp.dtp, lane, ill, ev, rd3, krd3, R.invA, cp.dtp * s.c0Dc, cp.dtp * cDN);
            solved = true;
          }
        }
        if (!solved) {
          cond_solve(y0, rd2, rd3, krd3, c, cp.dtp, 200, y1, ill, ev);
          if (per_warp && lane != 0) { ill = 0; ev = 0; }
        }
        n_ill += ill; n_es += ev;
        if (!per_warp || lane == 0) {
          const double r1 = sqrt(y1);
          n_es += 0x100000u; ++n_slow;
          s_con[e] = (float)((double)s_dn[e] * (r1 * r1 * r1 - r0 * y0) * 1e18);
          s_r[e] = (float)(r1 * 1e6);
        }
      }
      __syncthreads();
    }
  }

  for (int cl = tid; cl < nc; cl += T) {
    const int c = c_first + cl;
    const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
    const CellRec& R = s_cell[cl];
    th_f.at(i, j, k) = R.th;
    rv_f.at(i, j, k) = R.rv;
    cf.eta[c] = R.eta;   // air properties after the feedback, used by coalescence and sedimentation (v_term)
    cf.rho_a[c] = R.rhod * (1.0 + R.rv);
  }
  for (int q = by_cell ? warp : tid; q < (by_cell ? nc : M); q += by_cell ? NW : T) {
    int cl, t0, t1;
    if (by_cell) {
      cl = q; t0 = (int)segl[cl] + lane; t1 = (int)segl[cl + 1];
    } else {
      int lo = 0, hi = nc;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)q) lo = mid; else hi = mid; }
      cl = lo; t0 = q; t1 = q + 1;
    }
    const int b0 = (int)segl[cl];
    for (int t = t0; t < t1; t += 32) {
      const u32 s = s0 + t;
      const float r = s_r[b0 + rank[s]] * 1e-6f;
      a.rw2[s] = r * r;
    }
  }
  unsigned v0 = n_ill, v1 = n_es & 0xfffffu, v2 = n_es >> 20, v3 = n_slow;
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

// the two instantiations: sparse cells (5 CTAs of 128 threads per SM) and crowded cells (one CTA of 512)
#ifndef SDM_COND_CAP
#define SDM_COND_CAP 800   // SD slots of the small tile kernel
#define SDM_COND_MINB 5    // its CTAs per SM
#endif
#ifndef SDM_COND32_MINB
#define SDM_COND32_MINB 8  // CTAs per SM of the fp32-arithmetic small tile kernel
#endif
#ifndef SDM_COND32_CAP
#define SDM_COND32_CAP 800 // its SD slots
#endif
#ifndef SDM_COND32_T
#define SDM_COND32_T 128   // its threads
#endif
using CondSmall = Cond4<SDM_COND_CAP, 128>;
using CondMedium = Cond4<1280, 256>;   // 3 CTAs of 256 threads per SM: cells of ~1000 SDs
using CondLarge = Cond4<4096, 512>;    // one CTA of 512 threads per SM: cells of thousands of SDs
constexpr size_t kCondSmallBudget = (228 * 1024 - SDM_COND_MINB * 1024) / SDM_COND_MINB;   // per CTA, 1 KB reserved each
constexpr size_t kCondMediumBudget = (228 * 1024 - 3 * 1024) / 3;
constexpr size_t kCondLargeBudget = 227 * 1024;

// 1, 2, 3: small, medium, large tile kernel (in order of preference); 0: a tile of cpb cells with up to `need`
// SDs fits none of them
// most cells a tile of the small kernel can hold (its SD slots are a compile-time constant, the cell records take what is left)
int cond_max_cells(bool arith32) {
  int c = 1;
  if (arith32) { while (c < 128 && Cond4F<SDM_COND32_CAP, SDM_COND32_T>::smem(c + 1) <= (228 * 1024 - SDM_COND32_MINB * 1024) / SDM_COND32_MINB) ++c; }
  else { while (c < 128 && CondSmall::smem(c + 1) <= kCondSmallBudget) ++c; }
  return c;
}
int cond_variant(int cpb, int need) {
  if (cpb <= 128 && need <= SDM_COND_CAP && CondSmall::smem(cpb) <= kCondSmallBudget) return 1;
  if (cpb <= 256 && need <= 1280 && CondMedium::smem(cpb) <= kCondMediumBudget) return 2;
  if (cpb <= 512 && need <= 4096 && CondLarge::smem(cpb) <= kCondLargeBudget) return 3;
  return 0;
}

template <int CAP, int T, int MINB, typename R>
static cudaError_t launch_cond4(size_t smem, int grid, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g, Field th,
                                Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt, int cpb,
                                cudaStream_t st) {
  if (cp.adapt_tol > 0.0) {
    cudaError_t e = cudaFuncSetAttribute(k_cond4<CAP, T, MINB, R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_cond4<CAP, T, MINB, R, true><<<grid, T, smem, st>>>(a, rank, seg, g, th, rv, cf, cp, cnt, cpb);
  } else if (CAP == SDM_COND_CAP && cp.kfast == 4) {   // the default of the small tile kernel
    cudaError_t e = cudaFuncSetAttribute(k_cond4<CAP, T, MINB, R, false, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_cond4<CAP, T, MINB, R, false, 4><<<grid, T, smem, st>>>(a, rank, seg, g, th, rv, cf, cp, cnt, cpb);
  } else {
    cudaError_t e = cudaFuncSetAttribute(k_cond4<CAP, T, MINB, R, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_cond4<CAP, T, MINB, R, false><<<grid, T, smem, st>>>(a, rank, seg, g, th, rv, cf, cp, cnt, cpb);
  }
  return cudaGetLastError();
}

template <int CAP, int T, int MINB>
static cudaError_t launch_cond4f(size_t smem, int grid, const SdArraysT<float>& a, const u16* rank, const u32* seg, const Grid& g,
                                 Field th, Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt, int cpb,
                                 cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(k_cond4f<CAP, T, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_cond4f<CAP, T, MINB><<<grid, T, smem, st>>>(a, rank, seg, g, th, rv, cf, cp, cnt, cpb);
  return cudaGetLastError();
}

// as cond_variant, for the fp32-arithmetic tile kernels (28 instead of 52 bytes of shared memory per SD)
using Cond32Small = Cond4F<SDM_COND32_CAP, SDM_COND32_T>;
int cond_variant_f32(int cpb, int need) {
  constexpr size_t small_budget = (228 * 1024 - SDM_COND32_MINB * 1024) / SDM_COND32_MINB;
  if (cpb <= 128 && need <= SDM_COND32_CAP && Cond32Small::smem(cpb) <= small_budget) return 1;
  if (cpb <= 256 && need <= 1280 && Cond4F<1280, 256>::smem(cpb) <= (228 * 1024 - 4 * 1024) / 4) return 2;
  if (cpb <= 512 && need <= 4096 && Cond4F<4096, 512>::smem(cpb) <= 227 * 1024) return 3;
  return 0;
}

// fp32-arithmetic condensation for the tile variants 1..3 of cond_variant_f32; variant 0 (one crowded cell in global
// memory) has no fp32 form
cudaError_t launch_cond_f32(int cpb, int variant, const SdArraysT<float>& a, const u16* rank, const u32* seg, const Grid& g,
                            Field th, Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt, cudaStream_t st) {
  const int grid = (g.ncell + cpb - 1) / cpb;
  if (variant == 1)
    return launch_cond4f<SDM_COND32_CAP, SDM_COND32_T, SDM_COND32_MINB>(Cond32Small::smem(cpb), grid, a, rank, seg, g, th, rv, cf, cp, cnt, cpb, st);
  if (variant == 2) return launch_cond4f<1280, 256, 4>(Cond4F<1280, 256>::smem(cpb), grid, a, rank, seg, g, th, rv, cf, cp, cnt, cpb, st);
  if (variant == 3) return launch_cond4f<4096, 512, 1>(Cond4F<4096, 512>::smem(cpb), grid, a, rank, seg, g, th, rv, cf, cp, cnt, cpb, st);
  return cudaErrorInvalidValue;
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

// variant as returned by cond_variant(cpb, need); 0: work in place in global memory (cpb must be 1),
// `alt` = the idle ping-pong copy of the state used as scratch.
template <typename R>
cudaError_t launch_cond(int cpb, int variant, const SdArraysT<R>& a, const SdArraysT<R>& alt, const u16* rank, const u32* seg,
                        const Grid& g, Field th, Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt,
                        cudaStream_t st) {
  const int grid = (g.ncell + cpb - 1) / cpb;
  if (variant == 1)
    return launch_cond4<SDM_COND_CAP, 128, SDM_COND_MINB>(CondSmall::smem(cpb), grid, a, rank, seg, g, th, rv, cf, cp, cnt, cpb, st);
  if (variant == 2) return launch_cond4<1280, 256, 3>(CondMedium::smem(cpb), grid, a, rank, seg, g, th, rv, cf, cp, cnt, cpb, st);
  if (variant == 3) return launch_cond4<4096, 512, 1>(CondLarge::smem(cpb), grid, a, rank, seg, g, th, rv, cf, cp, cnt, cpb, st);
  k_cond<false, R><<<grid, COND_THREADS, cond_smem_bytes(cpb, 0), st>>>(a, alt, rank, seg, g, th, rv, cf, cp, cnt, cpb, 0);
  return cudaGetLastError();
}

#define SDM_INST(R)                                                                                                     \
  template cudaError_t launch_cond<R>(int, int, const SdArraysT<R>&, const SdArraysT<R>&, const u16*, const u32*, const Grid&, \
                                      Field, Field, const CellFields&, const CondParams&, const Counters&, cudaStream_t);
SDM_INSTANTIATE_REAL(SDM_INST)
#undef SDM_INST

void launch_thermo(const Grid& g, Field th, Field rv, const CellFields& cf, cudaStream_t st) {
  k_thermo<<<(g.ncell + 127) / 128, 128, 0, st>>>(g, th, rv, cf);
}

}  // namespace sdm
