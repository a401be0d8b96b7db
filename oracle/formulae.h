// ORACLE (test infrastructure, not the product): plain fp64 formulae of the
// particle-based scheme of arxiv 1310.1905. Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may use anything under oracle/. Shares no code with the CUDA path.
//
// Every function cites the PAPER.md passage it restates.  Formulae the paper
// cites but does not print are tagged [L] (literature form chosen in
// DESIGN.md "Readings"); their fidelity to the paper's code is "parity
// unpinned" -- they are pinned only by textbook values and limits
// (tests/test_oracle_pins.py).
#pragma once
#include <cmath>
#include <cstdint>
#include <algorithm>

namespace orc {

// ---- constants ------------------------------------------------------------
// printed in PAPER.md Table 2 (:1052-1108) and :1020
constexpr double rho_w   = 1000.0;   // :1065 density of liquid water
constexpr double sigma_w = 0.072;    // :1070 surface tension of water
constexpr double c_pd    = 1005.0;   // :1077
constexpr double c_pv    = 1850.0;   // :1077
constexpr double c_l     = 4218.0;   // :1077
constexpr double l_v0    = 2.5e6;    // :1086 latent heat at the triple point
constexpr double p_1000  = 1.0e5;    // :1020
// [L] not printed in the paper (reading R-const)
constexpr double R_d   = 287.0;
constexpr double R_v   = 461.5;
constexpr double T_0   = 273.16;     // triple point
constexpr double p_vs0 = 611.73;     // p_vs(T_0)
constexpr double g_acc = 9.81;
constexpr double D_0   = 2.21e-5;    // vapour diffusivity in air
constexpr double K_0   = 2.4e-2;     // thermal conductivity of air
constexpr double pi    = 3.14159265358979323846;

// ---- diagnosing T and p (PAPER.md :1042-1046, eq. 43-44) -------------------
inline double T_of(double th, double rhod) {
  // eq. 43: T = [theta (rhod R_d / p_1000)^(R_d/c_pd)]^(c_pd/(c_pd-R_d))
  return std::pow(th * std::pow(rhod * R_d / p_1000, R_d / c_pd), c_pd / (c_pd - R_d));
}
inline double p_of(double rhod, double rv, double T) {
  // eq. 44: p = rhod (R_d + rv R_v) T
  return rhod * (R_d + rv * R_v) * T;
}
// Table 2 (:1087): l_v(T) = l_v0 + (c_pv - c_l)(T - T_0)
inline double l_v(double T) { return l_v0 + (c_pv - c_l) * (T - T_0); }

// [L] saturation vapour pressure: the exact Clausius-Clapeyron integral for
// the linear l_v(T) above, d ln p_vs / dT = l_v / (R_v T^2).
inline double p_vs(double T) {
  const double a = (l_v0 + (c_l - c_pv) * T_0) / R_v;
  const double b = (c_l - c_pv) / R_v;
  return p_vs0 * std::exp(a * (1.0 / T_0 - 1.0 / T) - b * std::log(T / T_0));
}

// [L] dynamic viscosity of air (Sutherland-type form)
inline double eta_air(double T) {
  const double q = T / 273.0;
  return 1.72e-5 * (393.0 / (T + 120.0)) * (q * std::sqrt(q));
}

// ---- terminal velocity (PAPER.md :649, :606): Khvorostyanov & Curry 2002,
// eqs 2.7, 2.12, 2.13, 3.1 for a smooth sphere [L].  Best number
// X = (32/3) r^3 (rho_w-rho_a) g rho_a / eta^2, Re = (delta0^2/4)
// [sqrt(1+c1 sqrt(X)) - 1]^2 with c1 = 4/(delta0^2 sqrt(C0)), v = eta Re/(2 r rho_a).
// sqrt(1+e)-1 is written e/(sqrt(1+e)+1): the same number without cancellation.
inline double v_term(double r, double eta, double rho_a) {
  constexpr double delta0 = 9.06, C0 = 0.292;
  const double c1 = 4.0 / (delta0 * delta0 * std::sqrt(C0));
  const double X = (32.0 / 3.0) * (r * r * r) * (rho_w - rho_a) * g_acc * rho_a / (eta * eta);
  const double e = c1 * std::sqrt(X);
  const double s = e / (std::sqrt(1.0 + e) + 1.0);
  const double Re = (delta0 * delta0 / 4.0) * (s * s);
  return eta * Re / (2.0 * r * rho_a);
}

// ---- per-cell quantities used by condensation, coalescence, sedimentation ---
struct CellThermo {
  double T, p, rhod, rv;
  double lv, rho_vs, RH, A;        // condensation (PAPER.md :590-594, Table 2 :1056)
  double lambda_D, lambda_K;       // [L] Fuchs-Sutugin mean free paths
  double eta, rho_a;               // for v_term
  double Sc, Pr;                   // [L] Schmidt and Prandtl numbers
  double heat;                     // (rho_vs l_v / T)(l_v/(R_v T) - 1), eq. 21
};

inline CellThermo cell_thermo(double th, double rv, double rhod, double RH_max) {
  CellThermo c;
  c.rhod = rhod; c.rv = rv;
  c.T = T_of(th, rhod);
  c.p = p_of(rhod, rv, c.T);
  c.lv = l_v(c.T);
  c.rho_vs = p_vs(c.T) / (R_v * c.T);
  // eq. 30: rho_v = rv rhod; RH limited by opts.RH_max (:685, :665)
  c.RH = std::min(rv * rhod / c.rho_vs, RH_max);
  c.A = 2.0 * sigma_w / (R_v * c.T * rho_w);   // Table 2 :1056
  c.lambda_D = 2.0 * D_0 / std::sqrt(2.0 * R_v * c.T);
  c.lambda_K = (4.0 / 5.0) * K_0 * c.T / (c.p * std::sqrt(2.0 * R_d * c.T));
  c.eta = eta_air(c.T);
  c.rho_a = rhod * (1.0 + rv);
  c.Sc = c.eta / (c.rho_a * D_0);
  c.Pr = c.eta * c_pd / K_0;
  c.heat = (c.rho_vs * c.lv / c.T) * (c.lv / (R_v * c.T) - 1.0);
  return c;
}

// [L] Fuchs-Sutugin transition-regime factor, unit accommodation (:602)
inline double beta_FS(double Kn) { return (1.0 + Kn) / (1.0 + 1.71 * Kn + 1.33 * Kn * Kn); }

// [L] Sherwood / Nusselt number after Clift et al. (:602): twice the
// ventilation coefficient; X = Sc or Pr.
inline double vent(double Re, double X) {
  return 1.0 + std::cbrt(1.0 + Re * X) * std::max(1.0, std::pow(Re, 0.077));
}

// ---- drop growth (PAPER.md :581-602, eq. 20-24) -----------------------------
// d(r_w^2)/dt at y = r_w^2 for one SD. Sh, Nu are those of the substep's
// starting radius (reading R-vent).
inline double growth_f(double y, double rd3, double kappa, const CellThermo& c, double Sh, double Nu) {
  const double r = std::sqrt(y);
  const double D = D_0 * beta_FS(c.lambda_D / r) * Sh / 2.0;   // eq. 23
  const double K = K_0 * beta_FS(c.lambda_K / r) * Nu / 2.0;   // eq. 24
  const double Deff = 1.0 / (1.0 / D + c.heat / K);            // eq. 21
  const double r3 = y * r;
  const double aw = (r3 - rd3) / (r3 - rd3 * (1.0 - kappa));   // Table 2 :1074
  // eq. 20 with eq. 22; rho_v = RH rho_vs
  return 2.0 * (Deff / rho_w) * c.rho_vs * (c.RH - aw * std::exp(c.A / r));
}

// One condensation substep for one SD (PAPER.md :568-579, eq. 17-19 with the
// dt' factor of DESIGN.md reading R-bracket). Returns the new r_w^2.
// *ill_posed is set when the bracket branch (:579) was taken.
inline double cond_substep_sd(double y0, double rd3, double kappa, const CellThermo& c,
                              double dtp, int* ill_posed, long* n_eval) {
  const double r0 = std::sqrt(y0);
  const double vt = v_term(r0, c.eta, c.rho_a);
  const double Re = 2.0 * r0 * vt * c.rho_a / c.eta;
  const double Sh = vent(Re, c.Sc), Nu = vent(Re, c.Pr);
  auto g = [&](double y) { if (n_eval) ++*n_eval; return y - y0 - dtp * growth_f(y, rd3, kappa, c, Sh, Nu); };
  const double f0 = growth_f(y0, rd3, kappa, c, Sh, Nu);
  if (n_eval) ++*n_eval;
  const double rd2 = std::cbrt(rd3) * std::cbrt(rd3);
  double a = std::max(rd2, y0 + std::min(2.0 * dtp * f0, 0.0));   // eq. 18
  double b = y0 + std::max(2.0 * dtp * f0, 0.0);                  // eq. 19
  if (ill_posed) *ill_posed = 0;
  if (!(a < b)) return a;
  double ga = g(a), gb = g(b);
  if (ga == 0.0) return a;
  if (gb == 0.0) return b;
  if ((ga > 0.0) == (gb > 0.0)) {          // :579 bisection ill-posed -> (a+b)/2
    // counted only when the bracket is wider than 1e-9 b: below that the sign of g at the far end is
    // rounding noise of f and either branch returns the same value to 1e-9
    if (ill_posed) *ill_posed = (b - a > 1e-9 * b) ? 1 : 0;
    return 0.5 * (a + b);
  }
  while (b - a > 1e-15 * b) {               // bisection
    const double m = 0.5 * (a + b);
    if (m <= a || m >= b) break;
    const double gm = g(m);
    if (gm == 0.0) return m;
    if ((gm > 0.0) == (ga > 0.0)) { a = m; ga = gm; } else { b = m; gb = gm; }
  }
  return 0.5 * (a + b);
}

// ---- particle advection (PAPER.md :534-556, eq. 13-16) ----------------------
// closed-form backward-Euler position with linear Courant interpolation
inline double adve_1d(double x, double dx, double C_lo, double C_hi) {
  const double i = std::floor(x / dx);
  const double dC = C_hi - C_lo;
  return (x + dx * (C_lo - i * dC)) / (1.0 - dC);   // eq. 16
}

// ---- Philox-4x32-10 (Salmon et al. 2011; BASELINE.json north_star) ----------
inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

}  // namespace orc
