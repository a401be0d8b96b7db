// Stage a4: condensational growth, all sstp_cond substeps fused in one
// cell-resident kernel.  A group of G threads owns one grid cell: it stages the cell's SDs in shared
// memory in sorted order, and per substep (i) diagnoses T, p, rho_vs, RH.. from theta, r_v, rho_d
// (eq. 43-44, Table 2), (ii) solves eq. 17 for every SD by a bracketed Newton iteration on
// r_w^2 inside the interval of eq. 18-19 (the paper bisects, :579, and names a faster root finder as
// the first optimisation, :912), (iii) reduces sum N (r_w^3' - r_w^3) over the cell and applies the
// feedback of eq. 25-26 to r_v and theta.  fp64 throughout; this kernel is fp64-ALU bound.
#include "sdm_kernels.cuh"

namespace sdm {

struct CellC {   // per-cell constants of one substep
  double RH, A, c0, lD, lK, heat, eta, rho_a, Sc, Pr, T, lv;
};

__device__ __forceinline__ CellC cell_consts(double th, double rv, double rhod, double c_exn, double RH_max) {
  CellC c;
  // eq. 43: T = [theta (rhod R_d/p_1000)^(R_d/c_pd)]^(c_pd/(c_pd-R_d)); c_exn is the inner power (rhod is fixed)
  const double T = pow(th * c_exn, cst::c_pd / (cst::c_pd - cst::R_d));
  const double p = rhod * (cst::R_d + rv * cst::R_v) * T;                 // eq. 44
  const double lv = cst::l_v0 + (cst::c_pv - cst::c_l) * (T - cst::T_0);  // Table 2 :1087
  // [L] Clausius-Clapeyron integral for the linear l_v(T)
  const double ca = (cst::l_v0 + (cst::c_l - cst::c_pv) * cst::T_0) / cst::R_v;
  const double cb = (cst::c_l - cst::c_pv) / cst::R_v;
  const double pvs = cst::p_vs0 * exp(ca * (1.0 / cst::T_0 - 1.0 / T) - cb * log(T / cst::T_0));
  const double rho_vs = pvs / (cst::R_v * T);
  c.T = T; c.lv = lv;
  c.RH = fmin(rv * rhod / rho_vs, RH_max);                                // eq. 30, :685
  c.A = 2.0 * cst::sigma_w / (cst::R_v * T * cst::rho_w);                 // Table 2 :1056
  c.c0 = 2.0 * rho_vs / cst::rho_w;
  c.lD = 2.0 * cst::D_0 / sqrt(2.0 * cst::R_v * T);                       // [L] Fuchs-Sutugin lengths
  c.lK = (4.0 / 5.0) * cst::K_0 * T / (p * sqrt(2.0 * cst::R_d * T));
  c.heat = (rho_vs * lv / T) * (lv / (cst::R_v * T) - 1.0);               // eq. 21
  c.eta = eta_air(T);
  c.rho_a = rhod * (1.0 + rv);
  c.Sc = c.eta / (c.rho_a * cst::D_0);
  c.Pr = c.eta * cst::c_pd / cst::K_0;
  return c;
}

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

// Growth rate f(y) = d r_w^2/dt (eq. 20-24) and df/dy at y = r_w^2, written with one division:
//   beta_M = N_M/D_M, beta_T = N_T/D_T (Fuchs-Sutugin multiplied through by r^2),
//   D_eff = Dc Kc N_M N_T / Q,  Q = Kc N_T D_M + heat Dc N_M D_T,
//   a_w = P/W, P = r^3 - r_d^3, W = P + kappa r_d^3,  f = c0 D_eff (RH - a_w exp(A/r)).
__device__ __forceinline__ void growth_fd(double y, double rd3, double krd3, double Dc, double Kc, const CellC& c,
                                          double& f, double& df) {
  const double invr = rsqrt(y);
  const double r = y * invr;
  const double lDr = c.lD * r, lKr = c.lK * r;
  const double NM = y + lDr, DM = y + 1.71 * lDr + 1.33 * (c.lD * c.lD);
  const double NT = y + lKr, DT = y + 1.71 * lKr + 1.33 * (c.lK * c.lK);
  const double KN = Kc * NT, HN = c.heat * Dc * NM;
  const double Q = KN * DM + HN * DT;
  const double r3 = y * r;
  const double P = r3 - rd3, W = P + krd3;
  const double ex = exp(c.A * invr);
  const double invQW = 1.0 / (Q * W);
  const double invQ = invQW * W, invW = invQW * Q;
  const double Deff = Dc * KN * NM * invQ;
  const double aw = P * invW;
  const double S = c.RH - aw * ex;
  f = c.c0 * Deff * S;
  // derivative
  const double hr = 0.5 * invr;   // dr/dy
  const double NMp = 1.0 + c.lD * hr, DMp = 1.0 + 1.71 * c.lD * hr;
  const double NTp = 1.0 + c.lK * hr, DTp = 1.0 + 1.71 * c.lK * hr;
  const double Qp = Kc * (NTp * DM + NT * DMp) + c.heat * Dc * (NMp * DT + NM * DTp);
  const double dlnD = (NMp * NT + NTp * NM) / (NM * NT) - Qp * invQ;
  const double invr3 = invr * invr * invr;
  const double Sp = -ex * (1.5 * r * krd3 * invW * invW - aw * (0.5 * c.A * invr3));
  df = c.c0 * Deff * (dlnD * S + Sp);
}

// One condensation substep of one SD: root of g(y) = y - y0 - dt' f(y) in [a, b] of eq. 18-19
// (reading R-bracket), with the ill-posed-bracket rule of :579.
__device__ __forceinline__ double cond_solve(double y0, double rd2, double rd3, double krd3, const CellC& c, double dtp,
                                             unsigned& n_ill, unsigned& n_eval) {
  const double r0 = sqrt(y0);
  const double vt = v_term(r0, c.eta, c.rho_a);
  const double Re = 2.0 * r0 * vt * c.rho_a / c.eta;
  const double Dc = cst::D_0 * vent(Re, c.Sc) * 0.5;   // eq. 23 without beta_M
  const double Kc = cst::K_0 * vent(Re, c.Pr) * 0.5;   // eq. 24 without beta_T
  double f, df;
  growth_fd(y0, rd3, krd3, Dc, Kc, c, f, df);
  ++n_eval;
  const double two = 2.0 * dtp * f;
  const double a = fmax(rd2, y0 + fmin(two, 0.0));   // eq. 18
  const double b = y0 + fmax(two, 0.0);              // eq. 19
  if (!(a < b)) return a;
  // g(lo) < 0 < g(hi); the end that is not y0 has not been evaluated yet
  double lo = a, hi = b;
  bool lo_unv = !(f > 0.0), hi_unv = (f > 0.0);
  double y = y0, g = -dtp * f, gp = 1.0 - dtp * df;
  for (int it = 0; it < 100; ++it) {
    double yn = (gp > 0.0) ? y - g / gp : (g < 0.0 ? hi : lo);
    bool newton = true;
    if (!(yn > lo && yn < hi)) {
      newton = false;
      if (g < 0.0 && hi_unv) {   // heading out through b: is the bracket well-posed?
        double fb, dfb;
        growth_fd(b, rd3, krd3, Dc, Kc, c, fb, dfb);
        ++n_eval;
        const double gb = b - y0 - dtp * fb;
        if (gb == 0.0) return b;
        if (gb < 0.0) { n_ill += (b - a > 1e-9 * b); return 0.5 * (a + b); }   // :579; counted when wider than noise
        hi_unv = false;
      } else if (g > 0.0 && lo_unv) {
        double fa, dfa;
        growth_fd(a, rd3, krd3, Dc, Kc, c, fa, dfa);
        ++n_eval;
        const double ga = a - y0 - dtp * fa;
        if (ga == 0.0) return a;
        if (ga > 0.0) { n_ill += (b - a > 1e-9 * b); return 0.5 * (a + b); }
        lo_unv = false;
      }
      yn = 0.5 * (lo + hi);
    }
    const double step = fabs(yn - y);
    y = yn;
    // a Newton step this small leaves an error of order step^2/y; a bisection step bounds it directly
    if (step <= (newton ? 1e-9 : 2e-16) * y) break;
    if (!(hi - lo > 1e-15 * hi)) break;
    growth_fd(y, rd3, krd3, Dc, Kc, c, f, df);
    ++n_eval;
    g = y - y0 - dtp * f;
    gp = 1.0 - dtp * df;
    if (g == 0.0) break;
    if (g < 0.0) { lo = y; lo_unv = false; } else { hi = y; hi_unv = false; }
  }
  return y;
}

// Shared memory per group: cap x {dn, rw2, rd3, kappa*rd3, rd2} doubles.
template <int G, bool SMEM>
__global__ void __launch_bounds__(CtaOf<G>::threads) k_cond(SdArrays a, const u16* __restrict__ rank,
                                                            const u32* __restrict__ seg, Grid g, Field th_f, Field rv_f,
                                                            CellFields cf, CondParams cp, Counters cnt, int cap) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NG = CtaOf<G>::threads / G;
  __shared__ double red_scratch[32];
  const int gi = threadIdx.x / G;
  const Group<G> grp = make_group<G>(red_scratch);
  const int c = blockIdx.x * NG + gi;
  unsigned n_ill = 0, n_eval = 0, n_sub = 0;
  if (c < g.ncell) {
    double* sm = reinterpret_cast<double*>(smem_raw) + (size_t)gi * cap * 5;
    double* s_dn = sm;
    double* s_y = sm + cap;
    double* s_rd3 = sm + 2 * cap;
    double* s_krd3 = sm + 3 * cap;
    double* s_rd2 = sm + 4 * cap;
    const u32 s0 = seg[c];
    const int m = (int)(seg[c + 1] - s0);
    const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
    double th = th_f.at(i, j, k), rv = rv_f.at(i, j, k);
    const double rhod = cf.rhod[c];
    const double c_exn = pow(rhod * cst::R_d / cst::p_1000, cst::R_d / cst::c_pd);
    if (m > 0) {
      if constexpr (SMEM) {
        for (int t = grp.lane; t < m; t += G) {
          const int e = rank[s0 + t];
          const double rd3 = a.rd3[s0 + t];
          const double q = cbrt(rd3);
          s_dn[e] = (double)a.n[s0 + t];
          s_y[e] = a.rw2[s0 + t];
          s_rd3[e] = rd3;
          s_krd3[e] = a.kappa[s0 + t] * rd3;
          s_rd2[e] = q * q;
        }
        grp.sync();
      }
      const double fb = -(4.0 * cst::pi * cst::rho_w / 3.0) / (rhod * g.dV);   // eq. 25 prefactor
      for (int sub = 0; sub < cp.sstp; ++sub) {
        const CellC cc = cell_consts(th, rv, rhod, c_exn, cp.RH_max);
        double acc = 0.0;
        for (int e = grp.lane; e < m; e += G) {
          double dn, y0, rd3, krd3, rd2;
          if constexpr (SMEM) {
            dn = s_dn[e]; y0 = s_y[e]; rd3 = s_rd3[e]; krd3 = s_krd3[e]; rd2 = s_rd2[e];
          } else {
            dn = (double)a.n[s0 + e]; y0 = a.rw2[s0 + e]; rd3 = a.rd3[s0 + e];
            krd3 = a.kappa[s0 + e] * rd3;
            const double q = cbrt(rd3);
            rd2 = q * q;
          }
          const double y1 = cond_solve(y0, rd2, rd3, krd3, cc, cp.dtp, n_ill, n_eval);
          ++n_sub;
          acc += dn * (y1 * sqrt(y1) - y0 * sqrt(y0));
          if constexpr (SMEM) s_y[e] = y1; else a.rw2[s0 + e] = y1;
        }
        const double sum = grp.sum(acc);
        const double drv = fb * sum;                                          // eq. 25
        const double dth = drv * (-th * cc.lv / (cst::c_pd * cc.T));          // eq. 26, old theta and T
        rv += drv;
        th += dth;
      }
      if constexpr (SMEM) {
        grp.sync();
        for (int t = grp.lane; t < m; t += G) a.rw2[s0 + t] = s_y[rank[s0 + t]];
      }
    }
    if (grp.lane == 0) {
      th_f.at(i, j, k) = th;
      rv_f.at(i, j, k) = rv;
      // air properties after the feedback, used by coalescence and sedimentation (v_term)
      const double T = pow(th * c_exn, cst::c_pd / (cst::c_pd - cst::R_d));
      cf.eta[c] = eta_air(T);
      cf.rho_a[c] = rhod * (1.0 + rv);
    }
  }
  // counters: one atomic per warp and counter, spread over NSLOT addresses
  unsigned v0 = n_ill, v1 = n_eval, v2 = n_sub;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    v0 += __shfl_xor_sync(0xffffffffu, v0, d);
    v1 += __shfl_xor_sync(0xffffffffu, v1, d);
    v2 += __shfl_xor_sync(0xffffffffu, v2, d);
  }
  if ((threadIdx.x & 31) == 0) {
    const int slot = (blockIdx.x * (CtaOf<G>::threads / 32) + (threadIdx.x >> 5)) & (NSLOT - 1);
    if (v0) atomicAdd(&cnt.ill_posed[slot], (unsigned long long)v0);
    if (v1) atomicAdd(&cnt.f_evals[slot], (unsigned long long)v1);
    if (v2) atomicAdd(&cnt.sd_substeps[slot], (unsigned long long)v2);
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

size_t cond_smem_bytes(int G, int cap) {
  const int NG = (G <= 32 ? 128 : G) / G;
  return (size_t)NG * cap * 5 * sizeof(double);
}

template <int G>
static cudaError_t launch_cond_t(int cap, const SdArrays& a, const u16* rank, const u32* seg, const Grid& g, Field th,
                                 Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt, cudaStream_t st) {
  constexpr int NG = CtaOf<G>::threads / G;
  const int grid = (g.ncell + NG - 1) / NG;
  if (cap > 0) {
    const size_t smem = cond_smem_bytes(G, cap);
    cudaError_t e = cudaFuncSetAttribute(k_cond<G, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_cond<G, true><<<grid, CtaOf<G>::threads, smem, st>>>(a, rank, seg, g, th, rv, cf, cp, cnt, cap);
  } else {
    k_cond<G, false><<<grid, CtaOf<G>::threads, 0, st>>>(a, rank, seg, g, th, rv, cf, cp, cnt, 0);
  }
  return cudaGetLastError();
}

cudaError_t launch_cond(int G, int cap, const SdArrays& a, const u16* rank, const u32* seg, const Grid& g, Field th,
                        Field rv, const CellFields& cf, const CondParams& cp, const Counters& cnt, cudaStream_t st) {
  switch (G) {
    case 4: return launch_cond_t<4>(cap, a, rank, seg, g, th, rv, cf, cp, cnt, st);
    case 8: return launch_cond_t<8>(cap, a, rank, seg, g, th, rv, cf, cp, cnt, st);
    case 16: return launch_cond_t<16>(cap, a, rank, seg, g, th, rv, cf, cp, cnt, st);
    case 32: return launch_cond_t<32>(cap, a, rank, seg, g, th, rv, cf, cp, cnt, st);
    default: return launch_cond_t<256>(cap, a, rank, seg, g, th, rv, cf, cp, cnt, st);
  }
}

void launch_thermo(const Grid& g, Field th, Field rv, const CellFields& cf, cudaStream_t st) {
  k_thermo<<<(g.ncell + 127) / 128, 128, 0, st>>>(g, th, rv, cf);
}

}  // namespace sdm
