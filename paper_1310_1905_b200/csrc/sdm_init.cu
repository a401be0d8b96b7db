// init() of PAPER.md Listing 5.5 (:759-766): the initialisation of section 5.1.6 (:653-665) on the device.
// DESIGN.md reading R-init: positions uniform in the Lagrangian domain (:655), ln r_d uniform between the
// automatic limits of :657 (found on the host, sdm_init_ranges), multiplicity from the dry spectrum at STP scaled
// by rho_d / rho_STP (:659), wet radius in Koehler equilibrium with min(RH, 0.95) (:661-665).  Random numbers:
// Philox-4x32-10, counter (id, 0, 0, tag), tags 2..5 = x, y, z, ln r_d.  Compiled with -fmad=false so that
// positions (hence cell indices) are the plain IEEE expressions of the definition.
#include "sdm_kernels.cuh"
#include <cmath>
#include <vector>

namespace sdm {

enum : u32 { TAG_INIT_X = 2, TAG_INIT_Y = 3, TAG_INIT_Z = 4, TAG_INIT_LNR = 5 };

__device__ __forceinline__ double init_uniform(u32 id, u32 tag, u32 k0, u32 k1) {
  u32 a, b;
  philox4x32_10(id, 0u, 0u, tag, k0, k1, a, b);
  const u64 w = ((u64)a << 32) | b;
  return ((double)(w >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

// n(ln r_d) of spectrum g at STP: sum of its lognormal modes (eq. 3 :119)
__host__ __device__ inline double spectrum_density(const InitParams& ip, int g, double lnr) {
  double out = 0.0;
  for (int m = 0; m < ip.n_modes; ++m) {
    if (ip.mode_spectrum[m] != g) continue;
    const double d = lnr - ip.mode_lnr[m];
    out += ip.mode_amp[m] * exp(-(d * d) / ip.mode_2ls2[m]);
  }
  return out;
}

// per cell: RH the SDs are brought to equilibrium with, and the Kelvin length A (Table 2 :1056)
__global__ void k_init_cells(Grid g, Field th_f, Field rv_f, const double* __restrict__ rhod, double* __restrict__ RHeq,
                             double* __restrict__ Akel) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.ncell) return;
  const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
  const double th = th_f.at(i, j, k), rv = rv_f.at(i, j, k), rd = rhod[c];
  const double T = T_of(th, rd);
  const double ca = (cst::l_v0 + (cst::c_l - cst::c_pv) * cst::T_0) / cst::R_v;
  const double cb = (cst::c_l - cst::c_pv) / cst::R_v;
  const double pvs = cst::p_vs0 * exp(ca * (1.0 / cst::T_0 - 1.0 / T) - cb * log(T / cst::T_0));   // [L]
  const double rho_vs = pvs / (cst::R_v * T);
  RHeq[c] = fmin(rv * rd / rho_vs, 0.95);                                     // :665
  Akel[c] = 2.0 * cst::sigma_w / (cst::R_v * T * cst::rho_w);
}

template <typename R>
__global__ void __launch_bounds__(256) k_init_sd(SdArraysT<R> a, u32 N, Grid g, InitParams ip, const double* __restrict__ rhod,
                                                 const double* __restrict__ RHeq, const double* __restrict__ Akel) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int sp = (int)(i % (u32)ip.n_spectra);
  double x = 0.0, y = 0.0, z = 0.0;
  // (the stored value, rounded to R, is the position: the cell below is the cell of what is stored)
  if (g.hx) { x = (R)(ip.x0 + init_uniform(i, TAG_INIT_X, ip.seed_lo, ip.seed_hi) * (ip.x1 - ip.x0)); a.x[i] = (R)x; }
  if (g.hy) { y = (R)(ip.y0 + init_uniform(i, TAG_INIT_Y, ip.seed_lo, ip.seed_hi) * (ip.y1 - ip.y0)); a.y[i] = (R)y; }
  if (g.hz) { z = (R)(ip.z0 + init_uniform(i, TAG_INIT_Z, ip.seed_lo, ip.seed_hi) * (ip.z1 - ip.z0)); a.z[i] = (R)z; }
  const double lo = ip.lnr_lo[sp], hi = ip.lnr_hi[sp];
  const double lnr = lo + (hi - lo) * init_uniform(i, TAG_INIT_LNR, ip.seed_lo, ip.seed_hi);
  const double rd3 = (R)exp(3.0 * lnr);
  const double kappa = ip.kappa[sp];
  const u32 c = cell_of(g, x, y, z);
  const double mult = spectrum_density(ip, sp, lnr) * (hi - lo) / ip.sd_conc_spectrum * g.dV * (rhod[c] / ip.rho_stp);
  a.n[i] = (u64)fmax(1.0, floor(mult + 0.5));
  a.rd3[i] = rd3;
  a.kappa[i] = kappa;
  a.id[i] = i;
  // equilibrium wet radius: a_w(r) exp(A/r) = RH on the rising branch of the Koehler curve, r_d < r < r_crit
  const double A = Akel[c], RH = RHeq[c];
  double rl = cbrt(rd3), rh = sqrt(3.0 * kappa * rd3 / A);
  if (rh > rl) {
    for (int it = 0; it < 300 && rh - rl > 1e-15 * rh; ++it) {
      const double r = 0.5 * (rl + rh), r3 = r * r * r;
      const double S = (r3 - rd3) / (r3 - rd3 * (1.0 - kappa)) * exp(A / r);
      if (S < RH) rl = r; else rh = r;
    }
    rl = 0.5 * (rl + rh);
  }
  a.rw2[i] = rl * rl;
}

// Host: group the modes into spectra by kappa and find the limits of :657 for each.  The density does not
// depend on the limits, so it is tabulated once on the grid; the limits then follow from a threshold that
// depends on the width of the range: iterate to the fixed point.
int init_prepare(const sdm_mode_view* modes, int n_modes, double sd_conc_mean, double dV, InitParams& ip) {
  if (n_modes < 1 || n_modes > INIT_MAX_MODES) return -1;
  ip.n_modes = n_modes;
  ip.n_spectra = 0;
  for (int m = 0; m < n_modes; ++m) {
    if (!(modes[m].n_stp > 0) || !(modes[m].r_mean > 0) || !(modes[m].sigma_g > 1.0) || !(modes[m].kappa > 0)) return -1;
    int sp = -1;
    for (int q = 0; q < ip.n_spectra; ++q) if (ip.kappa[q] == modes[m].kappa) sp = q;
    if (sp < 0) { sp = ip.n_spectra++; ip.kappa[sp] = modes[m].kappa; }
    ip.mode_spectrum[m] = sp;
    const double ls = std::log(modes[m].sigma_g);
    ip.mode_lnr[m] = std::log(modes[m].r_mean);
    ip.mode_amp[m] = modes[m].n_stp / (std::sqrt(2.0 * 3.14159265358979323846) * ls);
    ip.mode_2ls2[m] = 2.0 * ls * ls;
  }
  ip.sd_conc_spectrum = sd_conc_mean / ip.n_spectra;
  ip.rho_stp = 101325.0 / (287.0 * 293.15);   // :130, R_d of DESIGN.md R-const
  const int NGRID = 200001;
  const double g0 = std::log(1e-10), g1 = std::log(1e-4);
  std::vector<double> dens(NGRID);
  for (int sp = 0; sp < ip.n_spectra; ++sp) {
    for (int q = 0; q < NGRID; ++q) dens[q] = spectrum_density(ip, sp, g0 + (g1 - g0) * ((double)q / (double)(NGRID - 1)));
    double lo = std::log(1e-9), hi = std::log(1e-5);
    for (int it = 0; it < 50; ++it) {
      int first = 0, last = NGRID - 1;
      while (first < NGRID && !(dens[first] * (hi - lo) / ip.sd_conc_spectrum * dV >= 1.0)) ++first;
      while (last >= 0 && !(dens[last] * (hi - lo) / ip.sd_conc_spectrum * dV >= 1.0)) --last;
      if (first > last) return -2;   // nowhere does an SD stand for at least one particle
      const double nlo = g0 + (g1 - g0) * ((double)first / (double)(NGRID - 1));
      const double nhi = g0 + (g1 - g0) * ((double)last / (double)(NGRID - 1));
      const bool done = std::fabs(nlo - lo) + std::fabs(nhi - hi) < 1e-9;
      lo = nlo; hi = nhi;
      if (done) break;
    }
    ip.lnr_lo[sp] = lo; ip.lnr_hi[sp] = hi;
  }
  return 0;
}

template <typename R>
void launch_init(const SdArraysT<R>& a, u32 N, const Grid& g, const InitParams& ip, Field th, Field rv, const double* rhod,
                 double* RHeq, double* Akel, cudaStream_t st) {
  k_init_cells<<<(g.ncell + 127) / 128, 128, 0, st>>>(g, th, rv, rhod, RHeq, Akel);
  if (N) k_init_sd<R><<<(N + 255) / 256, 256, 0, st>>>(a, N, g, ip, rhod, RHeq, Akel);
}

#define SDM_INST(R)                                                                                              \
  template void launch_init<R>(const SdArraysT<R>&, u32, const Grid&, const InitParams&, Field, Field, const double*, \
                               double*, double*, cudaStream_t);
SDM_INSTANTIATE_REAL(SDM_INST)
#undef SDM_INST

}  // namespace sdm
