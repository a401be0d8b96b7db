// ORACLE (test infrastructure, not the product): a plain, slow, serial-by-
// default fp64 CPU implementation of one super-droplet time step of the
// particle-based scheme of arxiv 1310.1905 (section 5.1), in the
// paper's order and notation.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may use it.  It shares no
// code with the CUDA path (paper_1310_1905_b200/csrc).
//
// Step order (PAPER.md :620, :641, :816; reading R-order):
//   [recycle N=0 ->] compact N=0 -> cell index + shuffle key -> sort (cell,key,id)
//   -> condensation x sstp_cond -> coalescence x sstp_coal -> advection+sedimentation
//
// Pins (tests/test_oracle_pins.py): Philox known answers; Golovin closed form;
// brute-force pair statistics; conservation of sum n r^3; Koehler closed forms;
// water conservation; eq. 13-15 residual; Stokes limit; brute-force moments.
// "parity unpinned" against the paper (forms not printed there, see
// formulae.h [L] tags): D_0, K_0, eta(T), Sh/Nu, beta forms, p_vs(T) form,
// kappa averaging rule, collision-efficiency table values.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC sdm_oracle.cpp -o liboracle.so
#include "formulae.h"
#include <vector>
#include <numeric>
#include <cstring>
#include <cstdio>
#ifdef _OPENMP
#include <omp.h>
#endif

using namespace orc;
typedef uint64_t u64;
typedef uint32_t u32;

extern "C" {
struct orc_init_t {
  int nx, ny, nz;            // 0 = dimension absent (PAPER.md :751 "zero (parcel) up to three")
  double dx, dy, dz, dt;     // absent dimensions still contribute their length to dV
  int kernel;                // 0 geometric (eq. 28, E=1), 1 golovin, 2 hydro_tab (eq. 28 with tabulated E)
  double golovin_b;
  int multi_coal;            // 1: gamma = floor(p) + [u < frac p]; 0: paper :645 (gamma = [u < p])
  u64 seed;
  int n_eff_R, n_eff_q;      // collision-efficiency table axes lengths
  const double* eff_R;       // collector radius axis [m], ascending
  const double* eff_q;       // radius ratio axis (small/large), ascending
  const double* eff_tab;     // [n_eff_R][n_eff_q]
};
struct orc_opts_t {          // PAPER.md Listing 5.1 (:677-689)
  int adve, sedi, cond, coal;
  double RH_max;
  int sstp_cond, sstp_coal;
  double cond_adapt_tol;     // > 0: per-cell number of condensation substeps (reading R-adapt; PAPER.md :566 "planned")
  int coal_adapt_max;        // > 1: per-cell number of coalescence substeps from P_ij (reading R-adapt-coal; PAPER.md :645 "planned")
};
struct orc_counters_t {
  long long pairs, collisions, near_ties, ill_posed, f_evals, sd_substeps;
};
}

enum { TAG_SHUFFLE = 0, TAG_COAL = 1 };

struct Ctx {
  orc_init_t o;
  std::vector<double> effR, effq, efftab;
  int NX, NY, NZ; long ncell;
  double dV;
  // particle state (SoA)
  std::vector<u64> n; std::vector<double> rw2, rd3, kappa, x, y, z; std::vector<u32> id;
  // per-step scratch
  std::vector<u32> cell, key; std::vector<long> order; std::vector<long> seg;   // seg[ncell+1]
  // Eulerian fields, dense C order (i,j,k), k fastest
  std::vector<double> th, rv, rhod, cx, cy, cz;
  std::vector<CellThermo> thermo;   // after condensation feedback, for v_term
  u32 step = 0;
  double rain_flux_step = 0, rain_flux_total = 0;
  orc_counters_t cnt{};
  int nthreads = 1;
  bool sorted = false;
  int recycle = 0;            // 1: PAPER.md :641 recycling of zero-multiplicity SDs before the compaction
  long long recycled = 0;     // SDs recycled so far
};

static inline u32 shuffle_key(const Ctx& c, u32 id, u32 step, u32 sub) {
  u32 ctr[4] = {id, step, sub, TAG_SHUFFLE}, k[2] = {(u32)c.o.seed, (u32)(c.o.seed >> 32)}, out[4];
  philox4x32_10(ctr, k, out);
  return out[0];
}
static inline double coal_uniform(const Ctx& c, u32 id_first, u32 step, u32 sub) {
  // u in (0,1): PAPER.md :639 "uniform distribution over the (0,1) interval"
  u32 ctr[4] = {id_first, step, sub, TAG_COAL}, k[2] = {(u32)c.o.seed, (u32)(c.o.seed >> 32)}, out[4];
  philox4x32_10(ctr, k, out);
  const u64 w = ((u64)out[0] << 32) | out[1];
  return ((double)(w >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

// PAPER.md :547 (eq. 15): index of the cell containing coordinate x
static inline int cell_1d(double x, double dx, int n) {
  int i = (int)std::floor(x / dx);
  if (i < 0) i = 0;
  if (i > n - 1) i = n - 1;
  return i;
}

static void compute_cells(Ctx& c) {
  const long N = (long)c.n.size();
  c.cell.resize(N);
  for (long s = 0; s < N; ++s) {
    const int i = c.o.nx > 0 ? cell_1d(c.x[s], c.o.dx, c.NX) : 0;
    const int j = c.o.ny > 0 ? cell_1d(c.y[s], c.o.dy, c.NY) : 0;
    const int k = c.o.nz > 0 ? cell_1d(c.z[s], c.o.dz, c.NZ) : 0;
    c.cell[s] = (u32)(((long)i * c.NY + j) * c.NZ + k);
  }
}

// stable removal of zero-multiplicity SDs (BASELINE.json "zero-multiplicity stream compaction")
static void compact(Ctx& c) {
  const long N = (long)c.n.size();
  long w = 0;
  for (long s = 0; s < N; ++s) {
    if (c.n[s] == 0) continue;
    if (w != s) {
      c.n[w] = c.n[s]; c.rw2[w] = c.rw2[s]; c.rd3[w] = c.rd3[s]; c.kappa[w] = c.kappa[s];
      c.x[w] = c.x[s]; c.y[w] = c.y[s]; c.z[w] = c.z[s]; c.id[w] = c.id[s];
    }
    ++w;
  }
  c.n.resize(w); c.rw2.resize(w); c.rd3.resize(w); c.kappa.resize(w);
  c.x.resize(w); c.y.resize(w); c.z.resize(w); c.id.resize(w);
}

// PAPER.md :641 "Particles with zero multiplicity are 'recycled' at the begining of each timestep.  The recycling
// procedure first looks for computational particles with highest multiplicites and then assignes their properties
// to the recycled particles halving the multiplicity"; :651 the same for SDs that left the domain.
// DESIGN.md reading R-recycle: with k SDs of zero multiplicity, the donors are the k SDs first in the order
// (multiplicity descending, id ascending) among those with multiplicity >= 2 (one real particle cannot be halved;
// fewer donors than k: the zero-multiplicity SDs of highest id stay dead and are compacted away); the i-th donor
// serves the zero-multiplicity SD of i-th smallest id, which takes the donor's r_w^2, r_d^3, kappa and position,
// keeps its own id (its random streams stay its own) and gets floor(N/2); the donor keeps N - floor(N/2).
// The selection is made once, from the multiplicities before any halving.
static void recycle(Ctx& c) {
  const long N = (long)c.n.size();
  std::vector<long> dead, donors;
  for (long s = 0; s < N; ++s) {
    if (c.n[s] == 0) dead.push_back(s);
    else if (c.n[s] >= 2) donors.push_back(s);
  }
  if (dead.empty() || donors.empty()) return;
  std::sort(dead.begin(), dead.end(), [&](long a, long b) { return c.id[a] < c.id[b]; });
  std::sort(donors.begin(), donors.end(), [&](long a, long b) {
    if (c.n[a] != c.n[b]) return c.n[a] > c.n[b];
    return c.id[a] < c.id[b];
  });
  const long k = (long)std::min(dead.size(), donors.size());
  for (long i = 0; i < k; ++i) {
    const long d = dead[i], s = donors[i];
    const u64 half = c.n[s] / 2;
    c.rw2[d] = c.rw2[s]; c.rd3[d] = c.rd3[s]; c.kappa[d] = c.kappa[s];
    c.x[d] = c.x[s]; c.y[d] = c.y[s]; c.z[d] = c.z[s];
    c.n[d] = half;
    c.n[s] -= half;
  }
  c.recycled += k;
}

// PAPER.md :624 "randomly grouped into non-overlapping pairs": the random grouping
// is the order of the SDs of a cell under the total order (cell, key, id).
static void sort_stage(Ctx& c) {
  if (c.recycle) recycle(c);
  compact(c);
  compute_cells(c);
  const long N = (long)c.n.size();
  c.key.resize(N);
  for (long s = 0; s < N; ++s) c.key[s] = shuffle_key(c, c.id[s], c.step, 0);
  c.order.resize(N);
  std::iota(c.order.begin(), c.order.end(), 0L);
  std::sort(c.order.begin(), c.order.end(), [&](long a, long b) {
    if (c.cell[a] != c.cell[b]) return c.cell[a] < c.cell[b];
    if (c.key[a] != c.key[b]) return c.key[a] < c.key[b];
    return c.id[a] < c.id[b];
  });
  c.seg.assign(c.ncell + 1, 0);
  for (long s = 0; s < N; ++s) c.seg[c.cell[s] + 1]++;
  for (long q = 0; q < c.ncell; ++q) c.seg[q + 1] += c.seg[q];
  c.sorted = true;
}

// PAPER.md :560-618: condensation substeps with feedback on r_v, theta (eq. 25-26)
// DESIGN.md reading R-adapt (PAPER.md :566: "the actual constraints for timestep length differ substantially, particularly
// with the distance from cloud base.  An adaptive timestep choice mechanism is planned"): the number of condensation
// substeps of a cell in this step.  What the substeps resolve is the explicit coupling of eq. 17 to r_v and theta, so the
// measure is how far the cell's own condensation would move its supersaturation in one step:
//   eps = |d r_v| / (r_v max(|RH - 1|, 1e-3)),  d r_v = eq. 25 with d(r_w^3) = (3/2) r_w dt f(y) at the start of the step
// (eq. 20 with the cell's thermodynamics and the ventilation of the SD's own radius).  The cell takes the smallest divisor d
// of sstp_cond with d >= sstp_cond eps / tol (eps >= tol: all sstp_cond substeps; haze in equilibrium: one).
static int adaptive_substeps(const Ctx& c, long q, const orc_opts_t& op) {
  const CellThermo ct = cell_thermo(c.th[q], c.rv[q], c.rhod[q], op.RH_max);
  double est = 0.0;   // sum_i N_i (3/2) r_i dt f_i, sorted order
  for (long p = c.seg[q]; p < c.seg[q + 1]; ++p) {
    const long i = c.order[p];
    const double y0 = c.rw2[i], r0 = std::sqrt(y0);
    const double vt = v_term(r0, ct.eta, ct.rho_a);
    const double Re = 2.0 * r0 * vt * ct.rho_a / ct.eta;
    const double f0 = growth_f(y0, c.rd3[i], c.kappa[i], ct, vent(Re, ct.Sc), vent(Re, ct.Pr));
    est += (double)c.n[i] * (1.5 * r0 * (c.o.dt * f0));
  }
  const double drv = (4.0 * pi * rho_w / 3.0) / (c.rhod[q] * c.dV) * std::fabs(est);
  const double eps = drv / (c.rv[q] * std::max(std::fabs(ct.RH - 1.0), 1e-3));
  const double want = op.sstp_cond * eps / op.cond_adapt_tol;
  for (int d = 1; d < op.sstp_cond; ++d)
    if (op.sstp_cond % d == 0 && (double)d >= want) return d;
  return op.sstp_cond;
}

static void cond_stage(Ctx& c, const orc_opts_t& op) {
  long long ill = 0, fev = 0, sds = 0;
#pragma omp parallel for schedule(dynamic, 16) num_threads(c.nthreads) reduction(+ : ill, fev, sds)
  for (long q = 0; q < c.ncell; ++q) {
    const long s0 = c.seg[q], s1 = c.seg[q + 1];
    const int nsub = op.cond_adapt_tol > 0.0 ? adaptive_substeps(c, q, op) : op.sstp_cond;
    const double dtp = c.o.dt / nsub;
    for (int sub = 0; sub < nsub; ++sub) {
      const CellThermo ct = cell_thermo(c.th[q], c.rv[q], c.rhod[q], op.RH_max);
      double sum = 0.0;   // sum_i N_i (r_w^3 new - r_w^3 old), sorted order, plain fp64
      for (long p = s0; p < s1; ++p) {
        const long i = c.order[p];
        const double y0 = c.rw2[i];
        int ip = 0; long ne = 0;
        const double y1 = cond_substep_sd(y0, c.rd3[i], c.kappa[i], ct, dtp, &ip, &ne);
        ill += ip; fev += ne; ++sds;
        sum += (double)c.n[i] * (y1 * std::sqrt(y1) - y0 * std::sqrt(y0));
        c.rw2[i] = y1;
      }
      // eq. 25
      const double drv = -(4.0 * pi * rho_w / 3.0) / (c.rhod[q] * c.dV) * sum;
      // eq. 26 with d theta / d r_v = -theta l_v / (c_pd T) (:195), old theta and T
      const double dth = drv * (-c.th[q] * ct.lv / (c_pd * ct.T));
      c.rv[q] += drv;
      c.th[q] += dth;
    }
  }
  c.cnt.ill_posed += ill; c.cnt.f_evals += fev; c.cnt.sd_substeps += sds;
}

static void thermo_stage(Ctx& c, const orc_opts_t& op) {
  c.thermo.resize(c.ncell);
  for (long q = 0; q < c.ncell; ++q) c.thermo[q] = cell_thermo(c.th[q], c.rv[q], c.rhod[q], op.RH_max);
}

// collision efficiency: bilinear in (collector radius, ratio), clamped at the table edges
static double eff_lookup(const Ctx& c, double R, double q) {
  const int nR = c.o.n_eff_R, nq = c.o.n_eff_q;
  const double* aR = c.effR.data(); const double* aq = c.effq.data(); const double* tab = c.efftab.data();
  R = std::min(std::max(R, aR[0]), aR[nR - 1]);
  q = std::min(std::max(q, aq[0]), aq[nq - 1]);
  int iR = (int)(std::upper_bound(aR, aR + nR, R) - aR) - 1; iR = std::min(std::max(iR, 0), nR - 2);
  int iq = (int)(std::upper_bound(aq, aq + nq, q) - aq) - 1; iq = std::min(std::max(iq, 0), nq - 2);
  const double t = (R - aR[iR]) / (aR[iR + 1] - aR[iR]);
  const double s = (q - aq[iq]) / (aq[iq + 1] - aq[iq]);
  const double e00 = tab[iR * nq + iq], e01 = tab[iR * nq + iq + 1];
  const double e10 = tab[(iR + 1) * nq + iq], e11 = tab[(iR + 1) * nq + iq + 1];
  return (1.0 - t) * ((1.0 - s) * e00 + s * e01) + t * ((1.0 - s) * e10 + s * e11);
}

// collection kernel K(r_j, r_k) [m^3/s]
static double coal_kernel(const Ctx& c, long j, long k, const CellThermo& ct) {
  const double rj = std::sqrt(c.rw2[j]), rk = std::sqrt(c.rw2[k]);
  if (c.o.kernel == 1) {   // Golovin K = b (v_j + v_k) (BASELINE.json configs[0])
    const double vj = (4.0 / 3.0) * pi * (c.rw2[j] * rj), vk = (4.0 / 3.0) * pi * (c.rw2[k] * rk);
    return c.o.golovin_b * (vj + vk);
  }
  // eq. 28: K = E pi (r_j + r_k)^2 |v_j - v_k|
  const double vj = v_term(rj, ct.eta, ct.rho_a), vk = v_term(rk, ct.eta, ct.rho_a);
  double K = pi * ((rj + rk) * (rj + rk)) * std::fabs(vj - vk);
  if (c.o.kernel == 2) {
    const double rl = std::max(rj, rk), rs = std::min(rj, rk);
    K = K * eff_lookup(c, rl, rs / rl);
  }
  return K;
}

// PAPER.md :622-645: SDM coalescence on the pairs (0,1),(2,3).. of each cell's sorted segment
// DESIGN.md reading R-adapt-coal (PAPER.md :645: "It is planned ... to use the values of P_ij to control an adaptive timestep
// logic"): with P_max the largest probability of eq. 27 among the pairs of the cell's first grouping, for the substep length
// dt / sstp_coal, the cell takes sstp_coal * m substeps, m = min(coal_adapt_max, ceil(P_max)) (at least 1): just enough for
// every pair of that grouping to have P <= 1, where an event stands for one collision per pair of real droplets.
static int coal_substep_multiplier(const Ctx& c, const std::vector<long>& L, const CellThermo& ct, const orc_opts_t& op) {
  const u64 nc = L.size();
  if (op.coal_adapt_max <= 1 || nc < 2) return 1;
  const double dtpp = c.o.dt / op.sstp_coal;
  const double scale = (double)(nc * (nc - 1) / 2) / (double)(nc / 2);
  double pmax = 0.0;
  for (u64 m = 0; m + 1 < nc; m += 2) {
    const long a = L[m], b = L[m + 1];
    long j, k;
    if (c.n[a] >= c.n[b]) { j = a; k = b; } else { j = b; k = a; }
    const double p = (((double)c.n[j] * coal_kernel(c, j, k, ct)) * (dtpp / c.dV)) * scale;
    pmax = std::max(pmax, p);
  }
  const double want = std::ceil(pmax);
  if (want >= (double)op.coal_adapt_max) return op.coal_adapt_max;
  return std::max(1, (int)want);
}

static void coal_stage(Ctx& c, const orc_opts_t& op) {
  if ((long)c.thermo.size() != c.ncell) thermo_stage(c, op);
  long long pairs = 0, colls = 0, ties = 0;
#pragma omp parallel for schedule(dynamic, 16) num_threads(c.nthreads) reduction(+ : pairs, colls, ties)
  for (long q = 0; q < c.ncell; ++q) {
    std::vector<long> L(c.order.begin() + c.seg[q], c.order.begin() + c.seg[q + 1]);
    const CellThermo& ct = c.thermo[q];
    const int nsub = op.sstp_coal * coal_substep_multiplier(c, L, ct, op);
    const double dtpp = c.o.dt / nsub;
    for (int sub = 0; sub < nsub; ++sub) {
      if (sub > 0) {   // new random grouping each substep (:624); SDs at N=0 drop out
        std::vector<long> M; M.reserve(L.size());
        for (long i : L) if (c.n[i] > 0) M.push_back(i);
        L.swap(M);
        std::vector<std::pair<u32, long>> kk; kk.reserve(L.size());
        for (long i : L) kk.push_back({shuffle_key(c, c.id[i], c.step, (u32)sub), i});
        std::sort(kk.begin(), kk.end(), [&](const std::pair<u32, long>& a, const std::pair<u32, long>& b) {
          if (a.first != b.first) return a.first < b.first;
          return c.id[a.second] < c.id[b.second];
        });
        for (size_t m = 0; m < L.size(); ++m) L[m] = kk[m].second;
      }
      const u64 nc = L.size();
      if (nc < 2) continue;
      // eq. 27 last factor: n(n-1)/2 / floor(n/2)
      const double scale = (double)(nc * (nc - 1) / 2) / (double)(nc / 2);
      for (u64 m = 0; m + 1 < nc; m += 2) {
        const long a = L[m], b = L[m + 1];
        long j, k;   // j: larger multiplicity; tie -> first in sorted order
        if (c.n[a] >= c.n[b]) { j = a; k = b; } else { j = b; k = a; }
        const double K = coal_kernel(c, j, k, ct);
        const double p = (((double)c.n[j] * K) * (dtpp / c.dV)) * scale;   // eq. 27
        const double u = coal_uniform(c, c.id[a], c.step, (u32)sub);
        const u64 qmax = c.n[j] / c.n[k];
        u64 g;
        if (c.o.multi_coal) {
          const double pf = std::floor(p);
          if (pf >= (double)qmax) g = qmax;
          else {
            const double frac = p - pf;
            if (std::fabs(u - frac) < 1e-12) ++ties;
            g = (u64)pf + (u < frac ? 1u : 0u);
            if (g > qmax) g = qmax;
          }
        } else {
          if (std::fabs(u - p) < 1e-12) ++ties;
          g = (u < p) ? 1u : 0u;   // :639 event iff P > u; :645 no multiple coalescence
        }
        ++pairs;
        if (g == 0) continue;
        ++colls;
        // g n_k droplets of j merge with the n_k droplets of k (:639-643, Shima 2009)
        const double gd = (double)g;
        const double rj = std::sqrt(c.rw2[j]), rk = std::sqrt(c.rw2[k]);
        const double rw3 = c.rw2[k] * rk + gd * (c.rw2[j] * rj);   // extensive: summed (:643)
        const double rd3j = gd * c.rd3[j];
        if (c.kappa[j] != c.kappa[k])                               // intensive: averaged (:643)
          c.kappa[k] = (rd3j * c.kappa[j] + c.rd3[k] * c.kappa[k]) / (rd3j + c.rd3[k]);
        c.rd3[k] = c.rd3[k] + rd3j;
        const double r = std::cbrt(rw3);
        c.rw2[k] = r * r;
        c.n[j] -= g * c.n[k];
      }
    }
  }
  c.cnt.pairs += pairs; c.cnt.collisions += colls; c.cnt.near_ties += ties;
}

static inline double wrap(double x, double X) {
  if (x < 0.0) x += X;
  if (x >= X) x -= X;
  return x;
}

// PAPER.md :534-558 advection (eq. 16), :647-651 sedimentation
static void move_stage(Ctx& c, const orc_opts_t& op) {
  if ((long)c.thermo.size() != c.ncell) thermo_stage(c, op);
  const long N = (long)c.n.size();
  const bool hx = c.o.nx > 0, hy = c.o.ny > 0, hz = c.o.nz > 0;
  const double X = c.o.dx * c.NX, Y = c.o.dy * c.NY, Z = c.o.dz * c.NZ;
  double flux = 0.0;
  for (long p = 0; p < N; ++p) {
    const long s = c.order[p];
    if (c.n[s] == 0) continue;
    const long q = c.cell[s];
    const int k = (int)(q % c.NZ), j = (int)((q / c.NZ) % c.NY), i = (int)(q / ((long)c.NZ * c.NY));
    const double rhod = c.rhod[q];
    double xn = c.x[s], yn = c.y[s], zn = c.z[s];
    if (op.adve) {
      if (hx) {   // rhod_courant_1 has shape (nx+1) x ny x nz (:751)
        const double Clo = c.cx[((long)i * c.NY + j) * c.NZ + k] / rhod;
        const double Chi = c.cx[((long)(i + 1) * c.NY + j) * c.NZ + k] / rhod;
        const double dC = Chi - Clo;
        xn = (c.x[s] + c.o.dx * (Clo - (double)i * dC)) / (1.0 - dC);
      }
      if (hy) {
        const double Clo = c.cy[((long)i * (c.NY + 1) + j) * c.NZ + k] / rhod;
        const double Chi = c.cy[((long)i * (c.NY + 1) + j + 1) * c.NZ + k] / rhod;
        const double dC = Chi - Clo;
        yn = (c.y[s] + c.o.dy * (Clo - (double)j * dC)) / (1.0 - dC);
      }
      if (hz) {
        const double Clo = c.cz[((long)i * c.NY + j) * (c.NZ + 1) + k] / rhod;
        const double Chi = c.cz[((long)i * c.NY + j) * (c.NZ + 1) + k + 1] / rhod;
        const double dC = Chi - Clo;
        zn = (c.z[s] + c.o.dz * (Clo - (double)k * dC)) / (1.0 - dC);
      }
    }
    if (op.sedi && hz) {   // explicit Euler (:649)
      const CellThermo& ct = c.thermo[q];
      zn = zn - v_term(std::sqrt(c.rw2[s]), ct.eta, ct.rho_a) * c.o.dt;
    }
    if (hx) xn = wrap(xn, X);   // periodic horizontal boundaries (:558)
    if (hy) yn = wrap(yn, Y);
    if (hz && (zn < 0.0 || !(zn < Z))) {   // left the domain (:651)
      if (zn < 0.0) flux += (double)c.n[s] * ((4.0 / 3.0) * pi * rho_w * (c.rw2[s] * std::sqrt(c.rw2[s])));
      c.n[s] = 0;
    }
    c.x[s] = xn; c.y[s] = yn; c.z[s] = zn;
  }
  c.rain_flux_step = flux;
  c.rain_flux_total += flux;
}

extern "C" {

void* orc_create(const orc_init_t* o) {
  Ctx* c = new Ctx();
  c->o = *o;
  if (o->n_eff_R > 0 && o->eff_R) {
    c->effR.assign(o->eff_R, o->eff_R + o->n_eff_R);
    c->effq.assign(o->eff_q, o->eff_q + o->n_eff_q);
    c->efftab.assign(o->eff_tab, o->eff_tab + (long)o->n_eff_R * o->n_eff_q);
  }
  c->NX = std::max(o->nx, 1); c->NY = std::max(o->ny, 1); c->NZ = std::max(o->nz, 1);
  c->ncell = (long)c->NX * c->NY * c->NZ;
  c->dV = o->dx * o->dy * o->dz;
  c->th.assign(c->ncell, 300.0); c->rv.assign(c->ncell, 0.0); c->rhod.assign(c->ncell, 1.0);
  c->cx.assign((long)(c->NX + 1) * c->NY * c->NZ, 0.0);
  c->cy.assign((long)c->NX * (c->NY + 1) * c->NZ, 0.0);
  c->cz.assign((long)c->NX * c->NY * (c->NZ + 1), 0.0);
  return c;
}
void orc_destroy(void* h) { delete (Ctx*)h; }
void orc_set_threads(void* h, int n) { ((Ctx*)h)->nthreads = std::max(n, 1); }
int orc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void orc_set_state(void* h, long N, const u64* n, const double* rw2, const double* rd3, const double* kappa,
                   const double* x, const double* y, const double* z, const u32* id) {
  Ctx& c = *(Ctx*)h;
  c.n.assign(n, n + N); c.rw2.assign(rw2, rw2 + N); c.rd3.assign(rd3, rd3 + N); c.kappa.assign(kappa, kappa + N);
  if (x) c.x.assign(x, x + N); else c.x.assign(N, 0.0);
  if (y) c.y.assign(y, y + N); else c.y.assign(N, 0.0);
  if (z) c.z.assign(z, z + N); else c.z.assign(N, 0.0);
  c.id.assign(id, id + N);
  c.sorted = false;
}
// dense C-order fields; NULL leaves a field unchanged
void orc_set_fields(void* h, const double* th, const double* rv, const double* rhod,
                    const double* cx, const double* cy, const double* cz) {
  Ctx& c = *(Ctx*)h;
  if (th) c.th.assign(th, th + c.ncell);
  if (rv) c.rv.assign(rv, rv + c.ncell);
  if (rhod) c.rhod.assign(rhod, rhod + c.ncell);
  if (cx) c.cx.assign(cx, cx + c.cx.size());
  if (cy) c.cy.assign(cy, cy + c.cy.size());
  if (cz) c.cz.assign(cz, cz + c.cz.size());
  c.thermo.clear();
}
// ---- initialisation (section 5.1.6 :653-665; init() of Listing 5.5 :759-766) --------------------
// DESIGN.md reading R-init.  modes: n_modes x {kappa, N_stp [m^-3], r_mean [m], sigma_g} (eq. 3 :119); modes
// with the same kappa form one spectrum n(ln r_d), different kappas are an external mixture (:659) whose
// spectra take the SDs in turn (SD i belongs to spectrum i mod G).  Uses the th, rv, rhod set before.
struct Spectrum { double kappa; std::vector<int> modes; double lo, hi; };
static double spectrum_density(const double* modes, const Spectrum& sp, double lnr) {   // n(ln r_d) at STP
  double out = 0.0;
  for (int m : sp.modes) {
    const double N = modes[4 * m + 1], lrm = std::log(modes[4 * m + 2]), ls = std::log(modes[4 * m + 3]);
    out += N / (std::sqrt(2.0 * pi) * ls) * std::exp(-((lnr - lrm) * (lnr - lrm)) / (2.0 * ls * ls));
  }
  return out;
}
// :657 "the particle multiplicity for both the minimal and the maximal radii be greater or equal one": the
// multiplicity at a radius depends on the width of the range, so iterate to the fixed point on a grid in ln r.
static void auto_range(const double* modes, Spectrum& sp, double sd_conc, double dV) {
  const int NG = 200001;
  const double g0 = std::log(1e-10), g1 = std::log(1e-4);
  double lo = std::log(1e-9), hi = std::log(1e-5);
  for (int it = 0; it < 50; ++it) {
    int first = -1, last = -1;
    for (int q = 0; q < NG; ++q) {
      const double lnr = g0 + (g1 - g0) * ((double)q / (double)(NG - 1));
      if (spectrum_density(modes, sp, lnr) * (hi - lo) / sd_conc * dV >= 1.0) { if (first < 0) first = q; last = q; }
    }
    if (first < 0) break;
    const double nlo = g0 + (g1 - g0) * ((double)first / (double)(NG - 1));
    const double nhi = g0 + (g1 - g0) * ((double)last / (double)(NG - 1));
    const bool done = std::fabs(nlo - lo) + std::fabs(nhi - hi) < 1e-9;
    lo = nlo; hi = nhi;
    if (done) break;
  }
  sp.lo = lo; sp.hi = hi;
}
static inline double init_uniform(const Ctx& c, u32 id, u32 tag) {
  u32 ctr[4] = {id, 0u, 0u, tag}, k[2] = {(u32)c.o.seed, (u32)(c.o.seed >> 32)}, out[4];
  philox4x32_10(ctr, k, out);
  const u64 w = ((u64)out[0] << 32) | out[1];
  return ((double)(w >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}
// wet radius in equilibrium with RH (zero on the left of eq. 20, :661): root of a_w(r) exp(A/r) = RH between
// r_d and the critical radius sqrt(3 kappa r_d^3 / A), where the Koehler curve rises monotonically
static double equilibrium_rw(double rd3, double kappa, double RH, double A) {
  double lo = std::cbrt(rd3), hi = std::sqrt(3.0 * kappa * rd3 / A);
  if (!(hi > lo)) return lo;
  for (int it = 0; it < 300 && hi - lo > 1e-15 * hi; ++it) {
    const double r = 0.5 * (lo + hi), r3 = r * r * r;
    const double S = (r3 - rd3) / (r3 - rd3 * (1.0 - kappa)) * std::exp(A / r);
    if (S < RH) lo = r; else hi = r;
  }
  return 0.5 * (lo + hi);
}

long orc_init(void* h, int n_modes, const double* modes, double sd_conc_mean, double x0, double y0, double z0,
              double x1, double y1, double z1, double* ranges_out) {
  Ctx& c = *(Ctx*)h;
  std::vector<Spectrum> sp;
  for (int m = 0; m < n_modes; ++m) {
    size_t g = 0;
    while (g < sp.size() && sp[g].kappa != modes[4 * m]) ++g;
    if (g == sp.size()) sp.push_back(Spectrum{modes[4 * m], {}, 0.0, 0.0});
    sp[g].modes.push_back(m);
  }
  const int G = (int)sp.size();
  const double sd_conc_g = sd_conc_mean / G;
  for (int g = 0; g < G; ++g) {
    auto_range(modes, sp[g], sd_conc_g, c.dV);
    if (ranges_out) { ranges_out[2 * g] = sp[g].lo; ranges_out[2 * g + 1] = sp[g].hi; }
  }
  double ncl = 1.0;
  if (c.o.nx > 0) ncl *= (x1 - x0) / c.o.dx;
  if (c.o.ny > 0) ncl *= (y1 - y0) / c.o.dy;
  if (c.o.nz > 0) ncl *= (z1 - z0) / c.o.dz;
  const long N = (long)std::floor(sd_conc_mean * ncl + 0.5);
  const double rho_stp = 101325.0 / (R_d * 293.15);   // :130 "T = 20 C and p = 1013.25 hPa"
  c.n.assign(N, 0); c.rw2.assign(N, 0.0); c.rd3.assign(N, 0.0); c.kappa.assign(N, 0.0);
  c.x.assign(N, 0.0); c.y.assign(N, 0.0); c.z.assign(N, 0.0); c.id.assign(N, 0u);
  for (long i = 0; i < N; ++i) {
    const Spectrum& s = sp[i % G];
    c.id[i] = (u32)i;
    if (c.o.nx > 0) c.x[i] = x0 + init_uniform(c, (u32)i, 2u) * (x1 - x0);   // :655 uniform in space
    if (c.o.ny > 0) c.y[i] = y0 + init_uniform(c, (u32)i, 3u) * (y1 - y0);
    if (c.o.nz > 0) c.z[i] = z0 + init_uniform(c, (u32)i, 4u) * (z1 - z0);
    const double lnr = s.lo + (s.hi - s.lo) * init_uniform(c, (u32)i, 5u);     // :657 uniform in ln r_d
    c.rd3[i] = std::exp(3.0 * lnr);
    c.kappa[i] = s.kappa;
    const int ci = c.o.nx > 0 ? cell_1d(c.x[i], c.o.dx, c.NX) : 0;
    const int cj = c.o.ny > 0 ? cell_1d(c.y[i], c.o.dy, c.NY) : 0;
    const int ck = c.o.nz > 0 ? cell_1d(c.z[i], c.o.dz, c.NZ) : 0;
    const long cell = ((long)ci * c.NY + cj) * c.NZ + ck;
    // :659 spectra are given at STP: concentrations scale with rho_d / rho_STP
    const double mult = spectrum_density(modes, s, lnr) * (s.hi - s.lo) / sd_conc_g * c.dV * (c.rhod[cell] / rho_stp);
    c.n[i] = (u64)std::max(1.0, std::floor(mult + 0.5));
    // :661-665 equilibrium at the cell's RH, at RH = 0.95 where the air is (nearly) saturated
    const CellThermo t = cell_thermo(c.th[cell], c.rv[cell], c.rhod[cell], 0.95);
    const double rw = equilibrium_rw(c.rd3[i], s.kappa, t.RH, t.A);
    c.rw2[i] = rw * rw;
  }
  c.step = 0; c.sorted = false;
  c.rain_flux_total = 0; c.cnt = orc_counters_t{};
  return N;
}

void orc_set_recycle(void* h, int on) { ((Ctx*)h)->recycle = on; }
long long orc_recycled(void* h) { return ((Ctx*)h)->recycled; }
void orc_stage_recycle(void* h) { recycle(*(Ctx*)h); }
void orc_set_step(void* h, u32 step) { ((Ctx*)h)->step = step; }
u32 orc_get_step(void* h) { return ((Ctx*)h)->step; }

// stage entry points (the tests drive them one by one; orc_step = all, in order)
void orc_stage_sort(void* h) { sort_stage(*(Ctx*)h); }
void orc_stage_cond(void* h, const orc_opts_t* op) { cond_stage(*(Ctx*)h, *op); }
void orc_stage_thermo(void* h, const orc_opts_t* op) { thermo_stage(*(Ctx*)h, *op); }
void orc_stage_coal(void* h, const orc_opts_t* op) { coal_stage(*(Ctx*)h, *op); }
void orc_stage_move(void* h, const orc_opts_t* op) { move_stage(*(Ctx*)h, *op); }

// the part of a step that alters th, rv (PAPER.md :816 step_sync)
void orc_step_sync(void* h, const orc_opts_t* op) {
  Ctx& c = *(Ctx*)h;
  sort_stage(c);
  if (op->cond) cond_stage(c, *op);
  thermo_stage(c, *op);
}
// the rest (PAPER.md :816 step_async); returns this step's rain flux [kg]
double orc_step_async(void* h, const orc_opts_t* op) {
  Ctx& c = *(Ctx*)h;
  c.rain_flux_step = 0.0;
  if (op->coal) coal_stage(c, *op);
  if (op->adve || op->sedi) move_stage(c, *op);
  c.step += 1;
  c.sorted = false;
  return c.rain_flux_step;
}
double orc_step(void* h, const orc_opts_t* op) {
  orc_step_sync(h, op);
  return orc_step_async(h, op);
}

long orc_n_sd(void* h) { return (long)((Ctx*)h)->n.size(); }
long orc_n_live(void* h) {
  Ctx& c = *(Ctx*)h; long w = 0;
  for (u64 v : c.n) w += (v != 0);
  return w;
}
void orc_get_state(void* h, u64* n, double* rw2, double* rd3, double* kappa, double* x, double* y, double* z, u32* id) {
  Ctx& c = *(Ctx*)h; const size_t N = c.n.size();
  if (n) memcpy(n, c.n.data(), N * 8);
  if (rw2) memcpy(rw2, c.rw2.data(), N * 8);
  if (rd3) memcpy(rd3, c.rd3.data(), N * 8);
  if (kappa) memcpy(kappa, c.kappa.data(), N * 8);
  if (x) memcpy(x, c.x.data(), N * 8);
  if (y) memcpy(y, c.y.data(), N * 8);
  if (z) memcpy(z, c.z.data(), N * 8);
  if (id) memcpy(id, c.id.data(), N * 4);
}
void orc_get_fields(void* h, double* th, double* rv) {
  Ctx& c = *(Ctx*)h;
  if (th) memcpy(th, c.th.data(), c.ncell * 8);
  if (rv) memcpy(rv, c.rv.data(), c.ncell * 8);
}
// after orc_stage_sort: ids in sorted order and the per-cell segment offsets
void orc_get_order(void* h, u32* ids_sorted, long* seg) {
  Ctx& c = *(Ctx*)h;
  for (size_t p = 0; p < c.order.size(); ++p) ids_sorted[p] = c.id[c.order[p]];
  memcpy(seg, c.seg.data(), (c.ncell + 1) * sizeof(long));
}
// One first-order upstream (donor-cell) step of a scalar field on the Arakawa-C grid (PAPER.md :219-235; the prototype
// transport solver of Figure 7, :831-852) with the rho_d x Courant arrays of the context: psi' = psi - sum_dims (F_hi - F_lo) /
// rho_d, F = max(rho_d C, 0) psi_donor-side + min(rho_d C, 0) psi_other; periodic in x and y, boundary value beyond bottom and top.
void orc_upstream_advect(void* h, double* psi) {
  const Ctx& c = *(Ctx*)h;
  const int NX = c.NX, NY = c.NY, NZ = c.NZ;
  const bool hx = c.o.nx > 0, hy = c.o.ny > 0, hz = c.o.nz > 0;
  std::vector<double> out(c.ncell);
  auto at = [&](int i, int j, int k) { return psi[((long)i * NY + j) * NZ + k]; };
  for (int i = 0; i < NX; ++i)
    for (int j = 0; j < NY; ++j)
      for (int k = 0; k < NZ; ++k) {
        const double pc = at(i, j, k);
        double acc = 0.0;
        if (hx) {
          const double pm = at(i == 0 ? NX - 1 : i - 1, j, k), pp = at(i == NX - 1 ? 0 : i + 1, j, k);
          const double Cl = c.cx[((long)i * NY + j) * NZ + k], Ch = c.cx[((long)(i + 1) * NY + j) * NZ + k];
          acc = acc + ((std::fmax(Ch, 0.0) * pc + std::fmin(Ch, 0.0) * pp) - (std::fmax(Cl, 0.0) * pm + std::fmin(Cl, 0.0) * pc));
        }
        if (hy) {
          const double pm = at(i, j == 0 ? NY - 1 : j - 1, k), pp = at(i, j == NY - 1 ? 0 : j + 1, k);
          const double Cl = c.cy[((long)i * (NY + 1) + j) * NZ + k], Ch = c.cy[((long)i * (NY + 1) + j + 1) * NZ + k];
          acc = acc + ((std::fmax(Ch, 0.0) * pc + std::fmin(Ch, 0.0) * pp) - (std::fmax(Cl, 0.0) * pm + std::fmin(Cl, 0.0) * pc));
        }
        if (hz) {
          const double pm = at(i, j, k == 0 ? 0 : k - 1), pp = at(i, j, k == NZ - 1 ? k : k + 1);
          const double Cl = c.cz[((long)i * NY + j) * (NZ + 1) + k], Ch = c.cz[((long)i * NY + j) * (NZ + 1) + k + 1];
          acc = acc + ((std::fmax(Ch, 0.0) * pc + std::fmin(Ch, 0.0) * pp) - (std::fmax(Cl, 0.0) * pm + std::fmin(Cl, 0.0) * pc));
        }
        out[((long)i * NY + j) * NZ + k] = pc - acc / c.rhod[((long)i * NY + j) * NZ + k];
      }
  std::copy(out.begin(), out.end(), psi);
}

void orc_get_counters(void* h, orc_counters_t* out) { *out = ((Ctx*)h)->cnt; }
double orc_rain_flux_total(void* h) { return ((Ctx*)h)->rain_flux_total; }

// PAPER.md :818-823 eq. 29: k-th moment of the wet (wet=1) or dry spectrum per cell over
// r in [r_mi, r_mx) (reading R-interval), divided by rhod dV. Uses current positions.
void orc_diag_mom(void* h, int wet, double r_mi, double r_mx, int k, double* out) {
  Ctx& c = *(Ctx*)h;
  compute_cells(c);
  for (long q = 0; q < c.ncell; ++q) out[q] = 0.0;
  for (size_t s = 0; s < c.n.size(); ++s) {
    if (c.n[s] == 0) continue;
    const double r = wet ? std::sqrt(c.rw2[s]) : std::cbrt(c.rd3[s]);
    if (r >= r_mi && r < r_mx) out[c.cell[s]] += (double)c.n[s] * std::pow(r, (double)k);
  }
  for (long q = 0; q < c.ncell; ++q) out[q] /= (c.rhod[q] * c.dV);
}
// PAPER.md :818 diag_sd_conc: number of computational particles per cell
void orc_diag_sd_conc(void* h, double* out) {
  Ctx& c = *(Ctx*)h;
  compute_cells(c);
  for (long q = 0; q < c.ncell; ++q) out[q] = 0.0;
  for (size_t s = 0; s < c.n.size(); ++s) if (c.n[s] != 0) out[c.cell[s]] += 1.0;
}

// ---- unit-level access for the pins -----------------------------------------
void orc_philox(const u32* ctr, const u32* key, u32* out) { philox4x32_10(ctr, key, out); }
double orc_T(double th, double rhod) { return T_of(th, rhod); }
double orc_p(double rhod, double rv, double T) { return p_of(rhod, rv, T); }
double orc_pvs(double T) { return p_vs(T); }
double orc_lv(double T) { return l_v(T); }
double orc_eta(double T) { return eta_air(T); }
double orc_vterm(double r, double T, double rhod, double rv) { return v_term(r, eta_air(T), rhod * (1.0 + rv)); }
// growth rate d r_w^2/dt with Sh, Nu of radius sqrt(y_vent)
double orc_growth_f(double y, double rd3, double kappa, double th, double rv, double rhod, double RH_max, double y_vent) {
  const CellThermo ct = cell_thermo(th, rv, rhod, RH_max);
  const double r0 = std::sqrt(y_vent);
  const double vt = v_term(r0, ct.eta, ct.rho_a);
  const double Re = 2.0 * r0 * vt * ct.rho_a / ct.eta;
  return growth_f(y, rd3, kappa, ct, vent(Re, ct.Sc), vent(Re, ct.Pr));
}
void orc_cell_thermo(double th, double rv, double rhod, double RH_max, double* out8) {
  const CellThermo ct = cell_thermo(th, rv, rhod, RH_max);
  out8[0] = ct.T; out8[1] = ct.p; out8[2] = ct.lv; out8[3] = ct.rho_vs; out8[4] = ct.RH; out8[5] = ct.A;
  out8[6] = ct.eta; out8[7] = ct.rho_a;
}
double orc_cond_substep(double y0, double rd3, double kappa, double th, double rv, double rhod, double RH_max,
                        double dtp, int* ill_posed) {
  const CellThermo ct = cell_thermo(th, rv, rhod, RH_max);
  return cond_substep_sd(y0, rd3, kappa, ct, dtp, ill_posed, nullptr);
}
double orc_adve_1d(double x, double dx, double C_lo, double C_hi) { return adve_1d(x, dx, C_lo, C_hi); }
double orc_eff(void* h, double R, double q) { return eff_lookup(*(Ctx*)h, R, q); }

}  // extern "C"
