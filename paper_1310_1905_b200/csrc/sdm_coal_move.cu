// Stages a5 + a6 in one cell-resident kernel: SDM coalescence on the pairs
// (0,1),(2,3).. of the cell's sorted segment (PAPER.md :622-645, eq. 27-28) followed by advection
// (eq. 16) and sedimentation (:647-651) of every SD of the cell.
// This translation unit is compiled with -fmad=false: the collision probability and the new
// positions use only IEEE +,-,*,/,sqrt in the oracle's order, so that collision decisions
// (u < frac p) and cell-border decisions are taken on bit-identical numbers whenever the inputs are.
#include "sdm_kernels.cuh"

namespace sdm {

template <bool SMEM, typename R> struct RealSel { typedef double type; };
template <typename R> struct RealSel<false, R> { typedef R type; };

// collision efficiency: bilinear in (collector radius, ratio), clamped at the table edges
__device__ __forceinline__ double eff_lookup(const CoalParams& kp, double R, double q) {
  const int nR = kp.n_eff_R, nq = kp.n_eff_q;
  R = fmin(fmax(R, kp.eff_R[0]), kp.eff_R[nR - 1]);
  q = fmin(fmax(q, kp.eff_q[0]), kp.eff_q[nq - 1]);
  int iR = 0, iq = 0;
  while (iR < nR - 2 && kp.eff_R[iR + 1] <= R) ++iR;   // last node <= R (upper_bound - 1), at most n-2
  while (iq < nq - 2 && kp.eff_q[iq + 1] <= q) ++iq;
  const double t = (R - kp.eff_R[iR]) / (kp.eff_R[iR + 1] - kp.eff_R[iR]);
  const double s = (q - kp.eff_q[iq]) / (kp.eff_q[iq + 1] - kp.eff_q[iq]);
  const double e00 = kp.eff_tab[iR * nq + iq], e01 = kp.eff_tab[iR * nq + iq + 1];
  const double e10 = kp.eff_tab[(iR + 1) * nq + iq], e11 = kp.eff_tab[(iR + 1) * nq + iq + 1];
  return (1.0 - t) * ((1.0 - s) * e00 + s * e01) + t * ((1.0 - s) * e10 + s * e11);
}

__device__ __forceinline__ double wrap(double x, double X) {
  if (x < 0.0) x += X;
  if (x >= X) x -= X;
  return x;
}

// Shared memory per group: cap x {n (u64), rw2, rd3, kappa (double), id (u32)} (SMEM) or cap x u16 slot
// indices (attributes left in HBM/L2), and for sstp_coal > 1 another P x {u64 key, u16 order}.
template <int G, bool SMEM, typename R>
__global__ void __launch_bounds__(CtaOf<G>::threads) k_coal_move(SdArraysT<R> a, const u16* __restrict__ rank,
                                                                 const u32* __restrict__ seg, Grid g, CellFields cf,
                                                                 CoalParams kp, CoalMoveParams mp, double* flux_slots,
                                                                 Counters cnt, int cap, int P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NG = CtaOf<G>::threads / G;
  __shared__ double red_scratch[32];
  const int gi = threadIdx.x / G;
  const Group<G> grp = make_group<G>(red_scratch);
  const int c = blockIdx.x * NG + gi;
  unsigned n_pairs = 0, n_coll = 0, n_tie = 0;
  double flux = 0.0;
  if (c < g.ncell) {
    const u32 s0 = seg[c];
    const int m = (int)(seg[c + 1] - s0);
    // per-group shared arrays, indexed by sorted position e.  SMEM: the attributes themselves;
    // otherwise (cells too large for shared memory) only the slot of position e, attributes stay in HBM/L2.
    const size_t attr_bytes = SMEM ? (size_t)cap * 36 : (size_t)cap * 2;
    unsigned char* base = smem_raw + (size_t)gi * (attr_bytes + (size_t)P * 10);
    using PT = typename RealSel<SMEM, R>::type;   // staged copies are doubles; in place, the storage type
    u64* pn; PT *prw2, *prd3, *pkap; u32* pid;
    u16* s_inv = reinterpret_cast<u16*>(base);
    if constexpr (SMEM) {
      pn = reinterpret_cast<u64*>(base);
      prw2 = reinterpret_cast<double*>(base) + cap;
      prd3 = reinterpret_cast<double*>(base) + 2 * cap;
      pkap = reinterpret_cast<double*>(base) + 3 * cap;
      pid = reinterpret_cast<u32*>(base + (size_t)cap * 32);
    } else {
      pn = a.n + s0; prw2 = a.rw2 + s0; prd3 = a.rd3 + s0; pkap = a.kappa + s0; pid = a.id + s0;
    }
    auto SL = [&](int e) -> int { if constexpr (SMEM) return e; else return (int)s_inv[e]; };
    u64* s_key = reinterpret_cast<u64*>(base + attr_bytes);
    u16* s_ord = reinterpret_cast<u16*>(base + attr_bytes + (size_t)P * 8);
    const double eta = cf.eta[c], rho_a = cf.rho_a[c];
    if (m > 0 && mp.coal) {
      for (int t = grp.lane; t < m; t += G) {
        const int e = rank[s0 + t];
        if constexpr (SMEM) {
          pn[e] = a.n[s0 + t];
          prw2[e] = a.rw2[s0 + t];
          prd3[e] = a.rd3[s0 + t];
          pkap[e] = a.kappa[s0 + t];
          pid[e] = a.id[s0 + t];
        } else {
          s_inv[e] = (u16)t;
        }
      }
      grp.sync();
      // R-adapt-coal (PAPER.md :645; oracle: coal_substep_multiplier): sstp_coal * m substeps, m = min(cap, ceil(largest P of
      // eq. 27 among the pairs of the first grouping, for dt / sstp_coal)); the same IEEE operations as in the pair loop below
      int nsub = mp.sstp_coal;
      if (mp.coal_adapt_max > 1 && m >= 2) {
        const double dt0 = g.dt / mp.sstp_coal;
        const double scale0 = (double)((u64)m * (u64)(m - 1) / 2) / (double)(m / 2);
        double pmax = 0.0;
        for (int pr = grp.lane; pr < m / 2; pr += G) {
          const int ea = SL(2 * pr), eb = SL(2 * pr + 1);
          const u64 na = pn[ea], nb = pn[eb];
          const int j = (na >= nb) ? ea : eb, k = (na >= nb) ? eb : ea;
          const u64 nj = (na >= nb) ? na : nb;
          const double yj = prw2[j], yk = prw2[k];
          const double rj = sqrt(yj), rk = sqrt(yk);
          double K;
          if (kp.kernel == 1) {
            const double vj = (4.0 / 3.0) * cst::pi * (yj * rj), vk = (4.0 / 3.0) * cst::pi * (yk * rk);
            K = kp.golovin_b * (vj + vk);
          } else {
            const double vj = v_term(rj, eta, rho_a), vk = v_term(rk, eta, rho_a);
            K = cst::pi * ((rj + rk) * (rj + rk)) * fabs(vj - vk);
            if (kp.kernel == 2) {
              const double rl = fmax(rj, rk), rs = fmin(rj, rk);
              K = K * eff_lookup(kp, rl, rs / rl);
            }
          }
          pmax = fmax(pmax, (((double)nj * K) * (dt0 / g.dV)) * scale0);
        }
        pmax = grp.max_nonneg(pmax);
        const double want = ceil(pmax);
        const int mult = want >= (double)mp.coal_adapt_max ? mp.coal_adapt_max : max(1, (int)want);
        nsub = mp.sstp_coal * mult;
      }
      const double dtpp = g.dt / nsub;
      int nc = m;   // SDs taking part in this substep
      for (int sub = 0; sub < nsub; ++sub) {
        if (sub > 0) {
          // new random grouping (:624): drop SDs that reached N = 0, draw new keys, sort again
          const int Pm = next_pow2(m);
          for (int t = grp.lane; t < Pm; t += G) {
            u64 key = ~0ull;
            if (t < m && pn[SL(t)] != 0) { const u32 sid = pid[SL(t)]; key = ((u64)shuffle_key(sid, mp.step, (u32)sub, kp.seed_lo, kp.seed_hi) << 32) | sid; }
            s_key[t] = key;
            s_ord[t] = (u16)t;
          }
          bitonic_sort<G, u16>(grp, s_key, s_ord, Pm);
          int live = 0;
          for (int t = grp.lane; t < m; t += G) live += (s_key[t] != ~0ull);
          nc = (int)grp.sum((unsigned long long)live);
        }
        if (nc >= 2) {
          // eq. 27 last factor n(n-1)/2 / floor(n/2)
          const double scale = (double)((u64)nc * (u64)(nc - 1) / 2) / (double)(nc / 2);
          for (int pr = grp.lane; pr < nc / 2; pr += G) {
            const int ea = SL((sub == 0) ? 2 * pr : s_ord[2 * pr]);
            const int eb = SL((sub == 0) ? 2 * pr + 1 : s_ord[2 * pr + 1]);
            const u64 na = pn[ea], nb = pn[eb];
            const int j = (na >= nb) ? ea : eb, k = (na >= nb) ? eb : ea;   // j: larger N; tie -> first in order
            const u64 nj = (na >= nb) ? na : nb, nk = (na >= nb) ? nb : na;
            const double yj = prw2[j], yk = prw2[k];
            const double rj = sqrt(yj), rk = sqrt(yk);
            double K;
            if (kp.kernel == 1) {   // Golovin
              const double vj = (4.0 / 3.0) * cst::pi * (yj * rj), vk = (4.0 / 3.0) * cst::pi * (yk * rk);
              K = kp.golovin_b * (vj + vk);
            } else {                // eq. 28
              const double vj = v_term(rj, eta, rho_a), vk = v_term(rk, eta, rho_a);
              K = cst::pi * ((rj + rk) * (rj + rk)) * fabs(vj - vk);
              if (kp.kernel == 2) {
                const double rl = fmax(rj, rk), rs = fmin(rj, rk);
                K = K * eff_lookup(kp, rl, rs / rl);
              }
            }
            const double p = (((double)nj * K) * (dtpp / g.dV)) * scale;   // eq. 27
            const double u = coal_uniform(pid[ea], mp.step, (u32)sub, kp.seed_lo, kp.seed_hi);
            const u64 qmax = nj / nk;
            u64 gam;
            if (kp.multi_coal) {
              const double pf = floor(p);
              if (pf >= (double)qmax) gam = qmax;
              else {
                const double frac = p - pf;
                if (fabs(u - frac) < 1e-12) ++n_tie;
                gam = (u64)pf + (u < frac ? 1u : 0u);
                if (gam > qmax) gam = qmax;
              }
            } else {
              if (fabs(u - p) < 1e-12) ++n_tie;
              gam = (u < p) ? 1u : 0u;   // :639, :645
            }
            ++n_pairs;
            if (gam == 0) continue;
            ++n_coll;
            const double gd = (double)gam;
            const double rw3 = yk * rk + gd * (yj * rj);    // extensive attributes are summed (:643)
            const double rd3j = gd * prd3[j];
            const double rd3k = prd3[k];
            const double kj = pkap[j], kk = pkap[k];
            if (kj != kk)                                    // intensive ones averaged (:643)
              pkap[k] = (rd3j * kj + rd3k * kk) / (rd3j + rd3k);
            prd3[k] = rd3k + rd3j;
            const double r = cbrt(rw3);
            prw2[k] = (PT)(double)(R)(r * r);   // what is stored is the radius from here on (as in k_coal_move_tile)
            pn[j] = nj - gam * nk;
          }
        }
        grp.sync();
      }
    }
    // ---- advection + sedimentation, SD by SD in storage order --------------------------------------
    if (m > 0 && (mp.coal || mp.adve || mp.sedi)) {
      const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
      const double rhod = cf.rhod[c];
      double Cxl = 0, Cxh = 0, Cyl = 0, Cyh = 0, Czl = 0, Czh = 0;
      if (mp.adve) {
        if (g.hx) { Cxl = cf.cx[((long long)i * g.NY + j) * g.NZ + k] / rhod; Cxh = cf.cx[((long long)(i + 1) * g.NY + j) * g.NZ + k] / rhod; }
        if (g.hy) { Cyl = cf.cy[((long long)i * (g.NY + 1) + j) * g.NZ + k] / rhod; Cyh = cf.cy[((long long)i * (g.NY + 1) + j + 1) * g.NZ + k] / rhod; }
        if (g.hz) { Czl = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k] / rhod; Czh = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k + 1] / rhod; }
      }
      for (int t = grp.lane; t < m; t += G) {
        const u32 s = s0 + t;
        u64 n; double y;
        if (SMEM && mp.coal) {
          const int e = rank[s];
          n = pn[e]; y = prw2[e];
          a.n[s] = n; a.rw2[s] = y; a.rd3[s] = prd3[e]; a.kappa[s] = pkap[e];
        } else {
          n = a.n[s]; y = a.rw2[s];
        }
        if (n == 0 || !(mp.adve || mp.sedi)) continue;
        double xn = 0, yn = 0, zn = 0;
        if (g.hx) xn = a.x[s];
        if (g.hy) yn = a.y[s];
        if (g.hz) zn = a.z[s];
        if (mp.adve) {   // eq. 16 with the Courant numbers at the edges of the SD's time-n cell
          if (g.hx) { const double dC = Cxh - Cxl; xn = (xn + g.dx * (Cxl - (double)i * dC)) / (1.0 - dC); }
          if (g.hy) { const double dC = Cyh - Cyl; yn = (yn + g.dy * (Cyl - (double)j * dC)) / (1.0 - dC); }
          if (g.hz) { const double dC = Czh - Czl; zn = (zn + g.dz * (Czl - (double)k * dC)) / (1.0 - dC); }
        }
        if (mp.sedi && g.hz) zn = zn - v_term(sqrt(y), eta, rho_a) * g.dt;   // explicit Euler (:649)
        if (g.hx) { if (!g.open_x) xn = wrap(xn, g.X); a.x[s] = xn; }         // periodic (:558) unless the context is a slab
        if (g.hy) { yn = wrap(yn, g.Y); a.y[s] = yn; }
        if (g.hz) {
          if (zn < 0.0 || !(zn < g.Z)) {                                       // left the domain (:651)
            if (zn < 0.0) flux += (double)n * ((4.0 / 3.0) * cst::pi * cst::rho_w * (y * sqrt(y)));
            a.n[s] = 0;
          }
          a.z[s] = zn;
        }
      }
    }
  }
  // rain flux and counters: warp-reduce, then one atomic per warp on spread addresses
  unsigned v0 = n_pairs, v1 = n_coll, v2 = n_tie;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    v0 += __shfl_xor_sync(0xffffffffu, v0, d);
    v1 += __shfl_xor_sync(0xffffffffu, v1, d);
    v2 += __shfl_xor_sync(0xffffffffu, v2, d);
    flux += __shfl_xor_sync(0xffffffffu, flux, d);
  }
  if ((threadIdx.x & 31) == 0) {
    const int slot = (blockIdx.x * (CtaOf<G>::threads / 32) + (threadIdx.x >> 5)) & (NSLOT - 1);
    if (v0) atomicAdd(&cnt.pairs[slot], (unsigned long long)v0);
    if (v1) atomicAdd(&cnt.collisions[slot], (unsigned long long)v1);
    if (v2) atomicAdd(&cnt.near_ties[slot], (unsigned long long)v2);
    if (flux != 0.0) atomicAdd(&flux_slots[slot], flux);
  }
}

// ---- k_coal_move_tile: the same stages for sstp_coal == 1, tile-resident -----------------------------
// A CTA of T threads owns a tile of `cpb` consecutive cells (at most CAP - cpb SDs).
//  * n, r_w^2, id and the positions of the tile's SDs are one contiguous run per attribute in storage order: thread 0
//    fetches each run with ONE bulk asynchronous copy (cp.async.bulk, the 1-D form of TMA: UBLKCP in SASS) signalled on an
//    mbarrier, while all threads build the inverse map of the sorted order.  Bulk copies move multiples of 16 bytes between
//    16-byte aligned addresses, so a run starts at the aligned element below its first one and element t of the tile sits
//    at index t + sh of every shared array, sh = (first slot) mod 4 (the state arrays are allocated with 4 elements to spare).
//  * The sorted order enters through inv[sorted position] = slot, built with every cell's segment padded to an even
//    length, so that thread t owns the pair of sorted positions (2t, 2t+1): all lanes are busy whatever the cell
//    populations are.  The thread of a pair does everything for its two SDs: terminal velocities, eq. 27-28, the Philox
//    uniform, the Shima update, then eq. 16 and sedimentation, the cell index of the NEW position and its place in the
//    next step's histogram.  There is no barrier between coalescence and movement and no per-SD search for the cell.
//  * r_d^3 and kappa are touched (in global memory) only by the rare pairs that collide, n and r_w^2 are written back only
//    where they changed; the new positions go back to shared memory and are stored coalesced in storage order.
//  * Next step's a0-a1 (PAPER.md :547, :641): `cell` and `off` of every SD and the histogram `count` are produced here, in the
//    pass that stores the new positions (lanes that go to the same cell share one atomic on count[cell], as in k_cellhist), so that
//    step_sync need not read the positions again (k_cellhist stays for the first step, recycling and the per-cell kernel).
//  * Arithmetic: the collision probability and the new positions need not be bit-identical to the oracle's (north_star
//    counts near-tie decisions; positions are compared to 1e-9), so divisions by per-cell constants are multiplications by
//    their IEEE reciprocals and square roots / reciprocals of per-SD values are the hardware seeds with two Newton steps
//    (<= 2 ulp).  The CELL INDEX is different: floor(x/dx) decides which SDs meet, so it is the oracle's IEEE quotient
//    whenever the fast quotient lies within 1e-9 of an integer.
struct __align__(8) CoalCell {
  double kX, kv, scale;          // v_term: X = kX r^3, v = kv s^2 / r; eq. 27 factor n(n-1)/2 / floor(n/2)
  double ax, bx, ay, by, az, bz; // eq. 16: x' = (x + a) b, a = dx (C_l - i dC), b = 1/(1 - dC)
};

// 1/sqrt(a) and 1/a: hardware seed (2^-22) and two Newton steps
__device__ __forceinline__ double rsqrt_nr(double a) {
  double x;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(a));
  const double h = 0.5 * a;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const double e = fma(-h * x, x, 0.5);
    x = fma(x, e, x);
  }
  return x;
}
__device__ __forceinline__ double rcp_nr2(double a) {
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(a));
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const double e = fma(-a, x, 1.0);
    x = fma(x, e, x);
  }
  return x;
}
// terminal velocity (PAPER.md :649, DESIGN.md R-vt) from y = r^2 with the cell's constants; also returns r
__device__ __forceinline__ double v_term_cell(double y, const CoalCell& C, double& r_out) {
  const double c1 = 4.0 / (cst::kc_delta0 * cst::kc_delta0 * 0.5403702434442518 /* sqrt(C0) */);
  const double rinv = rsqrt_nr(y);
  const double r = y * rinv;
  r_out = r;
  const double X = C.kX * (y * r);
  const double e = c1 * (X * rsqrt_nr(X));
  const double w = 1.0 + e;
  const double s = e * rcp_nr2(fma(w, rsqrt_nr(w), 1.0));
  return C.kv * (s * s) * rinv;
}
// cell index along one dimension, the oracle's floor(x/dx) clamped (eq. 15)
__device__ __noinline__ double ieee_quotient(double x, double dx) { return x / dx; }   // rare: kept out of the hot loop
__device__ __forceinline__ int cell_1d_fast(double x, double dx, double inv_dx, int n) {
  double q = x * inv_dx;
  const double f = q - floor(q);
  if (__builtin_expect(f < 1e-9 || f > 1.0 - 1e-9, 0)) q = ieee_quotient(x, dx);
  int i = (int)floor(q);
  i = max(i, 0);
  return min(i, n - 1);
}

// Outcome of gam collisions between j (the larger multiplicity, slot gj) and k (slot gk) in global memory (PAPER.md :639-643,
// DESIGN.md R-outcome, R-kappa); returns the new r_w^2 of k as stored.  Rare: kept out of the hot loop.
template <typename R>
__device__ __noinline__ double shima_update(const SdArraysT<R>& a, u32 gj, u32 gk, u64 gam, u64 nj2, double yj, double yk, double rj,
                                            double rk) {
  const double gd = (double)gam;
  const double rw3 = yk * rk + gd * (yj * rj);    // extensive attributes are summed (:643)
  const double rd3j = gd * a.rd3[gj];
  const double rd3k = a.rd3[gk];
  const double kj = a.kappa[gj], kk = a.kappa[gk];
  if (kj != kk)                                    // intensive ones averaged (:643)
    a.kappa[gk] = (rd3j * kj + rd3k * kk) / (rd3j + rd3k);
  a.rd3[gk] = rd3k + rd3j;
  const double r = cbrt(rw3);
  const R y2 = (R)(r * r);   // what is stored is the radius from here on
  a.rw2[gk] = y2;
  a.n[gj] = nj2;
  return (double)y2;
}

// eq. 16 per cell (PAPER.md :556-558): x' = (x + a) b with a = dx (C_l - i dC), b = 1 / (1 - dC), from the Courant numbers at the
// faces of the cell.  They change only when the caller hands new Courant fields or a new rho_d to step_sync, so they are a
// table (cf.mv, 6 doubles per cell), not something every tile works out again in every step behind its first barrier.
__global__ void __launch_bounds__(256) k_cell_move_consts(Grid g, CellFields cf) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.ncell) return;
  const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
  const double rhod = cf.rhod[c];
  double ax = 0.0, bx = 1.0, ay = 0.0, by = 1.0, az = 0.0, bz = 1.0;
  if (g.hx) {
    const double Cl = cf.cx[((long long)i * g.NY + j) * g.NZ + k] / rhod, Ch = cf.cx[((long long)(i + 1) * g.NY + j) * g.NZ + k] / rhod;
    const double dC = Ch - Cl;
    ax = g.dx * (Cl - (double)i * dC); bx = 1.0 / (1.0 - dC);
  }
  if (g.hy) {
    const double Cl = cf.cy[((long long)i * (g.NY + 1) + j) * g.NZ + k] / rhod, Ch = cf.cy[((long long)i * (g.NY + 1) + j + 1) * g.NZ + k] / rhod;
    const double dC = Ch - Cl;
    ay = g.dy * (Cl - (double)j * dC); by = 1.0 / (1.0 - dC);
  }
  if (g.hz) {
    const double Cl = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k] / rhod, Ch = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k + 1] / rhod;
    const double dC = Ch - Cl;
    az = g.dz * (Cl - (double)k * dC); bz = 1.0 / (1.0 - dC);
  }
  double2* o = reinterpret_cast<double2*>(cf.mv + (size_t)6 * c);
  o[0] = make_double2(ax, bx); o[1] = make_double2(ay, by); o[2] = make_double2(az, bz);
}
void launch_cell_move_consts(const Grid& g, const CellFields& cf, cudaStream_t st) {
  k_cell_move_consts<<<(g.ncell + 255) / 256, 256, 0, st>>>(g, cf);
}

template <int CAP, int T, typename R>
struct CoalTile {   // per slot: u64 n; R rw2, x, y, z; u32 id / new cell; u16 inv, rank; u8 cell of the pair
  static_assert(CAP % 16 == 0, "the arrays of the tile follow one another in shared memory: keep every one of them 16-byte aligned");
  static constexpr int SLOTS = CAP + 16;   // room for the alignment shift of the bulk copies
  static constexpr size_t fixed_bytes = (size_t)SLOTS * (8 + 4 * sizeof(R) + 4 + 2 + 2) + (size_t)(SLOTS / 2) * 2;
  static size_t smem(int cpb) { return fixed_bytes + (size_t)cpb * (sizeof(CoalCell) + 8) + 64; }
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, unsigned bytes, unsigned long long* mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"(smem_u32(mbar))
               : "memory");
}

template <int CAP, int T, int MINB, typename R>
__global__ void __launch_bounds__(T, MINB)
k_coal_move_tile(SdArraysT<R> a, const u16* __restrict__ rank, const u32* __restrict__ seg, Grid g, CellFields cf, CoalParams kp,
                 CoalMoveParams mp, double* __restrict__ flux_part, Counters cnt, int cpb, u32* __restrict__ cell_out,
                 u32* __restrict__ off_out, u32* __restrict__ count) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using L = CoalTile<CAP, T, R>;
  constexpr int SLOTS = L::SLOTS;
  constexpr int NW = T / 32;
  constexpr u16 NONE = 0xFFFFu;
  __shared__ __align__(8) unsigned long long mbar;
  __shared__ double s_flux[NW];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c_first = blockIdx.x * cpb;
  const int nc = min(cpb, g.ncell - c_first);
  u64* s_n = reinterpret_cast<u64*>(smem_raw);
  R* s_rw2 = reinterpret_cast<R*>(s_n + SLOTS);
  R* s_x = s_rw2 + SLOTS;
  R* s_y = s_x + SLOTS;
  R* s_z = s_y + SLOTS;
  u32* s_id = reinterpret_cast<u32*>(s_z + SLOTS);      // id until the pair is done, then the SD's new cell
  u16* inv = reinterpret_cast<u16*>(s_id + SLOTS);
  u16* s_rk = inv + SLOTS;                            // rank of the slot inside its cell (sdm_sort.cu), element t at t + (s0 mod 8)
  u16* s_pc = s_rk + SLOTS;                             // cell (tile-local) of pair p
  CoalCell* s_cell = reinterpret_cast<CoalCell*>(smem_raw + L::fixed_bytes);
  u32* segl = reinterpret_cast<u32*>(s_cell + cpb);     // storage offsets of the tile's cells
  u32* segp = segl + cpb + 1;                           // padded (even) offsets of the sorted positions
  // what the lanes that own a cell of the tile need from global memory, requested together with the tile's bounds below:
  // the whole CTA waits for these few lanes at the first barrier, so they should wait for ONE memory latency, not two
  struct CellIn { u32 b0, b1; double eta, rho_a; double2 mx, my, mz; };
  auto load_cell = [&](int c) {
    CellIn in;
    in.b0 = seg[c]; in.b1 = seg[c + 1];
    in.eta = cf.eta[c]; in.rho_a = cf.rho_a[c];
    in.mx = make_double2(0.0, 1.0); in.my = in.mx; in.mz = in.mx;
    if (mp.adve) {   // eq. 16 with the Courant numbers at the faces of the SD's time-n cell: the table of k_cell_move_consts
      const double2* mvp = reinterpret_cast<const double2*>(cf.mv + (size_t)6 * c);
      in.mx = mvp[0]; in.my = mvp[1]; in.mz = mvp[2];
    }
    return in;
  };
  CellIn pre;
  if (tid < nc) pre = load_cell(c_first + tid);
  const u32 s0 = seg[c_first];
  const int M = (int)(seg[c_first + nc] - s0);
  const int sh = (int)(s0 & 3u);
  const bool moving = mp.adve || mp.sedi;
  const bool need_vt = mp.sedi && g.hz;
  unsigned n_pairs = 0, n_coll = 0, n_tie = 0;
  double flux = 0.0;
  if (M > 0) {
    if (tid == 0) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&mbar)) : "memory");
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      // the runs, from the 16-byte aligned element at or below the first one
      const u32 lo4 = s0 - (u32)sh;                                   // 4-byte elements: multiple of 4
      const unsigned n4 = (unsigned)((M + sh + 3) & ~3) * 4u;
      const int sh8 = (int)(s0 & 1u);
      const u32 lo8 = s0 - (u32)sh8;                                  // 8-byte elements: multiple of 2
      const unsigned n8 = (unsigned)((M + sh8 + 1) & ~1) * 8u;
      const int d8 = sh - sh8;                                        // even: 16-byte aligned in shared memory
      constexpr bool R8 = sizeof(R) == 8;
      const unsigned nR = R8 ? n8 : n4;
      const u32 loR = R8 ? lo8 : lo4;
      const int dR = R8 ? d8 : 0;
      const int sh2 = (int)(s0 & 7u);                                 // 2-byte elements: multiple of 8
      const unsigned n2 = (unsigned)((M + sh2 + 7) & ~7) * 2u;
      unsigned total = n8 + nR + n2 + (mp.coal ? n4 : 0u);
      if (g.hx) total += nR;
      if (g.hy) total += nR;
      if (g.hz) total += nR;
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(&mbar)), "r"(total) : "memory");
      bulk_load(s_rk, rank + (s0 - (u32)sh2), n2, &mbar);
      bulk_load(s_n + d8, a.n + lo8, n8, &mbar);
      bulk_load(s_rw2 + dR, a.rw2 + loR, nR, &mbar);
      if (mp.coal) bulk_load(s_id, a.id + lo4, n4, &mbar);
      if (g.hx) bulk_load(s_x + dR, a.x + loR, nR, &mbar);
      if (g.hy) bulk_load(s_y + dR, a.y + loR, nR, &mbar);
      if (g.hz) bulk_load(s_z + dR, a.z + loR, nR, &mbar);
    }
    for (int cl = tid; cl < nc; cl += T) {
      const int c = c_first + cl;
      const CellIn in = cl == tid ? pre : load_cell(c);
      segl[cl] = in.b0 - s0;
      const int m = (int)(in.b1 - in.b0);
      CoalCell& C = s_cell[cl];
      const double eta = in.eta, rho_a = in.rho_a;
      const double2 mx = in.mx, my = in.my, mz = in.mz;
      C.kX = ((32.0 / 3.0 * cst::g) * ((cst::rho_w - rho_a) * rho_a)) * rcp_nr2(eta * eta);
      C.kv = (eta * (cst::kc_delta0 * cst::kc_delta0 / 8.0)) * rcp_nr2(rho_a);
      // eq. 27: n (n - 1) / 2 pairs over floor(n / 2) drawn = n - 1 for even n, n for odd n
      C.scale = m >= 2 ? (double)((m & 1) ? m : m - 1) : 0.0;
      C.ax = mx.x; C.bx = mx.y; C.ay = my.x; C.by = my.y; C.az = mz.x; C.bz = mz.y;
    }
    if (tid == 0) segl[nc] = (u32)M;
    __syncthreads();
    // padded offsets: warp scan over the cells, 32 at a time; every warp does it for itself when the tile has at most 32
    // cells (the same values from every warp: no barrier before the next phase)
    if (nc < 32 || tid < 32) {
      u32 carry = 0;
      for (int c0 = 0; c0 <= nc; c0 += 32) {
        const int cl = c0 + lane;
        u32 v = 0;
        if (cl < nc) { const u32 m = segl[cl + 1] - segl[cl]; v = m + (m & 1u); }
        u32 inc = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const u32 t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
        if (cl <= nc) segp[cl] = carry + inc - v;
        carry += __shfl_sync(0xffffffffu, inc, 31);
      }
      __syncwarp();
    }
    if (nc >= 32) __syncthreads();
    const int MP = (int)segp[nc];
    {   // the bulk copies have landed
      unsigned done = 0;
      while (!done)
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n selp.u32 %0, 1, 0, p;\n}" : "=r"(done) : "r"(smem_u32(&mbar)) : "memory");
    }
    // inverse map of the sorted order and the cell of every pair; populated cells: a warp takes a cell at a time
    const int sh2 = (int)(s0 & 7u);
    const bool by_cell = M >= 24 * nc;
    for (int q = by_cell ? warp : tid; q < (by_cell ? nc : M); q += by_cell ? NW : T) {
      int cl, t0, t1;
      if (by_cell) {
        cl = q; t0 = (int)segl[cl] + lane; t1 = (int)segl[cl + 1];
      } else {
        int lo = 0, hi = nc;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)q) lo = mid; else hi = mid; }
        cl = lo; t0 = q; t1 = q + 1;
      }
      const int p0 = (int)segp[cl];
      for (int t = t0; t < t1; t += 32) {
        const int e = p0 + (int)s_rk[t + sh2];
        inv[e] = (u16)(t + sh);
        if ((e & 1) == 0) s_pc[e >> 1] = (u16)cl;
      }
    }
    for (int cl = tid; cl < nc; cl += T) {   // the padding slot of an odd cell
      const u32 m = segl[cl + 1] - segl[cl];
      if (m & 1u) inv[segp[cl] + m] = NONE;
    }
    __syncthreads();
    // ---- pairs of sorted positions (2t, 2t+1): coalescence, then movement of both SDs ----------------------------------------
    const double dtdv = g.dt / g.dV;
    const double inv_dx = mp.inv_dx, inv_dy = mp.inv_dy, inv_dz = mp.inv_dz;
    for (int t = tid; 2 * t < MP; t += T) {
      const u32 both = reinterpret_cast<const u32*>(inv)[t];
      const int ia = (int)(both & 0xFFFFu), ib = (int)(both >> 16);
      const bool lone = ib == (int)NONE;
      const int cl = (int)s_pc[t];
      const CoalCell& C = s_cell[cl];
      u64 na = s_n[ia], nb = lone ? 0ull : s_n[ib];
      double ya = s_rw2[ia], yb = lone ? 1.0 : (double)s_rw2[ib];
      double ra = 0.0, rb = 0.0, va = 0.0, vb = 0.0;
      const bool geometric = kp.kernel != 1;
      if (need_vt || (mp.coal && geometric)) {
        va = v_term_cell(ya, C, ra);
        if (!lone) vb = v_term_cell(yb, C, rb);
      } else if (mp.coal) {
        ra = ya * rsqrt_nr(ya); rb = yb * rsqrt_nr(yb);
      }
      if (mp.coal && !lone) {
        const bool afirst = na >= nb;            // j: larger N; tie -> first in order
        const u64 nj = afirst ? na : nb, nk = afirst ? nb : na;
        const double yj = afirst ? ya : yb, yk = afirst ? yb : ya;
        const double rj = afirst ? ra : rb, rk = afirst ? rb : ra;
        double K;
        if (!geometric) {   // Golovin
          const double vj = (4.0 / 3.0) * cst::pi * (yj * rj), vk = (4.0 / 3.0) * cst::pi * (yk * rk);
          K = kp.golovin_b * (vj + vk);
        } else {            // eq. 28
          K = cst::pi * ((rj + rk) * (rj + rk)) * fabs(va - vb);
          if (kp.kernel == 2) {
            const double rl = fmax(rj, rk), rs = fmin(rj, rk);
            K = K * eff_lookup(kp, rl, rs / rl);
          }
        }
        const double p = (((double)nj * K) * dtdv) * C.scale;   // eq. 27
        const double u = coal_uniform(s_id[ia], mp.step, 0u, kp.seed_lo, kp.seed_hi);
        u64 gam;
        if (p < 1.0) {      // the usual case: floor(p) = 0, and nj >= nk allows one collision
          if (fabs(u - p) < 1e-12) ++n_tie;
          gam = (u < p) ? 1u : 0u;
        } else if (kp.multi_coal) {
          const u64 qmax = nj / nk;
          const double pf = floor(p);
          if (pf >= (double)qmax) gam = qmax;
          else {
            const double frac = p - pf;
            if (fabs(u - frac) < 1e-12) ++n_tie;
            gam = (u64)pf + (u < frac ? 1u : 0u);
            if (gam > qmax) gam = qmax;
          }
        } else {
          if (fabs(u - p) < 1e-12) ++n_tie;
          gam = 1u;   // u < 1 <= p (:639, :645)
        }
        ++n_pairs;
        if (gam != 0) {
          ++n_coll;
          // the rare pair that collides updates global memory itself (r_d^3 and kappa are not staged)
          const int j = afirst ? ia : ib, k = afirst ? ib : ia;
          const u32 gj = s0 + (u32)(j - sh), gk = s0 + (u32)(k - sh);
          const u64 nj2 = nj - gam * nk;
          const double y2 = shima_update(a, gj, gk, gam, nj2, yj, yk, rj, rk);
          double rr;
          const double v2 = need_vt ? v_term_cell(y2, C, rr) : 0.0;
          if (afirst) { na = nj2; yb = y2; vb = v2; } else { nb = nj2; ya = y2; va = v2; }
        }
      }
      // ---- eq. 16 + sedimentation of both SDs, the cell of the new position, its place in the next histogram --------
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        if (h == 1 && lone) break;
        const int sl = h ? ib : ia;
        const u64 n = h ? nb : na;
        const double yy = h ? yb : ya, vt = h ? vb : va;
        u32 cnew = CELL_DEAD;
        if (n != 0) {
          double xn = g.hx ? (double)s_x[sl] : 0.0, yn = g.hy ? (double)s_y[sl] : 0.0, zn = g.hz ? (double)s_z[sl] : 0.0;
          if (moving) {
            if (mp.adve) {
              if (g.hx) xn = (xn + C.ax) * C.bx;
              if (g.hy) yn = (yn + C.ay) * C.by;
              if (g.hz) zn = (zn + C.az) * C.bz;
            }
            if (need_vt) zn = zn - vt * g.dt;                                   // explicit Euler (:649)
            if (g.hx) { if (!g.open_x) xn = wrap(xn, g.X); s_x[sl] = (R)xn; xn = (double)(R)xn; }  // periodic (:558) unless a slab
            if (g.hy) { yn = wrap(yn, g.Y); s_y[sl] = (R)yn; yn = (double)(R)yn; }
            if (g.hz) { s_z[sl] = (R)zn; }
          }
          if (g.hz && moving && (zn < 0.0 || !(zn < g.Z))) {                     // left the domain (:651)
            if (zn < 0.0) flux += (double)n * ((4.0 / 3.0) * cst::pi * cst::rho_w * (yy * (yy * rsqrt_nr(yy))));
            a.n[s0 + (u32)(sl - sh)] = 0;
          } else {
            if (g.hz) zn = (double)(R)zn;
            const int ci = g.hx ? cell_1d_fast(xn, g.dx, inv_dx, g.NX) : 0;
            const int cj = g.hy ? cell_1d_fast(yn, g.dy, inv_dy, g.NY) : 0;
            const int ck = g.hz ? cell_1d_fast(zn, g.dz, inv_dz, g.NZ) : 0;
            cnew = (u32)((ci * g.NY + cj) * g.NZ + ck);
          }
        }
        if (mp.fold) s_id[sl] = cnew;
      }
    }
    __syncthreads();
    // ---- new positions back to global memory, coalesced in storage order; with mp.fold also the SD's cell and its place in
    // the next step's histogram, taken in STORAGE order (the reorder of the next step then writes runs, not a permutation of
    // each cell): lanes that go to the same cell take consecutive places with one atomic on count[cell], as k_cellhist does
    if (moving || mp.fold) {
      // the places are asked for first, for the whole tile (one atomic per group of lanes and pass, none waited for), the
      // positions are stored while they are on their way, and only then does the warp pick the answers up: the latency
      // of the atomics is paid once per tile, not once per 128 SDs
      constexpr int NIT = (CAP + T - 1) / T;
      u32 base_r[NIT];
      u32 peers_r[NIT];   // the groups of lanes that go to the same cell (a second __match_any per pass costs more than NIT registers)
      if (mp.fold) {
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
          base_r[it] = 0;
          peers_r[it] = 0;
          if (it * T < M) {
            const int t = it * T + tid;
            const u32 cnew = t < M ? s_id[t + sh] : CELL_DEAD;
            const u32 peers = __match_any_sync(0xffffffffu, cnew);
            if (cnew != CELL_DEAD && lane == __ffs(peers) - 1) base_r[it] = atomicAdd(&count[cnew], (u32)__popc(peers));
            peers_r[it] = peers;
          }
        }
      }
      if (moving) {
        for (int t = tid; t < M; t += T) {
          const u32 s = s0 + (u32)t;
          const int sl = t + sh;
          if (g.hx) a.x[s] = s_x[sl];
          if (g.hy) a.y[s] = s_y[sl];
          if (g.hz) a.z[s] = s_z[sl];
        }
      }
      if (mp.fold) {
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
          if (it * T < M) {
            const int t = it * T + tid;
            const bool in = t < M;
            const u32 cnew = in ? s_id[t + sh] : CELL_DEAD;
            const u32 peers = peers_r[it];
            const u32 base = __shfl_sync(0xffffffffu, base_r[it], __ffs(peers) - 1);
            if (in) {
              const u32 s = s0 + (u32)t;
              cell_out[s] = cnew;
              if (cnew != CELL_DEAD) off_out[s] = base + __popc(peers & ((1u << lane) - 1u));
            }
          }
        }
      }
    }
  }
  // integer counters by the warp-reduce instruction (REDUX), the flux by a butterfly in a fixed order
  const unsigned v0 = __reduce_add_sync(0xffffffffu, n_pairs), v1 = __reduce_add_sync(0xffffffffu, n_coll),
                 v2 = __reduce_add_sync(0xffffffffu, n_tie);
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) flux += __shfl_xor_sync(0xffffffffu, flux, d);
  if (lane == 0) {
    const int slot = (blockIdx.x * NW + warp) & (NSLOT - 1);
    if (v0) atomicAdd(&cnt.pairs[slot], (unsigned long long)v0);
    if (v1) atomicAdd(&cnt.collisions[slot], (unsigned long long)v1);
    if (v2) atomicAdd(&cnt.near_ties[slot], (unsigned long long)v2);
    s_flux[warp] = flux;
  }
  // rain flux: every thread sums its pairs in sorted order, the warp by a fixed butterfly, the CTA its warps in order, and
  // k_flux_sum the CTAs in order: the same bits run after run (atomics would add in arrival order)
  __syncthreads();
  if (tid == 0) {
    double f = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) f += s_flux[w];
    flux_part[blockIdx.x] = f;
  }
}

// Tile capacity and CTAs per SM by storage type (the kernel is bound by instruction issue and the latency of its square
// roots and reciprocals, so resident warps count): fp64 state 50 B of shared memory per SD -> 592 slots, 7 CTAs per SM;
// fp32 state 34 B per SD -> 864 slots, 7 CTAs.
#ifndef SDM_COAL_CAP
#define SDM_COAL_CAP 592
#define SDM_COAL_MINB 7
#endif
#ifndef SDM_COAL_CAP32
#define SDM_COAL_CAP32 864
#define SDM_COAL_MINB32 7
#endif
#ifndef SDM_COAL_T
#define SDM_COAL_T 128
#endif
template <typename R> constexpr int coal_minb() { return sizeof(R) == 4 ? SDM_COAL_MINB32 : SDM_COAL_MINB; }
template <typename R> constexpr int coal_cap() { return sizeof(R) == 4 ? SDM_COAL_CAP32 : SDM_COAL_CAP; }
// sparse cells (8 SDs per cell: the per-cell records, 88 B each, outweigh the SDs): fewer SD slots, room for 100 cells and more
template <typename R> constexpr int coal_cap_sparse() { return sizeof(R) == 4 ? 512 : 384; }
template <typename R, int CAP>
static bool coal_tile_fits_cap(int cpb, int need) {
  const size_t smem = CoalTile<CAP, SDM_COAL_T, R>::smem(cpb);
  return need + cpb <= CAP && cpb <= 4096 && smem <= (size_t)(228 * 1024 - coal_minb<R>() * 1024) / coal_minb<R>();
}
// can a tile of cpb cells whose most populated instance holds `need` SDs run in k_coal_move_tile?  1: the dense
// instantiation, 2: the sparse one, 0: no
template <typename R>
static int coal_tile_fits_t(int cpb, int need) {
  if (coal_tile_fits_cap<R, coal_cap<R>()>(cpb, need)) return 1;
  if (coal_tile_fits_cap<R, coal_cap_sparse<R>()>(cpb, need)) return 2;
  return 0;
}
bool coal_tile_fits(int cpb, int need, int real_bytes) {
  return (real_bytes == 8 ? coal_tile_fits_t<double>(cpb, need) : coal_tile_fits_t<float>(cpb, need)) != 0;
}
template <int CAP, typename R>
static cudaError_t launch_coal_move_tile_cap(int cpb, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g,
                                             const CellFields& cf, const CoalParams& kp, const CoalMoveParams& mp, double* flux_part,
                                             const Counters& cnt, u32* cell_out, u32* off_out, u32* count, cudaStream_t st) {
  const size_t smem = CoalTile<CAP, SDM_COAL_T, R>::smem(cpb);
  auto kern = k_coal_move_tile<CAP, SDM_COAL_T, coal_minb<R>(), R>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  CoalMoveParams mq = mp;
  mq.inv_dx = 1.0 / g.dx; mq.inv_dy = 1.0 / g.dy; mq.inv_dz = 1.0 / g.dz;
  kern<<<(g.ncell + cpb - 1) / cpb, SDM_COAL_T, smem, st>>>(a, rank, seg, g, cf, kp, mq, flux_part, cnt, cpb, cell_out, off_out, count);
  return cudaGetLastError();
}
template <typename R>
cudaError_t launch_coal_move_tile(int cpb, int need, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g,
                                  const CellFields& cf, const CoalParams& kp, const CoalMoveParams& mp, double* flux_part,
                                  const Counters& cnt, u32* cell_out, u32* off_out, u32* count, cudaStream_t st) {
  if (coal_tile_fits_t<R>(cpb, need) == 1)
    return launch_coal_move_tile_cap<coal_cap<R>(), R>(cpb, a, rank, seg, g, cf, kp, mp, flux_part, cnt, cell_out, off_out, count, st);
  return launch_coal_move_tile_cap<coal_cap_sparse<R>(), R>(cpb, a, rank, seg, g, cf, kp, mp, flux_part, cnt, cell_out, off_out, count, st);
}

// rain flux of the step: the per-CTA partial sums of k_coal_move_tile (n_part of them; every thread sums a strided subset in
// order, then a fixed tree) plus the NSLOT atomic slots of the per-cell kernel (summed in order, then cleared)
__global__ void __launch_bounds__(1024) k_flux_sum(double* flux_slots, const double* __restrict__ flux_part, int n_part, double* flux_out,
                                                   double* flux_total, const u32* __restrict__ d_flag) {
  __shared__ double sh[1024];
  double f = 0.0;
  for (int t = threadIdx.x; t < n_part; t += 1024) f += flux_part[t];
  for (int t = threadIdx.x; t < NSLOT; t += 1024) { f += flux_slots[t]; flux_slots[t] = 0.0; }
  sh[threadIdx.x] = f;
  __syncthreads();
  for (int d = 512; d >= 1; d >>= 1) {
    if ((int)threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    *flux_out = sh[0];
    *flux_total += sh[0];
    flux_out[2] = (double)*d_flag;   // the host reads flux and flag in one copy
  }
}

size_t coal_smem_bytes(int G, int cap, int sstp_coal, bool in_smem) {
  const int NG = (G <= 32 ? 128 : G) / G;
  const int P = sstp_coal > 1 ? next_pow2(cap) : 0;
  return (size_t)NG * ((size_t)cap * (in_smem ? 36 : 2) + (size_t)P * 10);
}

template <int G, typename R>
static cudaError_t launch_coal_move_t(int cap, bool in_smem, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g,
                                      const CellFields& cf, const CoalParams& kp, const CoalMoveParams& mp,
                                      double* flux_slots, const Counters& cnt, cudaStream_t st) {
  constexpr int NG = CtaOf<G>::threads / G;
  const int grid = (g.ncell + NG - 1) / NG;
  const bool multi = mp.sstp_coal > 1 || mp.coal_adapt_max > 1;
  const int P = multi ? next_pow2(cap) : 0;
  const size_t smem = coal_smem_bytes(G, cap, multi ? 2 : 1, in_smem);
  if (in_smem) {
    cudaError_t e = cudaFuncSetAttribute(k_coal_move<G, true, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_coal_move<G, true, R><<<grid, CtaOf<G>::threads, smem, st>>>(a, rank, seg, g, cf, kp, mp, flux_slots, cnt, cap, P);
  } else {
    cudaError_t e = cudaFuncSetAttribute(k_coal_move<G, false, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_coal_move<G, false, R><<<grid, CtaOf<G>::threads, smem, st>>>(a, rank, seg, g, cf, kp, mp, flux_slots, cnt, cap, P);
  }
  return cudaGetLastError();
}

template <typename R>
cudaError_t launch_coal_move(int G, int cap, bool in_smem, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g,
                             const CellFields& cf, const CoalParams& kp, const CoalMoveParams& mp, double* flux_slots,
                             const Counters& cnt, cudaStream_t st) {
  switch (G) {
    case 4: return launch_coal_move_t<4>(cap, in_smem, a, rank, seg, g, cf, kp, mp, flux_slots, cnt, st);
    case 8: return launch_coal_move_t<8>(cap, in_smem, a, rank, seg, g, cf, kp, mp, flux_slots, cnt, st);
    case 16: return launch_coal_move_t<16>(cap, in_smem, a, rank, seg, g, cf, kp, mp, flux_slots, cnt, st);
    case 32: return launch_coal_move_t<32>(cap, in_smem, a, rank, seg, g, cf, kp, mp, flux_slots, cnt, st);
    default: return launch_coal_move_t<256>(cap, in_smem, a, rank, seg, g, cf, kp, mp, flux_slots, cnt, st);
  }
}

#define SDM_INST(R)                                                                                                      \
  template cudaError_t launch_coal_move<R>(int, int, bool, const SdArraysT<R>&, const u16*, const u32*, const Grid&,          \
                                           const CellFields&, const CoalParams&, const CoalMoveParams&, double*, const Counters&, \
                                           cudaStream_t);                                                               \
  template cudaError_t launch_coal_move_tile<R>(int, int, const SdArraysT<R>&, const u16*, const u32*, const Grid&, const CellFields&, \
                                                const CoalParams&, const CoalMoveParams&, double*, const Counters&, u32*, u32*, u32*, \
                                                cudaStream_t);
SDM_INSTANTIATE_REAL(SDM_INST)
#undef SDM_INST

void launch_flux_sum(double* flux_slots, const double* flux_part, int n_part, double* flux_out, double* flux_total, const u32* d_flag,
                     cudaStream_t st) {
  k_flux_sum<<<1, 1024, 0, st>>>(flux_slots, flux_part, n_part, flux_out, flux_total, d_flag);
}

}  // namespace sdm
