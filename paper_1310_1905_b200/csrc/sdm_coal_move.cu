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
      const double dtpp = g.dt / mp.sstp_coal;
      int nc = m;   // SDs taking part in this substep
      for (int sub = 0; sub < mp.sstp_coal; ++sub) {
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
            prw2[k] = r * r;
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
        if (g.hx) { xn = wrap(xn, g.X); a.x[s] = xn; }                        // periodic (:558)
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
// A CTA of T threads owns a tile of `cpb` consecutive cells (at most CAP - cpb SDs).  n, r_w^2, id and the
// positions of the tile's SDs are copied into shared memory IN STORAGE ORDER by asynchronous copies
// (cp.async: no registers, no stall, every copy of the tile in flight at once); the sorted order enters
// through an inverse map inv[sorted position] = slot, built with every cell's segment padded to an even
// length, so that thread t owns the pair of sorted positions (2t, 2t+1): all lanes are busy whatever
// the cell populations are.  r_d^3 and kappa are touched (in global memory) only by the rare pairs that
// collide, and n, r_w^2 are written back only where they changed: per SD the kernel reads 46 B and writes
// 24 B of HBM.  The terminal velocity of every SD is evaluated once, in the pair pass (the lone SD of an
// odd cell by the thread of its padded slot), and reused by the sedimentation.  The arithmetic is,
// expression by expression, that of k_coal_move above (-fmad=false).
#ifndef SDM_COAL_UNROLL
#define SDM_COAL_UNROLL 1
#endif
constexpr int kCoalUnroll = SDM_COAL_UNROLL;
struct __align__(8) CoalCell {
  double eta, rho_a, scale;                 // air properties; eq. 27 factor n(n-1)/2 / floor(n/2)
  double Cxl, Cxh, Cyl, Cyh, Czl, Czh;      // Courant numbers at the cell's faces (rho_d C / rho_d)
  int i, j, k, pad;
};

template <int CAP, int T, typename R>
struct CoalTile {   // u64 n; R rw2, x, y, z; double vt; u32 id; u16 inv
  static_assert(CAP % 16 == 0, "the arrays of the tile follow one another in shared memory: keep every one of them 16-byte aligned");
  static constexpr size_t fixed_bytes = (size_t)CAP * (8 + 4 * sizeof(R) + 8 + 4 + 2);
  static size_t smem(int cpb) { return fixed_bytes + (size_t)cpb * sizeof(CoalCell) + (size_t)(cpb + 1) * 8 + 16; }
};

template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(d), "l"(gmem_src), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <int CAP, int T, int MINB, typename R>
__global__ void __launch_bounds__(T, MINB)
k_coal_move_tile(SdArraysT<R> a, const u16* __restrict__ rank, const u32* __restrict__ seg, Grid g, CellFields cf, CoalParams kp,
                 CoalMoveParams mp, double* flux_slots, Counters cnt, int cpb) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using L = CoalTile<CAP, T, R>;
  constexpr u16 NONE = 0xFFFFu;
  const int tid = threadIdx.x;
  const int c_first = blockIdx.x * cpb;
  const int nc = min(cpb, g.ncell - c_first);
  u64* s_n = reinterpret_cast<u64*>(smem_raw);
  double* s_vt = reinterpret_cast<double*>(smem_raw) + CAP;
  R* s_rw2 = reinterpret_cast<R*>(s_vt + CAP);
  R* s_x = s_rw2 + CAP;
  R* s_y = s_x + CAP;
  R* s_z = s_y + CAP;
  u32* s_id = reinterpret_cast<u32*>(s_z + CAP);
  u16* inv = reinterpret_cast<u16*>(s_id + CAP);
  CoalCell* s_cell = reinterpret_cast<CoalCell*>(smem_raw + L::fixed_bytes);
  u32* segl = reinterpret_cast<u32*>(s_cell + cpb);   // storage offsets of the tile's cells
  u32* segp = segl + cpb + 1;                          // padded (even) offsets of the sorted positions
  const u32 s0 = seg[c_first];
  const int M = (int)(seg[c_first + nc] - s0);
  const bool moving = mp.adve || mp.sedi;
  const bool need_vt = mp.sedi && g.hz;
  unsigned n_pairs = 0, n_coll = 0, n_tie = 0;
  double flux = 0.0;
  if (M > 0) {
    // everything that does not need the sorted order starts right away
#pragma unroll kCoalUnroll
    for (int t = tid; t < M; t += T) {
      const u32 s = s0 + t;
      cp_async<8>(s_n + t, a.n + s);
      cp_async<sizeof(R)>(s_rw2 + t, a.rw2 + s);
      if (mp.coal) cp_async<4>(s_id + t, a.id + s);
      if (moving) {
        if (g.hx) cp_async<sizeof(R)>(s_x + t, a.x + s);
        if (g.hy) cp_async<sizeof(R)>(s_y + t, a.y + s);
        if (g.hz) cp_async<sizeof(R)>(s_z + t, a.z + s);
      }
    }
    for (int cl = tid; cl < nc; cl += T) {
      const int c = c_first + cl;
      const u32 b0 = seg[c], b1 = seg[c + 1];
      segl[cl] = b0 - s0;
      const int m = (int)(b1 - b0);
      CoalCell& C = s_cell[cl];
      C.eta = cf.eta[c]; C.rho_a = cf.rho_a[c];
      C.scale = m >= 2 ? (double)((u64)m * (u64)(m - 1) / 2) / (double)(m / 2) : 0.0;
      const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
      C.i = i; C.j = j; C.k = k;
      const double rhod = cf.rhod[c];
      C.Cxl = C.Cxh = C.Cyl = C.Cyh = C.Czl = C.Czh = 0.0;
      if (mp.adve) {
        if (g.hx) { C.Cxl = cf.cx[((long long)i * g.NY + j) * g.NZ + k] / rhod; C.Cxh = cf.cx[((long long)(i + 1) * g.NY + j) * g.NZ + k] / rhod; }
        if (g.hy) { C.Cyl = cf.cy[((long long)i * (g.NY + 1) + j) * g.NZ + k] / rhod; C.Cyh = cf.cy[((long long)i * (g.NY + 1) + j + 1) * g.NZ + k] / rhod; }
        if (g.hz) { C.Czl = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k] / rhod; C.Czh = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k + 1] / rhod; }
      }
    }
    if (tid == 0) segl[nc] = (u32)M;
    __syncthreads();
    if (tid < 32) {   // padded offsets: warp scan over the cells, 32 at a time
      u32 carry = 0;
      for (int c0 = 0; c0 <= nc; c0 += 32) {
        const int cl = c0 + tid;
        u32 v = 0;
        if (cl < nc) { const u32 m = segl[cl + 1] - segl[cl]; v = m + (m & 1u); }
        u32 inc = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const u32 t = __shfl_up_sync(0xffffffffu, inc, d); if (tid >= d) inc += t; }
        if (cl <= nc) segp[cl] = carry + inc - v;
        carry += __shfl_sync(0xffffffffu, inc, 31);
      }
    }
    __syncthreads();
    const int MP = (int)segp[nc];
    // inverse map of the sorted order
    for (int t = tid; t < M; t += T) {
      int lo = 0, hi = nc;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)t) lo = mid; else hi = mid; }
      inv[(int)segp[lo] + rank[s0 + t]] = (u16)t;
    }
    for (int cl = tid; cl < nc; cl += T) {   // the padding slot of an odd cell
      const u32 m = segl[cl + 1] - segl[cl];
      if (m & 1u) inv[segp[cl] + m] = NONE;
    }
    cp_async_wait_all();
    __syncthreads();
    // ---- pairs of sorted positions (2t, 2t+1) -------------------------------------------------------------
    if (mp.coal || need_vt) {
      const double dtdv = g.dt / g.dV;
      for (int t = tid; 2 * t < MP; t += T) {
        const u32 both = reinterpret_cast<const u32*>(inv)[t];
        const int ia = (int)(both & 0xFFFFu), ib = (int)(both >> 16);
        const bool lone = ib == (int)NONE;
        int lo = 0, hi = nc;   // the pair's cell: segp[lo] <= 2t < segp[lo + 1]
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segp[mid] <= (u32)(2 * t)) lo = mid; else hi = mid; }
        const CoalCell& C = s_cell[lo];
        const double ya = s_rw2[ia];
        const double ra = sqrt(ya);
        if (lone || !mp.coal) {
          if (need_vt) {
            s_vt[ia] = v_term(ra, C.eta, C.rho_a);
            if (!lone) s_vt[ib] = v_term(sqrt((double)s_rw2[ib]), C.eta, C.rho_a);
          }
          continue;
        }
        const u64 na = s_n[ia], nb = s_n[ib];
        const double yb = s_rw2[ib];
        const double rb = sqrt(yb);
        const bool afirst = na >= nb;            // j: larger N; tie -> first in order
        const int j = afirst ? ia : ib, k = afirst ? ib : ia;
        const u64 nj = afirst ? na : nb, nk = afirst ? nb : na;
        const double yj = afirst ? ya : yb, yk = afirst ? yb : ya;
        const double rj = afirst ? ra : rb, rk = afirst ? rb : ra;
        double K;
        if (kp.kernel == 1) {   // Golovin
          const double vj = (4.0 / 3.0) * cst::pi * (yj * rj), vk = (4.0 / 3.0) * cst::pi * (yk * rk);
          K = kp.golovin_b * (vj + vk);
          if (need_vt) { s_vt[j] = v_term(rj, C.eta, C.rho_a); s_vt[k] = v_term(rk, C.eta, C.rho_a); }
        } else {                // eq. 28
          const double vj = v_term(rj, C.eta, C.rho_a), vk = v_term(rk, C.eta, C.rho_a);
          s_vt[j] = vj; s_vt[k] = vk;
          K = cst::pi * ((rj + rk) * (rj + rk)) * fabs(vj - vk);
          if (kp.kernel == 2) {
            const double rl = fmax(rj, rk), rs = fmin(rj, rk);
            K = K * eff_lookup(kp, rl, rs / rl);
          }
        }
        const double p = (((double)nj * K) * dtdv) * C.scale;   // eq. 27
        const double u = coal_uniform(s_id[ia], mp.step, 0u, kp.seed_lo, kp.seed_hi);
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
        // the rare pair that collides updates global memory itself (r_d^3 and kappa are not staged)
        const u32 gj = s0 + (u32)j, gk = s0 + (u32)k;
        const double gd = (double)gam;
        const double rw3 = yk * rk + gd * (yj * rj);    // extensive attributes are summed (:643)
        const double rd3j = gd * a.rd3[gj];
        const double rd3k = a.rd3[gk];
        const double kj = a.kappa[gj], kk = a.kappa[gk];
        if (kj != kk)                                    // intensive ones averaged (:643)
          a.kappa[gk] = (rd3j * kj + rd3k * kk) / (rd3j + rd3k);
        a.rd3[gk] = rd3k + rd3j;
        const double r = cbrt(rw3);
        const double y2 = (R)(r * r);   // what is stored is the radius from here on
        s_rw2[k] = (R)y2; a.rw2[gk] = (R)y2;
        s_n[j] = nj - gam * nk; a.n[gj] = nj - gam * nk;
        if (need_vt) s_vt[k] = v_term(sqrt(y2), C.eta, C.rho_a);
      }
      __syncthreads();
    }
    // ---- advection + sedimentation, SD by SD in storage order; everything is in shared memory -----------------
    if (moving) {
#pragma unroll kCoalUnroll
      for (int t = tid; t < M; t += T) {
        const u64 n = s_n[t];
        if (n == 0) continue;
        int lo = 0, hi = nc;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (segl[mid] <= (u32)t) lo = mid; else hi = mid; }
        const u32 s = s0 + t;
        const CoalCell& C = s_cell[lo];
        double xn = 0, yn = 0, zn = 0;
        if (g.hx) xn = s_x[t];
        if (g.hy) yn = s_y[t];
        if (g.hz) zn = s_z[t];
        if (mp.adve) {   // eq. 16 with the Courant numbers at the edges of the SD's time-n cell
          if (g.hx) { const double dC = C.Cxh - C.Cxl; xn = (xn + g.dx * (C.Cxl - (double)C.i * dC)) / (1.0 - dC); }
          if (g.hy) { const double dC = C.Cyh - C.Cyl; yn = (yn + g.dy * (C.Cyl - (double)C.j * dC)) / (1.0 - dC); }
          if (g.hz) { const double dC = C.Czh - C.Czl; zn = (zn + g.dz * (C.Czl - (double)C.k * dC)) / (1.0 - dC); }
        }
        if (need_vt) zn = zn - s_vt[t] * g.dt;                                // explicit Euler (:649)
        if (g.hx) { xn = wrap(xn, g.X); a.x[s] = xn; }                        // periodic (:558)
        if (g.hy) { yn = wrap(yn, g.Y); a.y[s] = yn; }
        if (g.hz) {
          if (zn < 0.0 || !(zn < g.Z)) {                                       // left the domain (:651)
            const double y = s_rw2[t];
            if (zn < 0.0) flux += (double)n * ((4.0 / 3.0) * cst::pi * cst::rho_w * (y * sqrt(y)));
            a.n[s] = 0;
          }
          a.z[s] = zn;
        }
      }
    }
  }
  unsigned v0 = n_pairs, v1 = n_coll, v2 = n_tie;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    v0 += __shfl_xor_sync(0xffffffffu, v0, d);
    v1 += __shfl_xor_sync(0xffffffffu, v1, d);
    v2 += __shfl_xor_sync(0xffffffffu, v2, d);
    flux += __shfl_xor_sync(0xffffffffu, flux, d);
  }
  if ((threadIdx.x & 31) == 0) {
    const int slot = (blockIdx.x * (T / 32) + (threadIdx.x >> 5)) & (NSLOT - 1);
    if (v0) atomicAdd(&cnt.pairs[slot], (unsigned long long)v0);
    if (v1) atomicAdd(&cnt.collisions[slot], (unsigned long long)v1);
    if (v2) atomicAdd(&cnt.near_ties[slot], (unsigned long long)v2);
    if (flux != 0.0) atomicAdd(&flux_slots[slot], flux);
  }
}

// Tile capacity and CTAs per SM by storage type (swept on the 3D workload at 16.7 M SDs; the kernel is bound by the latency
// of its IEEE divisions and square roots, so resident warps count): fp64 state 58 B of shared memory per SD -> 560 slots,
// 7 CTAs per SM, 72 registers (672 / 6: +7 %, 816 / 5: +17 %, 448 / 8: +7 %); fp32 state 38 B per SD -> 816 slots, 7 CTAs,
// 72 registers (5 CTAs: +23 %, 704 / 8: the same, 560 / 10: +9 %).  No spills in either.
#ifndef SDM_COAL_CAP
#define SDM_COAL_CAP 560
#define SDM_COAL_MINB 7
#endif
#ifndef SDM_COAL_CAP32
#define SDM_COAL_CAP32 816
#define SDM_COAL_MINB32 7
#endif
#ifndef SDM_COAL_T
#define SDM_COAL_T 128
#endif
template <typename R> constexpr int coal_minb() { return sizeof(R) == 4 ? SDM_COAL_MINB32 : SDM_COAL_MINB; }
template <typename R> constexpr int coal_cap() { return sizeof(R) == 4 ? SDM_COAL_CAP32 : SDM_COAL_CAP; }
// can a tile of cpb cells whose most populated instance holds `need` SDs run in k_coal_move_tile?
template <typename R>
static bool coal_tile_fits_t(int cpb, int need) {
  const size_t smem = CoalTile<coal_cap<R>(), SDM_COAL_T, R>::smem(cpb);
  return need + cpb <= coal_cap<R>() && cpb <= 4096 && smem <= (size_t)(228 * 1024 - coal_minb<R>() * 1024) / coal_minb<R>();
}
bool coal_tile_fits(int cpb, int need, int real_bytes) {
  return real_bytes == 8 ? coal_tile_fits_t<double>(cpb, need) : coal_tile_fits_t<float>(cpb, need);
}
template <typename R>
cudaError_t launch_coal_move_tile(int cpb, const SdArraysT<R>& a, const u16* rank, const u32* seg, const Grid& g,
                                  const CellFields& cf, const CoalParams& kp, const CoalMoveParams& mp, double* flux_slots,
                                  const Counters& cnt, cudaStream_t st) {
  const size_t smem = CoalTile<coal_cap<R>(), SDM_COAL_T, R>::smem(cpb);
  auto kern = k_coal_move_tile<coal_cap<R>(), SDM_COAL_T, coal_minb<R>(), R>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  kern<<<(g.ncell + cpb - 1) / cpb, SDM_COAL_T, smem, st>>>(a, rank, seg, g, cf, kp, mp, flux_slots, cnt, cpb);
  return cudaGetLastError();
}

// sums the NSLOT flux slots in a fixed order, then clears them
__global__ void k_flux_sum(double* flux_slots, double* flux_out, double* flux_total) {
  __shared__ double sh[NSLOT];
  for (int t = threadIdx.x; t < NSLOT; t += blockDim.x) { sh[t] = flux_slots[t]; flux_slots[t] = 0.0; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int t = 0; t < NSLOT; ++t) s += sh[t];
    *flux_out = s;
    *flux_total += s;
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
  const int P = mp.sstp_coal > 1 ? next_pow2(cap) : 0;
  const size_t smem = coal_smem_bytes(G, cap, mp.sstp_coal, in_smem);
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
  template cudaError_t launch_coal_move_tile<R>(int, const SdArraysT<R>&, const u16*, const u32*, const Grid&, const CellFields&, \
                                                const CoalParams&, const CoalMoveParams&, double*, const Counters&, cudaStream_t);
SDM_INSTANTIATE_REAL(SDM_INST)
#undef SDM_INST

void launch_flux_sum(const double* flux_slots, double* flux_out, double* flux_total, cudaStream_t st) {
  k_flux_sum<<<1, 256, 0, st>>>(const_cast<double*>(flux_slots), flux_out, flux_total);
}

}  // namespace sdm
