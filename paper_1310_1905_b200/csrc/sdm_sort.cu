// Stage a0-a3 of the step: zero-multiplicity compaction, cell index, and the
// sort on (cell, Philox key, id) as an MSD radix sort: one counting pass over the cell index (global
// histogram + scan + scatter; dead SDs get no slot, which is the compaction) and a per-cell bitonic
// sort of (key << 32 | id) in shared memory that yields each SD's rank inside its cell.
// PAPER.md :547 (cell index), :624 (random non-overlapping pairs), :641/:651 (N = 0 SDs).
#include "sdm_kernels.cuh"
#include <algorithm>

namespace sdm {

// ---- a0/a1: cell index + histogram (warp-aggregated atomics) ----------------------------------------
template <typename R>
__global__ void __launch_bounds__(256) k_cellhist(SdArraysT<R> a, const u32* __restrict__ d_nslots, Grid g,
                                                  u32* __restrict__ cell, u32* __restrict__ off,
                                                  u32* __restrict__ count) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  const u32 nslots = *d_nslots;
  u32 c = CELL_DEAD;
  if (i < nslots) {   // position loads do not wait for the multiplicity
    const u64 n = a.n[i];
    const double x = g.hx ? (double)a.x[i] : 0.0, y = g.hy ? (double)a.y[i] : 0.0, z = g.hz ? (double)a.z[i] : 0.0;
    if (n != 0) c = cell_of(g, x, y, z);
  }
  // lanes that fall in the same cell take consecutive slots with one atomic
  const u32 peers = __match_any_sync(0xffffffffu, c);
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(peers) - 1;
  u32 base = 0;
  if (c != CELL_DEAD && lane == leader) base = atomicAdd(&count[c], (u32)__popc(peers));
  base = __shfl_sync(0xffffffffu, base, leader);
  if (i < nslots) {
    cell[i] = c;
    if (c != CELL_DEAD) off[i] = base + __popc(peers & ((1u << lane) - 1u));
  }
}

// ---- a2: exclusive scan of the histogram -> segment offsets (3 small kernels) -----------------------
constexpr int SCAN_THREADS = 1024, SCAN_ITEMS = 4, SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ u32 block_excl_scan(u32 v, u32* warp_sums, u32& total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  u32 inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const u32 t = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= d) inc += t;
  }
  if (lane == 31) warp_sums[w] = inc;
  __syncthreads();
  if (w == 0) {
    u32 s = warp_sums[lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const u32 t = __shfl_up_sync(0xffffffffu, s, d);
      if (lane >= d) s += t;
    }
    warp_sums[lane] = s;   // inclusive over warps
  }
  __syncthreads();
  total = warp_sums[31];
  return inc - v + (w ? warp_sums[w - 1] : 0u);
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_partial(const u32* __restrict__ count, int ncell,
                                                               u32* __restrict__ blocksum, u32* __restrict__ d_maxcount) {
  __shared__ u32 ws[32];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  u32 s = 0, mx = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k)
    if (base + k < ncell) { const u32 v = count[base + k]; s += v; mx = max(mx, v); }
  u32 total;
  block_excl_scan(s, ws, total);
  mx = __reduce_max_sync(0xffffffffu, mx);
  if ((threadIdx.x & 31) == 0 && mx) atomicMax(d_maxcount, mx);
  if (threadIdx.x == 0) blocksum[blockIdx.x] = total;
}

// one CTA: exclusive scan of the block sums; publishes the live count
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_blocks(u32* __restrict__ blocksum, int nblocks,
                                                              u32* __restrict__ d_nslots_next, u32* __restrict__ seg_total) {
  __shared__ u32 ws[32];
  u32 carry = 0;
  for (int b0 = 0; b0 < nblocks; b0 += SCAN_THREADS) {
    const int b = b0 + threadIdx.x;
    const u32 v = b < nblocks ? blocksum[b] : 0u;
    u32 total;
    const u32 ex = block_excl_scan(v, ws, total);
    if (b < nblocks) blocksum[b] = carry + ex;
    carry += total;
    __syncthreads();
  }
  if (threadIdx.x == 0) { *d_nslots_next = carry; *seg_total = carry; }
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(u32* __restrict__ count, int ncell,
                                                             const u32* __restrict__ blocksum, u32* __restrict__ seg) {
  __shared__ u32 ws[32];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  u32 v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = base + k < ncell ? count[base + k] : 0u; s += v[k]; }
  u32 total;
  u32 ex = block_excl_scan(s, ws, total) + blocksum[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k)
    if (base + k < ncell) { seg[base + k] = ex; ex += v[k]; count[base + k] = 0u; }   // histogram is left zeroed
}

// Most populated tile of cpb consecutive cells, for the 4 candidate tile sizes cpb_k = cpb0, 3/4, 1/2, 1/4 of it:
// picks the tile size of the tile-resident condensation kernel (sdm_cond.cu).
__host__ __device__ inline int tile_candidate(int cpb0, int k) { return max(1, (cpb0 * (4 - k)) / 4); }
int cond_tile_candidate(int cpb0, int k) { return tile_candidate(cpb0, k); }
__global__ void __launch_bounds__(256) k_tile_max(const u32* __restrict__ seg, int ncell, int cpb0, u32* __restrict__ out4) {
  for (int k = 0; k < 4; ++k) {
    const int cpb = tile_candidate(cpb0, k);
    const int ntile = (ncell + cpb - 1) / cpb;
    u32 mx = 0;
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < ntile; t += gridDim.x * blockDim.x)
      mx = max(mx, seg[min((t + 1) * cpb, ncell)] - seg[t * cpb]);
    mx = __reduce_max_sync(0xffffffffu, mx);
    if ((threadIdx.x & 31) == 0 && mx) atomicMax(&out4[k], mx);
  }
}

// ---- a3: scatter the SoA state into cell-sorted storage (drops dead SDs) ----------------------------
// The eight attributes move in SCATTER_PARTS = 2 launches of four attributes each (n, r_w^2, r_d^3, kappa | x, y, z, id), each
// of which reads the SD's cell and offset again: with all eight in one kernel (9 read and 8 scattered write streams at once)
// the reorder ran at 0.79 of the copy rate on its DRAM bytes, in two halves at 0.90 although they move 8 B per SD more
// (1.72 -> 1.55 ms at 67 M SDs; three parts 1.64, four 1.81, eight 2.81 ms: profiles/r2_k_scatter_ncu_full.md).  Populations of a few
// million SDs gain nothing (8.4 M: 0.176 / 0.174 ms) or lose the second launch (2.1 M: 0.053 -> 0.056 ms): one part below 2^24 SDs.
constexpr int SCATTER_PARTS = 2;
int scatter_parts(u32 nslots_bound) { return nslots_bound < (1u << 24) ? 1 : SCATTER_PARTS; }
template <typename R, int PARTS, int PART>
__global__ void __launch_bounds__(256) k_scatter(SdArraysT<R> src, SdArraysT<R> dst, const u32* __restrict__ d_nslots, Grid g,
                                                 const u32* __restrict__ cell, const u32* __restrict__ off,
                                                 const u32* __restrict__ seg) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= *d_nslots) return;
  constexpr auto mine = [](int k) { return k * PARTS / 8 == PART; };   // attribute k = n, rw2, rd3, kappa, x, y, z, id
  // all loads first, and none of them behind the test for a dead SD: the two copies of the state are not declared
  // disjoint, so a store between two loads would order them
  const u32 c = cell[i];
  const u32 o = off[i];
  u64 n = 0; R rw2 = R(0), rd3 = R(0), kappa = R(0), x = R(0), y = R(0), z = R(0); u32 id = 0;
  if (mine(0)) n = src.n[i];
  if (mine(1)) rw2 = src.rw2[i];
  if (mine(2)) rd3 = src.rd3[i];
  if (mine(3)) kappa = src.kappa[i];
  if (mine(4) && g.hx) x = src.x[i];
  if (mine(5) && g.hy) y = src.y[i];
  if (mine(6) && g.hz) z = src.z[i];
  if (mine(7)) id = src.id[i];
  if (c == CELL_DEAD) return;
  const u32 d = seg[c] + o;
  if (mine(0)) dst.n[d] = n;
  if (mine(1)) dst.rw2[d] = rw2;
  if (mine(2)) dst.rd3[d] = rd3;
  if (mine(3)) dst.kappa[d] = kappa;
  if (mine(4) && g.hx) dst.x[d] = x;
  if (mine(5) && g.hy) dst.y[d] = y;
  if (mine(6) && g.hz) dst.z[d] = z;
  if (mine(7)) dst.id[d] = id;
}
template <typename R, int PARTS, int PART = 0>
static void launch_scatter_parts(const SdArraysT<R>& src, const SdArraysT<R>& dst, const u32* d_nslots, u32 nslots_bound, const Grid& g,
                                 const u32* cell, const u32* off, const u32* seg, cudaStream_t st) {
  k_scatter<R, PARTS, PART><<<(nslots_bound + 255) / 256, 256, 0, st>>>(src, dst, d_nslots, g, cell, off, seg);
  if constexpr (PART + 1 < PARTS) launch_scatter_parts<R, PARTS, PART + 1>(src, dst, d_nslots, nslots_bound, g, cell, off, seg, st);
}

// ---- a2 (second level): rank of every SD inside its cell under (Philox key, id) ----------------------
// One group of G threads per cell.  Shared memory per group: P u64 keys + P u16 indices.
template <int G>
__global__ void __launch_bounds__(CtaOf<G>::threads) k_rank(const u32* __restrict__ id, const u32* __restrict__ seg,
                                                            int ncell, u32 step, u32 seed_lo, u32 seed_hi, int P,
                                                            u16* __restrict__ rank, int* __restrict__ d_error) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NG = CtaOf<G>::threads / G;
  const int gi = threadIdx.x / G;
  const Group<G> grp = make_group<G>(nullptr);
  const int c = blockIdx.x * NG + gi;
  if (c >= ncell) return;
  u64* skey = reinterpret_cast<u64*>(smem_raw) + (size_t)gi * P;
  u16* sidx = reinterpret_cast<u16*>(smem_raw + (size_t)NG * P * sizeof(u64)) + (size_t)gi * P;
  const u32 s0 = seg[c];
  const int m = (int)(seg[c + 1] - s0);
  if (m > P) {   // host sized P from the measured maximum; cannot happen unless the state was corrupted
    if (grp.lane == 0) atomicExch(d_error, 1);
    return;
  }
  if (m == 0) return;
  if (m == 1) { if (grp.lane == 0) rank[s0] = 0; return; }
  const int Pm = next_pow2(m);   // sort only as many slots as this cell needs
  for (int t = grp.lane; t < Pm; t += G) {
    u64 key = ~0ull;
    if (t < m) {
      const u32 sid = id[s0 + t];
      key = ((u64)shuffle_key(sid, step, 0u, seed_lo, seed_hi) << 32) | sid;
    }
    skey[t] = key;
    sidx[t] = (u16)t;
  }
  bitonic_sort<G, u16>(grp, skey, sidx, Pm);
  for (int t = grp.lane; t < m; t += G) rank[s0 + sidx[t]] = (u16)t;
}

// The same ranks for sparsely populated cells (m <= P <= 128) by COUNTING: the keys are unique, so the
// rank of an SD is the number of keys of its cell below its own.  m^2 broadcast compares out of shared
// memory instead of a log^2 network of barriers and swaps: no synchronisation after the keys are staged
// and 3 instructions per compare, which for the ~64 SDs per cell of the 3D workload is several times
// cheaper than the bitonic network (the network wins for hundreds of SDs per cell and stays in k_rank).
template <int G>
__global__ void __launch_bounds__(128) k_rank_count(const u32* __restrict__ id, const u32* __restrict__ seg, int ncell,
                                                    u32 step, u32 seed_lo, u32 seed_hi, int P, u16* __restrict__ rank,
                                                    int* __restrict__ d_error) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NG = 128 / G;
  const int gi = threadIdx.x / G;
  const Group<G> grp = make_group<G>(nullptr);
  const int c = blockIdx.x * NG + gi;
  if (c >= ncell) return;
  u64* skey = reinterpret_cast<u64*>(smem_raw) + (size_t)gi * P;
  const u32 s0 = seg[c];
  const int m = (int)(seg[c + 1] - s0);
  if (m > P) { if (grp.lane == 0) atomicExch(d_error, 1); return; }
  if (m == 0) return;
  const int m2 = (m + 1) & ~1;   // the compare loop reads key pairs; pad with the largest key
  for (int t = grp.lane; t < m2; t += G) {
    u64 key = ~0ull;
    if (t < m) {
      const u32 sid = id[s0 + t];
      key = ((u64)shuffle_key(sid, step, 0u, seed_lo, seed_hi) << 32) | sid;
    }
    skey[t] = key;
  }
  grp.sync();
  const ulonglong2* sk2 = reinterpret_cast<const ulonglong2*>(skey);
  for (int t0 = grp.lane; t0 < m; t0 += 2 * G) {   // two of this lane's SDs per sweep over the cell's keys
    const int t1 = t0 + G;
    const u64 k0 = skey[t0], k1 = t1 < m ? skey[t1] : 0ull;
    int r0 = 0, r1 = 0;
#pragma unroll 4
    for (int j = 0; j < (m2 >> 1); ++j) {
      const ulonglong2 kk = sk2[j];
      r0 += (kk.x < k0) + (kk.y < k0);
      r1 += (kk.x < k1) + (kk.y < k1);
    }
    rank[s0 + t0] = (u16)r0;
    if (t1 < m) rank[s0 + t1] = (u16)r1;
  }
}

// Ranks for cells of tens to thousands of SDs (m <= 8192) by BUCKETS: the Philox keys are uniform, so the top bits of the key
// split a cell's SDs into P/16 buckets of ~16; a histogram and a scan give every bucket its place, the keys are
// scattered bucket by bucket, and an SD's rank is the start of its bucket plus the number of smaller keys inside
// it: ~16 compares per SD instead of the log^2 m barriers and swaps of the bitonic network (which stays for cells
// beyond 8192 SDs).  G = 32: a warp per cell, 4 cells per CTA; G = 256: a CTA per cell.
// Shared memory per group: u64 keys[P], u64 sorted[P], u32 hist[P/16].
// Buckets per cell for P key slots (P = the largest cell, rounded up to a power of two).  The compare loop inside the bucket is half
// of the kernel's instructions at ~8 keys per bucket, the histogram and its scan are cheap while they fit a few words per lane:
// ~2 keys per bucket up to 128 buckets (a cell of 64 SDs in P = 128: 0.73 -> 0.59 ms at 67 M SDs), ~16 for the CTA-wide path of
// crowded cells, whose scan runs on one warp.
#ifdef SDM_RANK_BUCKET_SHIFT
__host__ __device__ inline int rank_buckets(int P) { return (P >> SDM_RANK_BUCKET_SHIFT) > 4 ? (P >> SDM_RANK_BUCKET_SHIFT) : 4; }
#else
__host__ __device__ inline int rank_buckets(int P) {
  const int nb = P <= 256 ? P >> 1 : P <= 512 ? P >> 2 : P >> 4;
  return nb > 4 ? nb : 4;
}
#endif
template <int G>
__global__ void __launch_bounds__(CtaOf<G>::threads) k_rank_bucket(const u32* __restrict__ id, const u32* __restrict__ seg,
                                                                   int ncell, u32 step, u32 seed_lo, u32 seed_hi, int P,
                                                                   u16* __restrict__ rank, int* __restrict__ d_error) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NG = CtaOf<G>::threads / G;
  const int gi = threadIdx.x / G;
  const Group<G> grp = make_group<G>(nullptr);
  const int NB = rank_buckets(P);              // buckets (power of two)
  const int shift = 64 - (31 - __clz(NB));     // key >> shift = bucket
  unsigned char* base = smem_raw + (size_t)gi * ((size_t)P * 16 + (size_t)NB * 4);
  u64* skey = reinterpret_cast<u64*>(base);
  u64* ssort = skey + P;
  u32* hist = reinterpret_cast<u32*>(ssort + P);
  const int c = blockIdx.x * NG + gi;
  const bool live = c < ncell;                 // (no early return: CTA-wide groups meet at barriers)
  const u32 s0 = live ? seg[c] : 0u;
  int m = live ? (int)(seg[c + 1] - s0) : 0;
  if (m > P) { if (grp.lane == 0) atomicExch(d_error, 1); m = 0; }
  for (int b = grp.lane; b < NB; b += G) hist[b] = 0u;
  grp.sync();
  for (int t = grp.lane; t < m; t += G) {
    const u32 sid = id[s0 + t];
    const u64 key = ((u64)shuffle_key(sid, step, 0u, seed_lo, seed_hi) << 32) | sid;
    skey[t] = key;
    atomicAdd(&hist[(u32)(key >> shift)], 1u);
  }
  grp.sync();
  // exclusive scan of the histogram by the first W = min(G, 32) lanes of the group (NB/W consecutive buckets each)
  constexpr int W = G < 32 ? G : 32;
  if (grp.lane < W) {
    const int per = max(NB / W, 1);
    const int b0 = grp.lane * per;
    u32 sum = 0;
    if (b0 < NB) for (int b = b0; b < b0 + per; ++b) sum += hist[b];
    u32 inc = sum;
    const u32 mask = G >= 32 ? 0xffffffffu : grp.mask;
#pragma unroll
    for (int d = 1; d < W; d <<= 1) { const u32 v = __shfl_up_sync(mask, inc, d, W); if (grp.lane >= d) inc += v; }
    u32 run = inc - sum;
    if (b0 < NB) for (int b = b0; b < b0 + per; ++b) { const u32 h = hist[b]; hist[b] = run; run += h; }
  }
  grp.sync();
  for (int t = grp.lane; t < m; t += G) {      // scatter; afterwards hist[b] = end of bucket b
    const u64 key = skey[t];
    ssort[atomicAdd(&hist[(u32)(key >> shift)], 1u)] = key;
  }
  grp.sync();
  for (int t = grp.lane; t < m; t += G) {
    const u64 key = skey[t];
    const u32 b = (u32)(key >> shift);
    const int lo = b ? (int)hist[b - 1] : 0, hi = (int)hist[b];
    int r = lo;
    if constexpr (G < 256) {   // ~2 keys per bucket: a 4-fold unrolled loop with its remainder costs more than it saves (0.59 -> 0.54 ms)
#pragma unroll 1
      for (int j = lo; j < hi; ++j) r += (ssort[j] < key);
    } else {
      for (int j = lo; j < hi; ++j) r += (ssort[j] < key);
    }
    rank[s0 + t] = (u16)r;
  }
}

// ids in sorted order (parity export)
__global__ void k_export_order(const u32* __restrict__ id, const u16* __restrict__ rank, const u32* __restrict__ seg,
                               int ncell, u32* __restrict__ ids_sorted) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  const u32 s0 = seg[c], s1 = seg[c + 1];
  for (u32 s = s0; s < s1; ++s) ids_sorted[s0 + rank[s]] = id[s];
}

// ---- host launchers ----------------------------------------------------------------------------------
template <typename R>
void launch_cellhist(const SdArraysT<R>& a, const u32* d_nslots, u32 nslots_bound, const Grid& g, u32* cell, u32* off,
                     u32* count, cudaStream_t st) {
  if (nslots_bound == 0) return;
  k_cellhist<R><<<(nslots_bound + 255) / 256, 256, 0, st>>>(a, d_nslots, g, cell, off, count);
}

int scan_num_blocks(int ncell) { return (ncell + SCAN_TILE - 1) / SCAN_TILE; }

void launch_scan(u32* count, int ncell, u32* blocksum, u32* seg, u32* d_nslots_next, u32* d_maxcount, cudaStream_t st) {
  const int nb = scan_num_blocks(ncell);
  k_scan_partial<<<nb, SCAN_THREADS, 0, st>>>(count, ncell, blocksum, d_maxcount);
  k_scan_blocks<<<1, SCAN_THREADS, 0, st>>>(blocksum, nb, d_nslots_next, seg + ncell);
  k_scan_apply<<<nb, SCAN_THREADS, 0, st>>>(count, ncell, blocksum, seg);
}

void launch_tile_max(const u32* seg, int ncell, int cpb0, u32* d_tilemax4, cudaStream_t st) {
  const int nb = std::min((ncell + 255) / 256, 1184);
  k_tile_max<<<nb, 256, 0, st>>>(seg, ncell, cpb0, d_tilemax4);
}

template <typename R>
void launch_scatter(const SdArraysT<R>& src, const SdArraysT<R>& dst, const u32* d_nslots, u32 nslots_bound, const Grid& g,
                    const u32* cell, const u32* off, const u32* seg, cudaStream_t st) {
  if (nslots_bound == 0) return;
  if (scatter_parts(nslots_bound) == 1) launch_scatter_parts<R, 1>(src, dst, d_nslots, nslots_bound, g, cell, off, seg, st);
  else launch_scatter_parts<R, SCATTER_PARTS>(src, dst, d_nslots, nslots_bound, g, cell, off, seg, st);
}

#define SDM_INST(R)                                                                                              \
  template void launch_cellhist<R>(const SdArraysT<R>&, const u32*, u32, const Grid&, u32*, u32*, u32*, cudaStream_t); \
  template void launch_scatter<R>(const SdArraysT<R>&, const SdArraysT<R>&, const u32*, u32, const Grid&, const u32*,  \
                                  const u32*, const u32*, cudaStream_t);
SDM_INSTANTIATE_REAL(SDM_INST)
#undef SDM_INST

template <int G>
static cudaError_t launch_rank_t(const u32* id, const u32* seg, int ncell, u32 step, u32 seed_lo, u32 seed_hi, int P,
                                 u16* rank, int* d_error, cudaStream_t st) {
  constexpr int NG = CtaOf<G>::threads / G;
  const size_t smem = (size_t)NG * P * (sizeof(u64) + sizeof(u16));
  cudaError_t e = cudaFuncSetAttribute(k_rank<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_rank<G><<<(ncell + NG - 1) / NG, CtaOf<G>::threads, smem, st>>>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error);
  return cudaGetLastError();
}

template <int G>
static cudaError_t launch_rank_count_t(const u32* id, const u32* seg, int ncell, u32 step, u32 seed_lo, u32 seed_hi, int P,
                                       u16* rank, int* d_error, cudaStream_t st) {
  constexpr int NG = 128 / G;
  k_rank_count<G><<<(ncell + NG - 1) / NG, 128, (size_t)NG * P * sizeof(u64), st>>>(id, seg, ncell, step, seed_lo, seed_hi, P,
                                                                                  rank, d_error);
  return cudaGetLastError();
}

// P = power of two >= the most populated cell.  Sparse cells (P < 64, or small groups) take their ranks from
// counting all pairs, cells up to 8192 SDs from counting inside key buckets, beyond that from the bitonic network.
template <int G>
static cudaError_t launch_rank_bucket_t(const u32* id, const u32* seg, int ncell, u32 step, u32 seed_lo, u32 seed_hi, int P,
                                        u16* rank, int* d_error, cudaStream_t st) {
  constexpr int NG = CtaOf<G>::threads / G;
  const size_t smem = (size_t)NG * ((size_t)P * 16 + (size_t)rank_buckets(P) * 4);
  cudaError_t e = cudaFuncSetAttribute(k_rank_bucket<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_rank_bucket<G><<<(ncell + NG - 1) / NG, CtaOf<G>::threads, smem, st>>>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error);
  return cudaGetLastError();
}

cudaError_t launch_rank(int G, const u32* id, const u32* seg, int ncell, u32 step, u32 seed_lo, u32 seed_hi, int P,
                        u16* rank, int* d_error, cudaStream_t st) {
  if (P >= 256 && P <= 8192) {   // crowded cells: buckets (a warp per cell up to 512 SDs, else a CTA)
    if (P <= 512) return launch_rank_bucket_t<32>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
    return launch_rank_bucket_t<256>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
  }
  if (P >= 64 && P <= 128 && (G == 16 || G == 32)) {   // measured: buckets beat all-pairs counting from ~30 SDs per cell on
    if (G == 16) return launch_rank_bucket_t<16>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
    return launch_rank_bucket_t<32>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
  }
  if (P <= 128 && G <= 32) {
    switch (G) {
      case 4: return launch_rank_count_t<4>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
      case 8: return launch_rank_count_t<8>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
      case 16: return launch_rank_count_t<16>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
      default: return launch_rank_count_t<32>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
    }
  }
  switch (G) {
    case 4: return launch_rank_t<4>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
    case 8: return launch_rank_t<8>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
    case 16: return launch_rank_t<16>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
    case 32: return launch_rank_t<32>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
    default: return launch_rank_t<256>(id, seg, ncell, step, seed_lo, seed_hi, P, rank, d_error, st);
  }
}

void launch_export_order(const u32* id, const u16* rank, const u32* seg, int ncell, u32* ids_sorted, cudaStream_t st) {
  k_export_order<<<(ncell + 127) / 128, 128, 0, st>>>(id, rank, seg, ncell, ids_sorted);
}

}  // namespace sdm
