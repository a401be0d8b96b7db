// Recycling of zero-multiplicity super-droplets (PAPER.md :641 "Particles with zero multiplicity are 'recycled' at
// the begining of each timestep.  The recycling procedure first looks for computational particles with highest
// multiplicites and then assignes their properties to the recycled particles halving the multiplicity"; :651 the
// same for SDs that left the domain).  DESIGN.md reading R-recycle: with k dead SDs, the donors are the first k SDs
// in the order (multiplicity descending, id ascending) among those with multiplicity >= 2; the i-th donor serves the
// dead SD of i-th smallest id, which takes the donor's r_w^2, r_d^3, kappa and position, keeps its id and gets
// floor(N/2); the donor keeps N - floor(N/2).
//
// The paper's implementation sorts all SDs by multiplicity.  Here the k-th largest multiplicity is located with one
// histogram pass over N (2048 logarithmic bins, 32 per octave, built in shared memory), only the SDs in or above the
// threshold bin are collected (k plus the population of one bin), and that short list is ordered exactly by a
// bitonic network on (~N, id).  Three passes over the 8-byte multiplicities instead of a 67 M-element sort.
#include "sdm_kernels.cuh"
#include <algorithm>

namespace sdm {

namespace {

constexpr int REC_BINS = 2048;
constexpr int SORT_TILE = 2048;   // items one CTA orders in shared memory (32 KB)

// monotone non-decreasing in n for n >= 2: 32 bins per octave
__device__ __forceinline__ int rec_bin(u64 n) {
  const int lz = 63 - __clzll((long long)n);   // position of the leading bit, 1..63
  const u32 sub = lz >= 5 ? (u32)(n >> (lz - 5)) & 31u : (u32)(n << (5 - lz)) & 31u;
  return lz * 32 + (int)sub;
}

// info: [0] dead SDs, [1] k = SDs to recycle, [2] candidates collected, [3] threshold bin, [4] append counter
__global__ void __launch_bounds__(256) k_rec_scan(const u64* __restrict__ n, const u32* __restrict__ id, u32 nslots,
                                                  RecItem* __restrict__ dead, u32* __restrict__ info, u32* __restrict__ hist) {
  __shared__ u32 sh[REC_BINS];
  for (int b = threadIdx.x; b < REC_BINS; b += blockDim.x) sh[b] = 0u;
  __syncthreads();
  const u32 stride = gridDim.x * blockDim.x;
  for (u32 s = blockIdx.x * blockDim.x + threadIdx.x; s < nslots; s += stride) {
    const u64 v = n[s];
    if (v == 0) {
      const u32 w = atomicAdd(&info[0], 1u);
      dead[w] = RecItem{0ull, id[s], s};
    } else if (v >= 2) {
      atomicAdd(&sh[rec_bin(v)], 1u);
    }
  }
  __syncthreads();
  for (int b = threadIdx.x; b < REC_BINS; b += blockDim.x)
    if (sh[b]) atomicAdd(&hist[b], sh[b]);
}

// one warp: k = min(dead, donors); threshold bin = the highest bin b with count(bins >= b) >= k
__global__ void k_rec_threshold(u32* __restrict__ info, const u32* __restrict__ hist) {
  const int lane = threadIdx.x;
  const u32 nd = info[0];
  u32 above = 0;   // population of the bins above the current group of 32
  int bstar = 0;
  u32 k = 0;
  bool found = false;
  for (int base = REC_BINS - 32; base >= 0 && !found; base -= 32) {
    const u32 c = hist[base + lane];
    // suffix sum inside the group: lanes holding higher bins first
    u32 suf = c;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const u32 o = __shfl_down_sync(0xffffffffu, suf, d);
      if (lane + d < 32) suf += o;
    }
    const unsigned hit = __ballot_sync(0xffffffffu, above + suf >= nd);
    if (hit && nd > 0) {
      bstar = base + (31 - __clz((int)hit));
      found = true;
      k = nd;
    }
    above += __shfl_sync(0xffffffffu, suf, 0);
  }
  if (!found) { bstar = 0; k = min(nd, above); }   // fewer donors than dead SDs: all of them give
  if (lane == 0) { info[1] = k; info[3] = (u32)bstar; }
}

__global__ void __launch_bounds__(256) k_rec_collect(const u64* __restrict__ n, const u32* __restrict__ id, u32 nslots,
                                                     RecItem* __restrict__ cand, u32* __restrict__ info) {
  const int bstar = (int)info[3];
  const u32 lane = threadIdx.x & 31u;
  const u32 stride = gridDim.x * blockDim.x;
  for (u32 s0 = blockIdx.x * blockDim.x + (threadIdx.x & ~31u); s0 < nslots; s0 += stride) {   // warp-uniform trip count
    const u32 s = s0 + lane;
    const u64 v = s < nslots ? n[s] : 0ull;
    const bool take = v >= 2 && rec_bin(v) >= bstar;
    const unsigned m = __ballot_sync(0xffffffffu, take);
    if (m == 0u) continue;
    u32 base = 0;
    if (lane == 0) base = atomicAdd(&info[2], (u32)__popc(m));   // warp-aggregated append
    base = __shfl_sync(0xffffffffu, base, 0);
    if (take) cand[base + __popc(m & ((1u << lane) - 1u))] = RecItem{~v, id[s], s};
  }
}

__global__ void k_rec_pad(RecItem* __restrict__ a, u32 from, u32 to) {
  const u32 i = from + blockIdx.x * blockDim.x + threadIdx.x;
  if (i < to) a[i] = RecItem{~0ull, 0xFFFFFFFFu, 0xFFFFFFFFu};
}

__device__ __forceinline__ bool rec_less(const RecItem& a, const RecItem& b) {
  return a.key < b.key || (a.key == b.key && a.id < b.id);
}

// ---- bitonic network on (key, id), ascending, for L = 2^m items ---------------------------------------------------
// compare-exchange partner i ^ j inside blocks of size kk: ascending where (i & kk) == 0
__device__ __forceinline__ void cmpx(RecItem& a, RecItem& b, bool asc) {
  if (rec_less(b, a) == asc) { const RecItem t = a; a = b; b = t; }
}

// all steps with j < SORT_TILE for kk = kk_first .. kk_last (doubling), one tile of SORT_TILE items per CTA
__global__ void __launch_bounds__(SORT_TILE / 2) k_bitonic_tile(RecItem* __restrict__ a, u32 L, u32 kk_first, u32 kk_last) {
  __shared__ RecItem sh[SORT_TILE];
  const u32 t0 = blockIdx.x * SORT_TILE;
  const u32 len = min((u32)SORT_TILE, L - t0);   // L is a power of two: len is SORT_TILE or L itself
  for (u32 i = threadIdx.x; i < len; i += blockDim.x) sh[i] = a[t0 + i];
  __syncthreads();
  for (u32 kk = kk_first; kk <= kk_last; kk <<= 1) {
    for (u32 j = min(kk >> 1, (u32)SORT_TILE >> 1); j > 0; j >>= 1) {
      for (u32 p = threadIdx.x; p < len / 2; p += blockDim.x) {
        const u32 i = ((p & ~(j - 1)) << 1) | (p & (j - 1));   // lower element of pair p
        cmpx(sh[i], sh[i | j], ((t0 + i) & kk) == 0);
      }
      __syncthreads();
    }
  }
  for (u32 i = threadIdx.x; i < len; i += blockDim.x) a[t0 + i] = sh[i];
}

// one step (kk, j) with j >= SORT_TILE in global memory
__global__ void __launch_bounds__(256) k_bitonic_global(RecItem* __restrict__ a, u32 L, u32 kk, u32 j) {
  const u32 p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= L / 2) return;
  const u32 i = ((p & ~(j - 1)) << 1) | (p & (j - 1));
  RecItem x = a[i], y = a[i | j];
  if (rec_less(y, x) == (((i & kk) == 0))) { a[i] = y; a[i | j] = x; }
}

template <typename R>
__global__ void __launch_bounds__(256) k_rec_apply(SdArraysT<R> a, int hx, int hy, int hz, const RecItem* __restrict__ dead,
                                                   const RecItem* __restrict__ cand, const u32* __restrict__ info) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= info[1]) return;
  const u32 d = dead[i].slot, s = cand[i].slot;
  const u64 v = a.n[s], half = v >> 1;
  a.rw2[d] = a.rw2[s]; a.rd3[d] = a.rd3[s]; a.kappa[d] = a.kappa[s];
  if (hx) a.x[d] = a.x[s];   // coordinates of absent dimensions are not stored
  if (hy) a.y[d] = a.y[s];
  if (hz) a.z[d] = a.z[s];
  a.n[d] = half;
  a.n[s] = v - half;
}

u32 pow2_at_least(u32 v) { u32 p = 1; while (p < v) p <<= 1; return p; }

// ascending order on (key, id) of a[0..count); a must have room for the next power of two.  Returns launches.
int sort_items(RecItem* a, u32 count, cudaStream_t st) {
  if (count < 2) return 0;
  int launches = 0;
  const u32 L = pow2_at_least(count);
  if (L > count) { k_rec_pad<<<(L - count + 255) / 256, 256, 0, st>>>(a, count, L); ++launches; }
  const u32 tiles = (L + SORT_TILE - 1) / SORT_TILE;
  k_bitonic_tile<<<tiles, SORT_TILE / 2, 0, st>>>(a, L, 2u, min(L, (u32)SORT_TILE));
  ++launches;
  for (u32 kk = 2u * SORT_TILE; kk <= L && kk != 0; kk <<= 1) {
    for (u32 j = kk >> 1; j >= SORT_TILE; j >>= 1) {
      k_bitonic_global<<<(L / 2 + 255) / 256, 256, 0, st>>>(a, L, kk, j);
      ++launches;
    }
    k_bitonic_tile<<<tiles, SORT_TILE / 2, 0, st>>>(a, L, kk, kk);
    ++launches;
  }
  return launches;
}

}  // namespace

size_t recycle_items_capacity(u64 cap_sd) { return (size_t)pow2_at_least((u32)std::max<u64>(cap_sd, 2)); }

void launch_recycle_scan(const u64* n, const u32* id, u32 nslots, RecItem* dead, u32* info, u32* hist, cudaStream_t st) {
  cudaMemsetAsync(info, 0, 8 * sizeof(u32), st);
  cudaMemsetAsync(hist, 0, REC_BINS * sizeof(u32), st);
  const int grid = (int)std::min<u64>(148 * 8, ((u64)nslots + 255) / 256);
  k_rec_scan<<<std::max(grid, 1), 256, 0, st>>>(n, id, nslots, dead, info, hist);
  k_rec_threshold<<<1, 32, 0, st>>>(info, hist);
}

template <typename R>
int launch_recycle_apply(const SdArraysT<R>& a, const Grid& g, u32 nslots, u32 n_dead, u32 k, RecItem* dead, RecItem* cand,
                         u32* info, u32* h_ncand, cudaStream_t st) {
  int launches = 1;
  const int grid = (int)std::min<u64>(148 * 8, ((u64)nslots + 255) / 256);
  k_rec_collect<<<std::max(grid, 1), 256, 0, st>>>(a.n, a.id, nslots, cand, info);
  // the number of candidates sizes the sorting network
  cudaMemcpyAsync(h_ncand, info + 2, sizeof(u32), cudaMemcpyDeviceToHost, st);
  cudaStreamSynchronize(st);
  launches += sort_items(cand, *h_ncand, st);
  launches += sort_items(dead, n_dead, st);
  k_rec_apply<R><<<(k + 255) / 256, 256, 0, st>>>(a, g.hx, g.hy, g.hz, dead, cand, info);
  return launches + 1;
}
#define INST(R) template int launch_recycle_apply<R>(const SdArraysT<R>&, const Grid&, u32, u32, u32, RecItem*, RecItem*, u32*, u32*, cudaStream_t);
SDM_INSTANTIATE_REAL(INST)
#undef INST

}  // namespace sdm
