// Domain decomposition along x (PAPER.md :843 "a group of solver threads ... in case of domain
// decomposition"): every stage of the step but movement is local to a cell, so a rank owns a slab of columns and, after
// step_async, hands the SDs whose new x lies outside its slab to its two neighbours.  This file holds the two kernels of
// that exchange, count + pack (leavers out of the SoA state into contiguous buffers, their slots marked N = 0 for the next
// compaction) and unpack (arrivals appended behind the live slots, x shifted into the receiver's coordinates).  The
// transport itself (NCCL / gloo send-recv) is the caller's: paper_1310_1905_b200/slab.py.
#include "sdm_kernels.cuh"

namespace sdm {

// side of the slab an SD left through: 0 = left (x < 0), 1 = right (x >= X), -1 = still inside (or dead)
template <typename R>
__device__ __forceinline__ int leaver_side(const SdArraysT<R>& a, u32 i, double X) {
  if (a.n[i] == 0) return -1;
  const double x = (double)a.x[i];
  return x < 0.0 ? 0 : (x >= X ? 1 : -1);
}

template <typename R>
__global__ void __launch_bounds__(256) k_count_leavers(SdArraysT<R> a, u32 nslots, double X, u32* __restrict__ cnt2) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  const int side = i < nslots ? leaver_side(a, i, X) : -1;
  const unsigned l = __ballot_sync(0xffffffffu, side == 0), r = __ballot_sync(0xffffffffu, side == 1);
  if ((threadIdx.x & 31) == 0) {
    if (l) atomicAdd(&cnt2[0], (u32)__popc(l));
    if (r) atomicAdd(&cnt2[1], (u32)__popc(r));
  }
}

template <typename R>
__global__ void __launch_bounds__(256) k_pack_leavers(SdArraysT<R> a, u32 nslots, Grid g, SdArraysT<R> left, SdArraysT<R> right,
                                                      u32* __restrict__ cnt2) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  const int side = i < nslots ? leaver_side(a, i, g.X) : -1;
  const int lane = threadIdx.x & 31;
  for (int sd = 0; sd < 2; ++sd) {   // warp-aggregated append to the list of this side
    const unsigned m = __ballot_sync(0xffffffffu, side == sd);
    if (!m) continue;
    u32 base = 0;
    if (lane == __ffs(m) - 1) base = atomicAdd(&cnt2[sd], (u32)__popc(m));
    base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
    if (side == sd) {
      const SdArraysT<R>& o = sd ? right : left;
      const u32 d = base + __popc(m & ((1u << lane) - 1u));
      o.n[d] = a.n[i]; o.rw2[d] = a.rw2[i]; o.rd3[d] = a.rd3[i]; o.kappa[d] = a.kappa[i];
      o.x[d] = a.x[i];
      if (g.hy) o.y[d] = a.y[i];
      if (g.hz) o.z[d] = a.z[i];
      o.id[d] = a.id[i];
      a.n[i] = 0;   // gone from this slab: the next step_sync compacts the slot away
    }
  }
}

template <typename R>
__global__ void __launch_bounds__(256) k_unpack_arrivals(SdArraysT<R> a, u32 first, u32 count, Grid g, SdArraysT<R> in, double x_shift) {
  const u32 t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  const u32 d = first + t;
  a.n[d] = in.n[t]; a.rw2[d] = in.rw2[t]; a.rd3[d] = in.rd3[t]; a.kappa[d] = in.kappa[t];
  a.x[d] = (R)((double)in.x[t] + x_shift);
  if (g.hy) a.y[d] = in.y[t];
  if (g.hz) a.z[d] = in.z[t];
  a.id[d] = in.id[t];
}

template <typename R>
void launch_count_leavers(const SdArraysT<R>& a, u32 nslots, const Grid& g, u32* cnt2, cudaStream_t st) {
  cudaMemsetAsync(cnt2, 0, 2 * sizeof(u32), st);
  if (nslots) k_count_leavers<R><<<(nslots + 255) / 256, 256, 0, st>>>(a, nslots, g.X, cnt2);
}
template <typename R>
void launch_pack_leavers(const SdArraysT<R>& a, u32 nslots, const Grid& g, const SdArraysT<R>& left, const SdArraysT<R>& right, u32* cnt2,
                         cudaStream_t st) {
  cudaMemsetAsync(cnt2, 0, 2 * sizeof(u32), st);
  if (nslots) k_pack_leavers<R><<<(nslots + 255) / 256, 256, 0, st>>>(a, nslots, g, left, right, cnt2);
}
template <typename R>
void launch_unpack_arrivals(const SdArraysT<R>& a, u32 first, u32 count, const Grid& g, const SdArraysT<R>& in, double x_shift,
                            cudaStream_t st) {
  if (count) k_unpack_arrivals<R><<<(count + 255) / 256, 256, 0, st>>>(a, first, count, g, in, x_shift);
}

#define SDM_INST(R)                                                                                                          \
  template void launch_count_leavers<R>(const SdArraysT<R>&, u32, const Grid&, u32*, cudaStream_t);                          \
  template void launch_pack_leavers<R>(const SdArraysT<R>&, u32, const Grid&, const SdArraysT<R>&, const SdArraysT<R>&, u32*, cudaStream_t); \
  template void launch_unpack_arrivals<R>(const SdArraysT<R>&, u32, u32, const Grid&, const SdArraysT<R>&, double, cudaStream_t);
SDM_INSTANTIATE_REAL(SDM_INST)
#undef SDM_INST

}  // namespace sdm
