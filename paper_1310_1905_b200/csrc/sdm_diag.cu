// Stage a7: per-cell spectral-moment diagnostics (PAPER.md :818-823, eq. 29)
// and the strided -> dense copy of the Eulerian input fields (arrinfo_t, :730-745).
#include "sdm_kernels.cuh"

namespace sdm {

// M^k[cell] += N r^k for r in [r_mi, r_mx); SDs are visited in storage order, which is cell-sorted
// up to the last move, so lanes of a warp that hit the same cell are first summed in lane order and
// issue one atomic per distinct cell.
template <typename R>
__global__ void __launch_bounds__(256) k_diag_mom(SdArraysT<R> a, const u32* __restrict__ d_nslots, Grid g, int wet,
                                                  double r_mi, double r_mx, int k, int count_only,
                                                  double* __restrict__ out) {
  const u32 i = blockIdx.x * blockDim.x + threadIdx.x;
  const u32 nslots = *d_nslots;
  u32 c = CELL_DEAD;
  double v = 0.0;
  if (i < nslots) {
    const u64 n = a.n[i];
    if (n != 0) {
      if (count_only) {
        v = 1.0;
        c = cell_of(g, g.hx ? a.x[i] : 0.0, g.hy ? a.y[i] : 0.0, g.hz ? a.z[i] : 0.0);
      } else {
        const double r = wet ? sqrt((double)a.rw2[i]) : cbrt((double)a.rd3[i]);
        if (r >= r_mi && r < r_mx) {
          v = (double)n * pow(r, (double)k);
          c = cell_of(g, g.hx ? a.x[i] : 0.0, g.hy ? a.y[i] : 0.0, g.hz ? a.z[i] : 0.0);
        }
      }
    }
  }
  const u32 peers = __match_any_sync(0xffffffffu, c);
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(peers) - 1;
  double s = 0.0;
  for (u32 mset = peers; mset; mset &= mset - 1) {   // same trip count for all peers of a cell
    const int src = __ffs(mset) - 1;
    s += __shfl_sync(peers, v, src);
  }
  if (c != CELL_DEAD && lane == leader) atomicAdd(&out[c], s);
}

__global__ void k_diag_norm(double* __restrict__ out, const double* __restrict__ rhod, int ncell, double dV) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c < ncell) out[c] = out[c] / (rhod[c] * dV);
}

__global__ void k_dense_copy(Field src, double* __restrict__ dst, int n0, int n1, int n2) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long tot = (long long)n0 * n1 * n2;
  if (t >= tot) return;
  const int k = (int)(t % n2), j = (int)((t / n2) % n1), i = (int)(t / ((long long)n2 * n1));
  dst[t] = src.at(i, j, k);
}

template <typename R>
void launch_diag_mom(const SdArraysT<R>& a, const u32* d_nslots, u32 nslots_bound, const Grid& g, int wet, double r_mi,
                     double r_mx, int k, int count_only, const double* rhod, double* out, cudaStream_t st) {
  cudaMemsetAsync(out, 0, sizeof(double) * g.ncell, st);
  if (nslots_bound)
    k_diag_mom<R><<<(nslots_bound + 255) / 256, 256, 0, st>>>(a, d_nslots, g, wet, r_mi, r_mx, k, count_only, out);
  if (!count_only) k_diag_norm<<<(g.ncell + 255) / 256, 256, 0, st>>>(out, rhod, g.ncell, g.dV);
}

#define SDM_INST(R)                                                                                             \
  template void launch_diag_mom<R>(const SdArraysT<R>&, const u32*, u32, const Grid&, int, double, double, int, int, \
                                   const double*, double*, cudaStream_t);
SDM_INSTANTIATE_REAL(SDM_INST)
#undef SDM_INST

void launch_dense_copy(Field src, double* dst, int n0, int n1, int n2, cudaStream_t st) {
  const long long tot = (long long)n0 * n1 * n2;
  k_dense_copy<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(src, dst, n0, n1, n2);
}

}  // namespace sdm
