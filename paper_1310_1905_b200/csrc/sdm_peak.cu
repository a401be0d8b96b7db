// sdm_measure_fp64_peak (include/sdm.h): the fp64 FMA rate this device sustains, measured by a register-only DFMA
// kernel.  It is the denominator of the roofline of the condensation kernel, which is bound by the fp64 pipe
// (SURVEY.md section 8d asks for a MEASURED fp64-FMA peak; MEASURED_PEAKS.json has none).  Not part of the step.
#include "../../include/sdm.h"
#include "sdm_common.cuh"

namespace sdm {

// 8 independent dependent-DFMA chains per thread (a dependent DFMA issues every ~9 cycles on sm_100, the pipe takes a
// warp instruction every 2: four chains per scheduler saturate it, 8 warps x 8 chains are ample), `iters` rounds.
__global__ void __launch_bounds__(256) k_dfma_peak(double* out, long long* cycles, int iters, double a, double b) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  const long long t0 = clock64();
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  const long long t1 = clock64();
  out[blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

}  // namespace sdm

extern "C" int sdm_measure_fp64_peak(double* fma_tflops, double* dfma_per_clk_per_sm, void* stream) {
  using namespace sdm;
  if (!fma_tflops) return SDM_ERR_INVALID;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, n_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) {
    cudaGetLastError();
    return SDM_ERR_NO_DEVICE;
  }
  const int threads = 256, ctas_per_sm = 4, grid = n_sm * ctas_per_sm, iters = 1 << 14;
  double* out = nullptr;
  long long* cyc = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc = SDM_ERR_CUDA;
  double best_ms = 1e300, best_rate = 0.0;
  if (cudaMalloc((void**)&out, sizeof(double) * grid * threads) != cudaSuccess) goto done;
  if (cudaMalloc((void**)&cyc, sizeof(long long) * grid) != cudaSuccess) goto done;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) goto done;
  for (int rep = 0; rep < 6; ++rep) {   // the first repetition warms up clocks and instruction cache
    if (cudaEventRecord(e0, st) != cudaSuccess) goto done;
    k_dfma_peak<<<grid, threads, 0, st>>>(out, cyc, iters, 0.999999, 1e-6);
    if (cudaEventRecord(e1, st) != cudaSuccess || cudaEventSynchronize(e1) != cudaSuccess) goto done;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) goto done;
    if (rep == 0) continue;
    if (ms < best_ms) {
      best_ms = ms;
      long long h[4096];
      const int n = grid < 4096 ? grid : 4096;
      if (cudaMemcpy(h, cyc, sizeof(long long) * n, cudaMemcpyDeviceToHost) != cudaSuccess) goto done;
      long long mx = 1;
      for (int i = 0; i < n; ++i) mx = h[i] > mx ? h[i] : mx;
      // all CTAs are resident at once (4 x 256 threads per SM): an SM retires ctas_per_sm * threads * 8 * iters DFMAs in mx cycles
      best_rate = (double)ctas_per_sm * threads * 8.0 * iters / (double)mx;
    }
  }
  *fma_tflops = 2.0 * (double)grid * threads * 8.0 * iters / (best_ms * 1e-3) / 1e12;
  if (dfma_per_clk_per_sm) *dfma_per_clk_per_sm = best_rate;
  rc = SDM_OK;
done:
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(out);
  cudaFree(cyc);
  if (rc != SDM_OK) cudaGetLastError();
  return rc;
}
