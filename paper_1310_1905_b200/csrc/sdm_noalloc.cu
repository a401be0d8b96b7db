// sdm_cell_offsets_noalloc (include/sdm.h): the segment offsets of the counting sort by cell (the
// exclusive prefix sum that turns the per-cell histogram of super-droplets into the start of every cell's segment in the
// sorted order, PAPER.md :641 "sorting by cell"), as an entry point that ALLOCATES NOTHING.  For callers that cannot call
// cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
//
// The step's own scan (sdm_sort.cu: k_scan_partial / k_scan_blocks / k_scan_apply) keeps the sums of its 4096-cell blocks in
// a buffer that sdm_create allocates.  The variant here keeps them in a file-scope __device__ array of NA_MAX_BLOCKS = 4096
// words (16 KB, held by every GPU that loads the library until the process exits), which bounds the grid it accepts to
// NA_MAX_BLOCKS * 4096 = 16 777 216 cells (SDM_NOALLOC_MAX_CELLS).  It differs from the step's kernels in what it leaves alone: the
// histogram is read-only here (the step's scan zeroes it for the next step) and no maximum is taken.
//
// The array's name is a device symbol: in host code it is a host-side stand-in, not a device address, so the host asks
// cudaGetSymbolAddress for the address ONCE PER DEVICE, with that device current (set-up; scratch_of_current_device), and
// the kernels are given that pointer.
//
// Every call on a device shares the one array, and the array keeps the last call's contents.  Nothing in it has to start
// at zero: a call of nb blocks writes words [0, nb) in its first kernel before its second and third read them, and reads
// no other word.  Calls that OVERLAP on the GPU (two streams, or two host threads on one device) race on it; calls on one
// stream, or otherwise ordered, do not.
#include <cstdio>
#include <mutex>
#include <string>

#include "../../include/sdm.h"
#include "sdm_common.cuh"

namespace sdm {

constexpr int NA_THREADS = 1024, NA_ITEMS = 4, NA_TILE = NA_THREADS * NA_ITEMS;   // the geometry of the step's scan
constexpr int NA_MAX_BLOCKS = 4096;
constexpr long long NA_MAX_CELLS = (long long)NA_MAX_BLOCKS * NA_TILE;
static_assert(NA_MAX_CELLS == SDM_NOALLOC_MAX_CELLS, "include/sdm.h states the limit");

static __device__ __align__(256) u32 g_noalloc_blocksum[NA_MAX_BLOCKS];   // the scratch: sums, then offsets, of the blocks

__device__ __forceinline__ u32 na_block_excl_scan(u32 v, u32* warp_sums, u32& total) {
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

// sum of every block of NA_TILE cells
__global__ void __launch_bounds__(NA_THREADS) k_na_partial(const u32* __restrict__ count, long long ncell, u32* __restrict__ blocksum) {
  __shared__ u32 ws[32];
  const long long base = (long long)blockIdx.x * NA_TILE + threadIdx.x * NA_ITEMS;
  u32 s = 0;
#pragma unroll
  for (int k = 0; k < NA_ITEMS; ++k)
    if (base + k < ncell) s += count[base + k];
  u32 total;
  na_block_excl_scan(s, ws, total);
  if (threadIdx.x == 0) blocksum[blockIdx.x] = total;
}

// one CTA: exclusive scan of the block sums in place; the grand total is seg[ncell]
__global__ void __launch_bounds__(NA_THREADS) k_na_blocks(u32* __restrict__ blocksum, int nblocks, u32* __restrict__ seg_total) {
  __shared__ u32 ws[32];
  u32 carry = 0;
  for (int b0 = 0; b0 < nblocks; b0 += NA_THREADS) {
    const int b = b0 + threadIdx.x;
    const u32 v = b < nblocks ? blocksum[b] : 0u;
    u32 total;
    const u32 ex = na_block_excl_scan(v, ws, total);
    if (b < nblocks) blocksum[b] = carry + ex;
    carry += total;
    __syncthreads();
  }
  if (threadIdx.x == 0) *seg_total = carry;
}

__global__ void __launch_bounds__(NA_THREADS) k_na_apply(const u32* __restrict__ count, long long ncell, const u32* __restrict__ blocksum,
                                                         u32* __restrict__ seg) {
  __shared__ u32 ws[32];
  const long long base = (long long)blockIdx.x * NA_TILE + threadIdx.x * NA_ITEMS;
  u32 v[NA_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < NA_ITEMS; ++k) { v[k] = base + k < ncell ? count[base + k] : 0u; s += v[k]; }
  u32 total;
  u32 ex = na_block_excl_scan(s, ws, total) + blocksum[blockIdx.x];
#pragma unroll
  for (int k = 0; k < NA_ITEMS; ++k)
    if (base + k < ncell) { seg[base + k] = ex; ex += v[k]; }
}

namespace {
thread_local std::string g_na_error;
constexpr int kMaxDevices = 64;
std::mutex g_na_mutex;
u32* g_na_scratch[kMaxDevices] = {};   // device address of g_noalloc_blocksum on each device, looked up once

int na_fail(int code, const std::string& msg) {
  g_na_error = msg;
  return code;
}

// the device address of the scratch on the CURRENT device (cudaGetSymbolAddress resolves the symbol in the current context)
int scratch_of_current_device(u32** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return na_fail(SDM_ERR_NO_DEVICE, std::string("sdm_cell_offsets_noalloc: no CUDA device (") + cudaGetErrorString(e) + ")");
  }
  if (dev < 0 || dev >= kMaxDevices) return na_fail(SDM_ERR_INVALID, "sdm_cell_offsets_noalloc: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (!g_na_scratch[dev]) {
    u32* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_blocksum);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return na_fail(e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? SDM_ERR_NO_DEVICE : SDM_ERR_CUDA,
                     std::string("sdm_cell_offsets_noalloc: cudaGetSymbolAddress of the scratch array failed (") + cudaGetErrorString(e) + ")");
    }
    g_na_scratch[dev] = p;
  }
  *out = g_na_scratch[dev];
  return SDM_OK;
}
}  // namespace
}  // namespace sdm

extern "C" const char* sdm_noalloc_last_error(void) { return sdm::g_na_error.c_str(); }

extern "C" int sdm_cell_offsets_noalloc_setup(void) {
  uint32_t* p = nullptr;
  return sdm::scratch_of_current_device(&p);
}

extern "C" int sdm_cell_offsets_noalloc(const uint32_t* count, int64_t ncell, uint32_t* seg, void* stream) {
  using namespace sdm;
  if (ncell < 0) return na_fail(SDM_ERR_INVALID, "sdm_cell_offsets_noalloc: ncell < 0");
  if (!seg || (ncell > 0 && !count)) return na_fail(SDM_ERR_INVALID, "sdm_cell_offsets_noalloc: NULL count or seg");
  if (ncell > NA_MAX_CELLS) {
    char msg[200];
    snprintf(msg, sizeof msg, "sdm_cell_offsets_noalloc: %lld cells exceed the static scratch of %d block sums (limit %lld cells)",
             (long long)ncell, NA_MAX_BLOCKS, NA_MAX_CELLS);
    return na_fail(SDM_ERR_CAPACITY, msg);
  }
  u32* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch);   // a table look-up after the first call on this device
  if (rc != SDM_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const int nb = (int)((ncell + NA_TILE - 1) / NA_TILE);
  if (nb) k_na_partial<<<nb, NA_THREADS, 0, st>>>(count, (long long)ncell, scratch);
  k_na_blocks<<<1, NA_THREADS, 0, st>>>(scratch, nb, seg + ncell);
  if (nb) k_na_apply<<<nb, NA_THREADS, 0, st>>>(count, (long long)ncell, scratch, seg);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return na_fail(SDM_ERR_CUDA, std::string("sdm_cell_offsets_noalloc: launch failed (") + cudaGetErrorString(e) + ")");
  return SDM_OK;
}
