// Shared device-side definitions of libsdm (sm_100a only).  Nothing here is used by oracle/.
// Citations are PAPER.md line numbers; [L] marks literature forms chosen in DESIGN.md "Readings".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef uint64_t u64;
typedef uint32_t u32;
typedef uint16_t u16;

namespace sdm {

// ---- constants (Table 2 :1052-1108; [L] where not printed) ----------------------------
namespace cst {
__device__ constexpr double rho_w = 1000.0, sigma_w = 0.072, c_pd = 1005.0, c_pv = 1850.0, c_l = 4218.0;
__device__ constexpr double l_v0 = 2.5e6, p_1000 = 1.0e5;
__device__ constexpr double R_d = 287.0, R_v = 461.5, T_0 = 273.16, p_vs0 = 611.73, g = 9.81;   // [L]
__device__ constexpr double D_0 = 2.21e-5, K_0 = 2.4e-2;                                         // [L]
__device__ constexpr double pi = 3.14159265358979323846;
__device__ constexpr double kc_delta0 = 9.06, kc_C0 = 0.292;   // Khvorostyanov & Curry 2002 [L]
}  // namespace cst

enum : u32 { TAG_SHUFFLE = 0, TAG_COAL = 1 };
constexpr u32 CELL_DEAD = 0xFFFFFFFFu;
constexpr int NSLOT = 1024;   // spread-address accumulators for counters and rain flux

// ---- launch-time descriptors ---------------------------------------------------------------------
struct Grid {
  int NX, NY, NZ;        // max(n?,1)
  int hx, hy, hz;        // dimension present
  int open_x;            // x is not periodic: this context is a slab of a larger domain (sdm_opts_init.open_x)
  int ncell;
  double dx, dy, dz, dt, dV;
  double X, Y, Z;
};
template <typename R>
struct SdArraysT {       // SoA particle state in HBM (PAPER.md :510-520, Table 1 :162-169); R = real_t of the
  u64* n;                // paper's templates (double or float): the STORAGE type of the real attributes.  The
  R *rw2, *rd3, *kappa;  // kernels load them into fp64, compute in fp64 and round on store; multiplicities are
  R *x, *y, *z;          // 64-bit integers either way.
  u32* id;               // persistent unique id (keys every Philox draw)
};
using SdArrays = SdArraysT<double>;
#define SDM_INSTANTIATE_REAL(MACRO) MACRO(double) MACRO(float)
struct Field {           // arrinfo_t mapped on (i,j,k) (PAPER.md :730-745)
  double* p;
  long long s0, s1, s2;
  __device__ __forceinline__ double& at(int i, int j, int k) const { return p[i * s0 + j * s1 + k * s2]; }
};
struct Counters {        // device accumulators, NSLOT spread slots each
  unsigned long long* pairs;
  unsigned long long* collisions;
  unsigned long long* near_ties;
  unsigned long long* ill_posed;
  unsigned long long* f_evals;
  unsigned long long* sd_substeps;
  unsigned long long* cond_slow;
};
constexpr int N_COUNTERS = 7;
struct CoalParams {
  int kernel, multi_coal;
  double golovin_b;
  int n_eff_R, n_eff_q;
  const double *eff_R, *eff_q, *eff_tab;   // DEVICE copies
  u32 seed_lo, seed_hi;
};

// ---- Philox-4x32-10 (Salmon et al. 2011; BASELINE.json north_star) --------------------------------
__device__ __forceinline__ void philox4x32_10(u32 c0, u32 c1, u32 c2, u32 c3, u32 k0, u32 k1, u32& o0, u32& o1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const u32 hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const u32 hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  o0 = c0; o1 = c1;
}
__device__ __forceinline__ u32 shuffle_key(u32 id, u32 step, u32 sub, u32 k0, u32 k1) {
  u32 a, b;
  philox4x32_10(id, step, sub, TAG_SHUFFLE, k0, k1, a, b);
  return a;
}
// u in (0,1) (PAPER.md :639)
__device__ __forceinline__ double coal_uniform(u32 id_first, u32 step, u32 sub, u32 k0, u32 k1) {
  u32 a, b;
  philox4x32_10(id_first, step, sub, TAG_COAL, k0, k1, a, b);
  const u64 w = ((u64)a << 32) | b;
  return ((double)(w >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

// ---- cell index (PAPER.md :547 eq. 15) -------------------------------------------------------------
__device__ __forceinline__ int cell_1d(double x, double dx, int n) {
  int i = (int)floor(x / dx);
  i = max(i, 0);
  return min(i, n - 1);
}
__device__ __forceinline__ u32 cell_of(const Grid& g, double x, double y, double z) {
  const int i = g.hx ? cell_1d(x, g.dx, g.NX) : 0;
  const int j = g.hy ? cell_1d(y, g.dy, g.NY) : 0;
  const int k = g.hz ? cell_1d(z, g.dz, g.NZ) : 0;
  return (u32)((i * g.NY + j) * g.NZ + k);
}

// ---- thermodynamics (PAPER.md :1042-1046 eq. 43-44, Table 2) ----------------------------------------
__device__ __forceinline__ double T_of(double th, double rhod) {
  return pow(th * pow(rhod * cst::R_d / cst::p_1000, cst::R_d / cst::c_pd), cst::c_pd / (cst::c_pd - cst::R_d));
}
__device__ __forceinline__ double eta_air(double T) {   // [L]
  const double q = T / 273.0;
  return 1.72e-5 * (393.0 / (T + 120.0)) * (q * sqrt(q));
}
// terminal velocity, Khvorostyanov & Curry 2002 smooth sphere (PAPER.md :649) [L]
__device__ __forceinline__ double v_term(double r, double eta, double rho_a) {
  const double c1 = 4.0 / (cst::kc_delta0 * cst::kc_delta0 * sqrt(cst::kc_C0));
  const double X = (32.0 / 3.0) * (r * r * r) * (cst::rho_w - rho_a) * cst::g * rho_a / (eta * eta);
  const double e = c1 * sqrt(X);
  const double s = e / (sqrt(1.0 + e) + 1.0);
  const double Re = (cst::kc_delta0 * cst::kc_delta0 / 4.0) * (s * s);
  return eta * Re / (2.0 * r * rho_a);
}

// ---- group primitives: G threads cooperate on one cell ---------------------------------------------
// G <= 32: a lane group inside a warp (shuffles, __syncwarp).  G > 32: the whole CTA (G == blockDim.x).
template <int G>
struct Group {
  static_assert(G == 4 || G == 8 || G == 16 || G == 32 || G == 64 || G == 128 || G == 256 || G == 512 || G == 1024, "G");
  static constexpr bool kWarp = (G <= 32);
  int lane;       // rank inside the group
  u32 mask;       // shuffle / syncwarp mask (kWarp)
  double* red;    // shared scratch of G/32 doubles (!kWarp)
  __device__ __forceinline__ void sync() const {
    if constexpr (kWarp) __syncwarp(mask); else __syncthreads();
  }
  // sum over the group; every thread gets the bit-identical result (xor butterfly)
  __device__ __forceinline__ double sum(double v) const {
    if constexpr (kWarp) {
#pragma unroll
      for (int d = G / 2; d >= 1; d >>= 1) v += __shfl_xor_sync(mask, v, d, 32);
      return v;
    } else {
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d, 32);
      __syncthreads();   // protect red from the previous use
      if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
      __syncthreads();
      double t = 0.0;
#pragma unroll
      for (int w = 0; w < G / 32; ++w) t += red[w];
      return t;
    }
  }
  // largest value over the group (v >= 0), the same on every thread
  __device__ __forceinline__ double max_nonneg(double v) const {
    if constexpr (kWarp) {
#pragma unroll
      for (int d = G / 2; d >= 1; d >>= 1) v = fmax(v, __shfl_xor_sync(mask, v, d, 32));
      return v;
    } else {
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, d, 32));
      __syncthreads();
      if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
      __syncthreads();
      double t = 0.0;
#pragma unroll
      for (int w = 0; w < G / 32; ++w) t = fmax(t, red[w]);
      return t;
    }
  }
  __device__ __forceinline__ unsigned long long sum(unsigned long long v) const {
    if constexpr (kWarp) {
#pragma unroll
      for (int d = G / 2; d >= 1; d >>= 1) v += __shfl_xor_sync(mask, v, d, 32);
      return v;
    } else {
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d, 32);
      __syncthreads();
      unsigned long long* r = reinterpret_cast<unsigned long long*>(red);
      if ((threadIdx.x & 31) == 0) r[threadIdx.x >> 5] = v;
      __syncthreads();
      unsigned long long t = 0;
#pragma unroll
      for (int w = 0; w < G / 32; ++w) t += r[w];
      return t;
    }
  }
};

template <int G>
__device__ __forceinline__ Group<G> make_group(double* red_scratch) {
  Group<G> g;
  if constexpr (G <= 32) {
    const int wl = threadIdx.x & 31;
    g.lane = wl & (G - 1);
    g.mask = (G == 32) ? 0xffffffffu : (((1u << G) - 1u) << (wl & ~(G - 1)));
    g.red = nullptr;
  } else {
    g.lane = threadIdx.x;
    g.mask = 0xffffffffu;
    g.red = red_scratch;
  }
  return g;
}

// Sort the m composite keys (shuffle key << 32 | id) held in shared memory `skey[0..P)` (P = power of
// two >= m, padded with ~0) by a bitonic network run by the group, carrying `sidx` along.
template <int G, typename IdxT>
__device__ __forceinline__ void bitonic_sort(const Group<G>& grp, u64* skey, IdxT* sidx, int P) {
  for (int k = 2; k <= P; k <<= 1) {
    for (int j = k >> 1; j > 0; j >>= 1) {
      grp.sync();
      for (int t = grp.lane; t < (P >> 1); t += G) {
        // t-th compare-exchange of this stage: i has bit j clear
        const int i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
        const int l = i | j;
        const bool up = ((i & k) == 0);
        const u64 a = skey[i], b = skey[l];
        if ((a > b) == up) {
          skey[i] = b; skey[l] = a;
          const IdxT ia = sidx[i]; sidx[i] = sidx[l]; sidx[l] = ia;
        }
      }
    }
  }
  grp.sync();
}

__host__ __device__ __forceinline__ int next_pow2(int v) {
  int p = 1;
  while (p < v) p <<= 1;
  return p;
}

}  // namespace sdm
