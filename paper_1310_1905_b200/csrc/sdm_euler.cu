// The "prototype transport equation solver" of PAPER.md Figure 7 (:831-852), for the calling sequence of section 5.2.2:
// one first-order upstream (donor-cell) step of a scalar field on the Arakawa-C grid (the scheme of PAPER.md :219-235 and
// the first pass of MPDATA, :347, :1116), driven by the rho_d x Courant arrays the context already holds (:751).  It is what
// the host model does between step_sync and the next step_sync while step_async runs (:816); libsdm's own step never
// calls it.  Compiled with -fmad=false: the same IEEE operations in the same order as the oracle's restatement.
#include "../../include/sdm.h"
#include "sdm_kernels.cuh"

namespace sdm {

// psi_c' = psi_c - [sum over dimensions of (F_hi - F_lo)] / rho_d,  F = max(rho_d C, 0) psi_upwind-side + min(rho_d C, 0) psi_other
// at each face; periodic in x and y, the field continued by its boundary value through bottom and top.
__global__ void __launch_bounds__(256) k_upstream(Field psi, Grid g, CellFields cf, double* __restrict__ out) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.ncell) return;
  const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
  const double pc = psi.at(i, j, k);
  double acc = 0.0;
  if (g.hx) {
    const double pm = psi.at(i == 0 ? g.NX - 1 : i - 1, j, k), pp = psi.at(i == g.NX - 1 ? 0 : i + 1, j, k);
    const double Cl = cf.cx[((long long)i * g.NY + j) * g.NZ + k], Ch = cf.cx[((long long)(i + 1) * g.NY + j) * g.NZ + k];
    const double Fl = fmax(Cl, 0.0) * pm + fmin(Cl, 0.0) * pc, Fh = fmax(Ch, 0.0) * pc + fmin(Ch, 0.0) * pp;
    acc = acc + (Fh - Fl);
  }
  if (g.hy) {
    const double pm = psi.at(i, j == 0 ? g.NY - 1 : j - 1, k), pp = psi.at(i, j == g.NY - 1 ? 0 : j + 1, k);
    const double Cl = cf.cy[((long long)i * (g.NY + 1) + j) * g.NZ + k], Ch = cf.cy[((long long)i * (g.NY + 1) + j + 1) * g.NZ + k];
    const double Fl = fmax(Cl, 0.0) * pm + fmin(Cl, 0.0) * pc, Fh = fmax(Ch, 0.0) * pc + fmin(Ch, 0.0) * pp;
    acc = acc + (Fh - Fl);
  }
  if (g.hz) {
    const double pm = psi.at(i, j, k == 0 ? 0 : k - 1), pp = psi.at(i, j, k == g.NZ - 1 ? k : k + 1);
    const double Cl = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k], Ch = cf.cz[((long long)i * g.NY + j) * (g.NZ + 1) + k + 1];
    const double Fl = fmax(Cl, 0.0) * pm + fmin(Cl, 0.0) * pc, Fh = fmax(Ch, 0.0) * pc + fmin(Ch, 0.0) * pp;
    acc = acc + (Fh - Fl);
  }
  out[c] = pc - acc / cf.rhod[c];
}

__global__ void __launch_bounds__(256) k_store_field(const double* __restrict__ src, Field dst, Grid g) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= g.ncell) return;
  const int k = c % g.NZ, j = (c / g.NZ) % g.NY, i = c / (g.NZ * g.NY);
  dst.at(i, j, k) = src[c];
}

void launch_upstream(Field psi, const Grid& g, const CellFields& cf, double* tmp, cudaStream_t st) {
  const int grid = (g.ncell + 255) / 256;
  k_upstream<<<grid, 256, 0, st>>>(psi, g, cf, tmp);
  k_store_field<<<grid, 256, 0, st>>>(tmp, psi, g);
}

}  // namespace sdm
