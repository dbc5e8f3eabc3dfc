// pupil_prior.cu - slide-level pupil prior (reading B9 of DESIGN.md).
//
// PAPER.md:171 / Fig. 4(b) show the recovered pupil varying smoothly from region to region of a slide; the paper
// states no algorithm that uses it.  B9: the Zernike coefficients recovered per tile are fitted, coefficient by
// coefficient, by a polynomial of total degree <= order in the tile's slide coordinates (terms 1, X, Y, X^2, XY, Y^2)
// by unweighted least squares over the tiles with status 0; the fit evaluated at a tile is that tile's prior
// (apic_reconstruct_prior starts the aberration fit from it).  If the successful tiles do not determine the
// polynomial the fit falls back to their mean, and to zero if there are none.
//
// One CTA: the normal matrix (<= 6 x 6) and the right-hand sides (<= 6 per coefficient) are accumulated in fp64 over
// the tiles by 4 tile groups x 64 coefficient lanes, reduced in group order, solved per coefficient by a Cholesky
// factorisation in registers, and the polynomial is evaluated for every tile.  A slide is 10^4 tiles x <= 64
// coefficients: microseconds, off the hot path.
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/apic.h"

namespace apic {
namespace {

constexpr int kLanes = 64, kGroups = 4, kTerms = 6, kPairs = 21;

__device__ __forceinline__ void terms_of(float x, float y, double (&b)[kTerms]) {
  b[0] = 1.0; b[1] = x; b[2] = y; b[3] = double(x) * x; b[4] = double(x) * y; b[5] = double(y) * y;
}

__global__ void __launch_bounds__(kLanes * kGroups) pupil_field_fit_kernel(const float* __restrict__ coef,
                                                                           const int32_t* __restrict__ status,
                                                                           const float* __restrict__ xy, int tiles, int nz,
                                                                           int nt, float* __restrict__ fit,
                                                                           float* __restrict__ poly) {
  __shared__ double s_rhs[kGroups][kLanes][kTerms];
  __shared__ double s_nrm[kGroups][kPairs];
  __shared__ double s_poly[kTerms][kLanes];
  const int j = threadIdx.x % kLanes, g = threadIdx.x / kLanes;
  double rhs[kTerms], nrm[kPairs];
#pragma unroll
  for (int i = 0; i < kTerms; ++i) rhs[i] = 0.0;
#pragma unroll
  for (int i = 0; i < kPairs; ++i) nrm[i] = 0.0;
  for (int t = g; t < tiles; t += kGroups) {
    if (status[t] != 0) continue;
    double b[kTerms];
    terms_of(xy[2 * t], xy[2 * t + 1], b);
    const double c = j < nz ? double(coef[size_t(t) * nz + j]) : 0.0;
    int p = 0;
#pragma unroll
    for (int a = 0; a < kTerms; ++a) {
      rhs[a] += b[a] * c;
#pragma unroll
      for (int q = a; q < kTerms; ++q) nrm[p++] += b[a] * b[q];
    }
  }
#pragma unroll
  for (int i = 0; i < kTerms; ++i) s_rhs[g][j][i] = rhs[i];
  if (j == 0) {
#pragma unroll
    for (int i = 0; i < kPairs; ++i) s_nrm[g][i] = nrm[i];
  }
  __syncthreads();
  if (g == 0) {
    // totals in group order, then the nt x nt system of this coefficient
    double n[kTerms][kTerms], r[kTerms];
    int p = 0;
    for (int a = 0; a < kTerms; ++a)
      for (int q = a; q < kTerms; ++q, ++p) {
        double s = 0.0;
        for (int k = 0; k < kGroups; ++k) s += s_nrm[k][p];
        n[a][q] = s;
        n[q][a] = s;
      }
    for (int a = 0; a < kTerms; ++a) {
      double s = 0.0;
      for (int k = 0; k < kGroups; ++k) s += s_rhs[k][j][a];
      r[a] = s;
    }
    const double n_ok = n[0][0];
    double sol[kTerms] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    bool ok = n_ok > 0.0;
    if (ok) {
      // Cholesky n = L L^T on the leading nt x nt block; a pivot that is not clearly positive = rank deficient
      double L[kTerms][kTerms];
      for (int a = 0; a < nt && ok; ++a) {
        for (int q = 0; q <= a; ++q) {
          double s = n[a][q];
          for (int k = 0; k < q; ++k) s -= L[a][k] * L[q][k];
          if (q == a) {
            if (!(s > 1e-10 * n[a][a]) || !(n[a][a] > 0.0)) { ok = false; break; }
            L[a][a] = sqrt(s);
          } else {
            L[a][q] = s / L[q][q];
          }
        }
      }
      if (ok) {
        double y[kTerms];
        for (int a = 0; a < nt; ++a) {
          double s = r[a];
          for (int k = 0; k < a; ++k) s -= L[a][k] * y[k];
          y[a] = s / L[a][a];
        }
        for (int a = nt - 1; a >= 0; --a) {
          double s = y[a];
          for (int k = a + 1; k < nt; ++k) s -= L[k][a] * sol[k];
          sol[a] = s / L[a][a];
        }
      } else {
        sol[0] = r[0] / n_ok;                            // fallback: the mean over the successful tiles
      }
    }
    for (int a = 0; a < kTerms; ++a) {
      s_poly[a][j] = sol[a];
      if (j < nz) poly[a * nz + j] = float(sol[a]);
    }
  }
  __syncthreads();
  if (j < nz) {
    for (int t = g; t < tiles; t += kGroups) {
      double b[kTerms];
      terms_of(xy[2 * t], xy[2 * t + 1], b);
      double s = 0.0;
#pragma unroll
      for (int a = 0; a < kTerms; ++a) s += b[a] * s_poly[a][j];
      fit[size_t(t) * nz + j] = float(s);
    }
  }
}

}  // namespace
}  // namespace apic

extern "C" int apic_pupil_field_fit(const float* d_zernike, const int32_t* d_status, const float* d_xy, int tiles,
                                    int n_zernike, int order, float* d_fit, float* d_poly, void* cuda_stream) {
  using namespace apic;
  if (!d_zernike || !d_status || !d_xy || !d_fit || !d_poly) return APIC_EINVAL;
  if (tiles < 1 || n_zernike < 1 || n_zernike > kLanes || order < 0 || order > 2) return APIC_EINVAL;
  const int nt = order == 0 ? 1 : order == 1 ? 3 : 6;
  cudaGetLastError();
  pupil_field_fit_kernel<<<1, kLanes * kGroups, 0, static_cast<cudaStream_t>(cuda_stream)>>>(d_zernike, d_status, d_xy, tiles,
                                                                                           n_zernike, nt, d_fit, d_poly);
  return cudaGetLastError() == cudaSuccess ? APIC_OK : APIC_ECUDA;
}
