// Pieces of the evaluation shared by the real-path kernel (qmc_kernels4.cuh) and, for the exponents, the complex-path
// kernel (qmc_kernels5.cuh): compile-time integer powers, the exponents of U^ and F^, and the product form of the
// eps-expanded subtracted integrand folded one singular variable at a time (Eqs. 10-12).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "qmc_kernels.cuh"  // complex helpers, block_sum
#include "qmc_launch.h"
#include "qmc_tables.h"

namespace qmc2 {

template <int E>
__device__ __forceinline__ double ipow_c(double x) {  // x^E, E >= 0 compile time
  if (E == 0) return 1.0;
  if (E == 1) return x;
  double h = ipow_c<E / 2>(x);
  h *= h;
  return (E & 1) ? h * x : h;
}

// exponents of U^{aU0 + aU1 eps} F^{aF0 + aF1 eps} for P = NDIM + 1 propagators of power 1, L loops (Eq. 6)
template <int NDIM, int L>
struct Expo {
  static constexpr int aU0 = NDIM - 1 - 2 * L, aU1 = L + 1, aF0 = -(NDIM + 1 - 2 * L), aF1 = -L;
};

// per-sector state shared by the fold
template <int NS, int K>
struct Ctx2 {
  double bt[NS > 0 ? NS : 1];                     // t_k / beta_k
  double cL[NS > 0 ? NS : 1][K > 1 ? K - 1 : 1];  // (beta_k ln t_k)^p / p!, p = 0 .. K-2
  double W[1 << NS], Lam[1 << NS];                // index X = set of singular variables NOT set to zero
};

// The subtracted, eps-expanded integrand in product form is
//   sum_Z g_Z prod_{j notin Z} A_j prod_{j in Z} (B_j - A_j),   A_j = t_j^-1 e^{eps beta_j ln t_j},  B_j = 1/(beta_j eps).
// With prod_j t_j^-1 taken out (it sits in the sector's G0', qmc_image4.cpp) the factors are
//   a_j = e^{eps beta_j ln t_j}   and   b_j - a_j,  b_j = (t_j / beta_j) / eps:
// no multiplication by 1/t_j inside the fold.
// Fold2<LEVEL, ZMASK>: series of sum over Z' subset of {LEVEL..NS-1} of g_{ZMASK u Z'} prod_{j >= LEVEL, j notin Z'} a_j prod_{j in Z'} (b_j - a_j)
// window: orders -(NS-LEVEL) .. KMAX + popcount(ZMASK)  (what the remaining factors of levels < LEVEL can still use).
template <int NS, int KMAX, int K, int LEVEL, int ZMASK>
struct Fold2 {
  static constexpr int LEN = NS - LEVEL + KMAX + __builtin_popcount(ZMASK) + 1;
  static __device__ __forceinline__ void eval(const Ctx2<NS, K> &c, double (&out)[LEN]) {
    double a[LEN - 1], b[LEN];
    Fold2<NS, KMAX, K, LEVEL + 1, ZMASK>::eval(c, a);
    Fold2<NS, KMAX, K, LEVEL + 1, ZMASK | (1 << LEVEL)>::eval(c, b);
    const double bt = c.bt[LEVEL];
    double d[LEN - 1];
#pragma unroll
    for (int i = 0; i < LEN - 1; ++i) d[i] = a[i] - b[i];
    out[0] = bt * b[0];
#pragma unroll
    for (int i = 1; i < LEN; ++i) {
      double s = fma(bt, b[i], d[i - 1]);
#pragma unroll
      for (int p = 1; p < i; ++p) s = fma(c.cL[LEVEL][p], d[i - 1 - p], s);
      out[i] = s;
    }
  }
};
template <int NS, int KMAX, int K, int ZMASK>
struct Fold2<NS, KMAX, K, NS, ZMASK> {
  static constexpr int LEN = KMAX + __builtin_popcount(ZMASK) + 1;
  static __device__ __forceinline__ void eval(const Ctx2<NS, K> &c, double (&out)[LEN]) {
    constexpr int X = ((1 << NS) - 1) ^ ZMASK;
    out[0] = c.W[X];
#pragma unroll
    for (int p = 1; p < LEN; ++p) out[p] = out[p - 1] * (c.Lam[X] * (1.0 / p));
  }
};

__device__ __forceinline__ bool finite_hi(double v) { return (__double2hiint(v) & 0x7ff00000) != 0x7ff00000; }

}  // namespace qmc2
