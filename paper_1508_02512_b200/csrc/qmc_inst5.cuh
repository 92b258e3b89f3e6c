// One translation unit per dimension instantiates the version-5 (complex path, constant-bank tables) kernel for L = 1, 2 loops and eps_order 0..2.
#pragma once
#include "qmc_kernels5.cuh"

template <int NDIM, int L, int KMAX>
static cudaError_t qmc5_op(int op, dim3 grid, size_t smem, cudaStream_t st, const Qmc5Launch *p, int *bps) {
  auto kern = qmc5_eval_kernel<NDIM, L, KMAX>;
  if (op == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(bps, kern, QMC3_THREADS, smem);
  }
  kern<<<grid, QMC3_THREADS, smem, st>>>(*p);
  return cudaGetLastError();
}

template <int NDIM>
static cudaError_t qmc5_dim_ops(int loops, int kmax, int op, dim3 grid, size_t smem, cudaStream_t st, const Qmc5Launch *p,
                                int *bps) {
  constexpr int L2 = NDIM >= 2 ? 2 : 1;  // L <= NDIM
  switch (loops * 4 + kmax) {
    case 4: return qmc5_op<NDIM, 1, 0>(op, grid, smem, st, p, bps);
    case 5: return qmc5_op<NDIM, 1, 1>(op, grid, smem, st, p, bps);
    case 6: return qmc5_op<NDIM, 1, 2>(op, grid, smem, st, p, bps);
    case 8: return NDIM >= 2 ? qmc5_op<NDIM, L2, 0>(op, grid, smem, st, p, bps) : cudaErrorInvalidValue;
    case 9: return NDIM >= 2 ? qmc5_op<NDIM, L2, 1>(op, grid, smem, st, p, bps) : cudaErrorInvalidValue;
    case 10: return NDIM >= 2 ? qmc5_op<NDIM, L2, 2>(op, grid, smem, st, p, bps) : cudaErrorInvalidValue;
    default: return cudaErrorInvalidValue;
  }
}

#define QMC5_DEFINE_DIM(N)                                                                                        \
  cudaError_t qmc5_ops_d##N(int loops, int kmax, int op, dim3 grid, size_t smem, cudaStream_t st, const Qmc5Launch *p, \
                            int *bps) {                                                                           \
    return qmc5_dim_ops<N>(loops, kmax, op, grid, smem, st, p, bps);                                              \
  }
