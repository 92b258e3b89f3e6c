// One translation unit per dimension instantiates the evaluation kernel for every (eps_order, real/complex).
#pragma once
#include "qmc_kernels.cuh"

template <int NDIM, int KMAX, bool CPLX, int NSCAP, bool TAYLOR = false>
static cudaError_t qmc_op(int op, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch *p, int *bps) {
  auto kern = qmc_eval_kernel<NDIM, KMAX, CPLX, NSCAP, TAYLOR>;
  if (op == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(bps, kern, QMC_THREADS, smem);
  }
  kern<<<grid, QMC_THREADS, smem, st>>>(*p);
  return cudaGetLastError();
}

template <int NDIM>
static cudaError_t qmc_dim_ops(int kmax, int flavor /* 0 real, 1 complex, 2 complex with <= 1 singular variable, 3 real with Taylor sectors */, int op, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch *p, int *bps) {
  if (flavor == 3) switch (kmax) {
    case 0: return qmc_op<NDIM, 0, false, 4, true>(op, grid, smem, st, p, bps);
    case 1: return qmc_op<NDIM, 1, false, 4, true>(op, grid, smem, st, p, bps);
    case 2: return qmc_op<NDIM, 2, false, 4, true>(op, grid, smem, st, p, bps);
    default: return cudaErrorInvalidValue;
  }
  switch (kmax * 3 + flavor) {
    case 0: return qmc_op<NDIM, 0, false, 4>(op, grid, smem, st, p, bps);
    case 1: return qmc_op<NDIM, 0, true, 4>(op, grid, smem, st, p, bps);
    case 2: return qmc_op<NDIM, 0, true, 1>(op, grid, smem, st, p, bps);
    case 3: return qmc_op<NDIM, 1, false, 4>(op, grid, smem, st, p, bps);
    case 4: return qmc_op<NDIM, 1, true, 4>(op, grid, smem, st, p, bps);
    case 5: return qmc_op<NDIM, 1, true, 1>(op, grid, smem, st, p, bps);
    case 6: return qmc_op<NDIM, 2, false, 4>(op, grid, smem, st, p, bps);
    case 7: return qmc_op<NDIM, 2, true, 4>(op, grid, smem, st, p, bps);
    case 8: return qmc_op<NDIM, 2, true, 1>(op, grid, smem, st, p, bps);
    default: return cudaErrorInvalidValue;
  }
}

#define QMC_DEFINE_DIM(N)                                                                                          \
  cudaError_t qmc_ops_d##N(int kmax, int cplx, int op, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch *p, \
                           int *bps) {                                                                             \
    return qmc_dim_ops<N>(kmax, cplx, op, grid, smem, st, p, bps);                                                 \
  }
