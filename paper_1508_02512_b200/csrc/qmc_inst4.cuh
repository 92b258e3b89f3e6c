// One translation unit per dimension instantiates the version-4 (real path, constant-bank tables) kernel for L = 1, 2 loops and eps_order 0..2.
#pragma once
#include "qmc_kernels4.cuh"

// op: 0 = prepare (shared-memory opt-in + occupancy), 1 = launch; threads = 128 or QMC4_TBIG per block; tpl = dense-position template
template <int NDIM, int L, int KMAX, int T, int TPL>
static cudaError_t qmc4_op_t(int op, dim3 grid, size_t smem, cudaStream_t st, const Qmc4Launch *p, int *bps) {
  auto kern = qmc4_eval_kernel<NDIM, L, KMAX, T, TPL>;
  if (op == 0) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(bps, kern, T, smem);
  }
  kern<<<grid, T, smem, st>>>(*p);
  return cudaGetLastError();
}
template <int NDIM, int L, int KMAX>
static cudaError_t qmc4_op(int op, int threads, int tpl, dim3 grid, size_t smem, cudaStream_t st, const Qmc4Launch *p, int *bps) {
  if (threads == 128)
    return tpl ? qmc4_op_t<NDIM, L, KMAX, 128, 1>(op, grid, smem, st, p, bps) : qmc4_op_t<NDIM, L, KMAX, 128, 0>(op, grid, smem, st, p, bps);
  return tpl ? qmc4_op_t<NDIM, L, KMAX, QMC4_TBIG, 1>(op, grid, smem, st, p, bps) : qmc4_op_t<NDIM, L, KMAX, QMC4_TBIG, 0>(op, grid, smem, st, p, bps);
}

template <int NDIM>
static cudaError_t qmc4_dim_ops(int loops, int kmax, int op, int threads, int tpl, dim3 grid, size_t smem, cudaStream_t st, const Qmc4Launch *p,
                                int *bps) {
  constexpr int L2 = NDIM >= 2 ? 2 : 1;  // L <= NDIM
  switch (loops * 4 + kmax) {
    case 4: return qmc4_op<NDIM, 1, 0>(op, threads, tpl, grid, smem, st, p, bps);
    case 5: return qmc4_op<NDIM, 1, 1>(op, threads, tpl, grid, smem, st, p, bps);
    case 6: return qmc4_op<NDIM, 1, 2>(op, threads, tpl, grid, smem, st, p, bps);
    case 8: return NDIM >= 2 ? qmc4_op<NDIM, L2, 0>(op, threads, tpl, grid, smem, st, p, bps) : cudaErrorInvalidValue;
    case 9: return NDIM >= 2 ? qmc4_op<NDIM, L2, 1>(op, threads, tpl, grid, smem, st, p, bps) : cudaErrorInvalidValue;
    case 10: return NDIM >= 2 ? qmc4_op<NDIM, L2, 2>(op, threads, tpl, grid, smem, st, p, bps) : cudaErrorInvalidValue;
    default: return cudaErrorInvalidValue;
  }
}

#define QMC4_DEFINE_DIM(N)                                                                                        \
  cudaError_t qmc4_ops_d##N(int loops, int kmax, int op, int threads, int tpl, dim3 grid, size_t smem, cudaStream_t st, \
                            const Qmc4Launch *p, int *bps) {                                                      \
    return qmc4_dim_ops<N>(loops, kmax, op, threads, tpl, grid, smem, st, p, bps);                                        \
  }
