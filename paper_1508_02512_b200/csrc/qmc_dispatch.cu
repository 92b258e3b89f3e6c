// Dimension dispatch of the evaluation kernel (instantiations live in qmc_inst_d<N>.cu).
#include "qmc_launch.h"

#define QMC_DECL(N) \
  cudaError_t qmc_ops_d##N(int, bool, int, dim3, size_t, cudaStream_t, const QmcLaunch *, int *);
QMC_DECL(1) QMC_DECL(2) QMC_DECL(3) QMC_DECL(4) QMC_DECL(5) QMC_DECL(6)

static cudaError_t ops(int ndim, int kmax, bool cplx, int op, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch *p, int *bps) {
  switch (ndim) {
    case 1: return qmc_ops_d1(kmax, cplx, op, grid, smem, st, p, bps);
    case 2: return qmc_ops_d2(kmax, cplx, op, grid, smem, st, p, bps);
    case 3: return qmc_ops_d3(kmax, cplx, op, grid, smem, st, p, bps);
    case 4: return qmc_ops_d4(kmax, cplx, op, grid, smem, st, p, bps);
    case 5: return qmc_ops_d5(kmax, cplx, op, grid, smem, st, p, bps);
    case 6: return qmc_ops_d6(kmax, cplx, op, grid, smem, st, p, bps);
    default: return cudaErrorInvalidValue;
  }
}

cudaError_t qmc_kernel_prepare(int ndim, int kmax, bool cplx, size_t smem, int *blocks_per_sm) {
  return ops(ndim, kmax, cplx, 0, dim3(1), smem, nullptr, nullptr, blocks_per_sm);
}
cudaError_t qmc_kernel_launch(int ndim, int kmax, bool cplx, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch &p) {
  return ops(ndim, kmax, cplx, 1, grid, smem, st, &p, nullptr);
}
