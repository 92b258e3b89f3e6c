// Dimension dispatch of the evaluation kernel (instantiations live in qmc_inst_d<N>.cu).
#include "qmc_launch.h"

#define QMC_DECL(N) \
  cudaError_t qmc_ops_d##N(int, int, int, dim3, size_t, cudaStream_t, const QmcLaunch *, int *);
QMC_DECL(1) QMC_DECL(2) QMC_DECL(3) QMC_DECL(4) QMC_DECL(5) QMC_DECL(6)

static cudaError_t ops(int ndim, int kmax, int cplx, int op, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch *p, int *bps) {
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

cudaError_t qmc_kernel_prepare(int ndim, int kmax, int flavor, size_t smem, int *blocks_per_sm) {
  return ops(ndim, kmax, flavor, 0, dim3(1), smem, nullptr, nullptr, blocks_per_sm);
}
cudaError_t qmc_kernel_launch(int ndim, int kmax, int flavor, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch &p) {
  return ops(ndim, kmax, flavor, 1, grid, smem, st, &p, nullptr);
}

// ---- version 4 (real path, constant-bank tables) -------------------------------------------------------------
#define QMC4_DECL(N) \
  cudaError_t qmc4_ops_d##N(int, int, int, int, int, dim3, size_t, cudaStream_t, const Qmc4Launch *, int *);
QMC4_DECL(1) QMC4_DECL(2) QMC4_DECL(3) QMC4_DECL(4) QMC4_DECL(5) QMC4_DECL(6)

static cudaError_t ops4(int ndim, int loops, int kmax, int op, int threads, int tpl, dim3 grid, size_t smem, cudaStream_t st,
                        const Qmc4Launch *p, int *bps) {
  switch (ndim) {
    case 1: return qmc4_ops_d1(loops, kmax, op, threads, tpl, grid, smem, st, p, bps);
    case 2: return qmc4_ops_d2(loops, kmax, op, threads, tpl, grid, smem, st, p, bps);
    case 3: return qmc4_ops_d3(loops, kmax, op, threads, tpl, grid, smem, st, p, bps);
    case 4: return qmc4_ops_d4(loops, kmax, op, threads, tpl, grid, smem, st, p, bps);
    case 5: return qmc4_ops_d5(loops, kmax, op, threads, tpl, grid, smem, st, p, bps);
    case 6: return qmc4_ops_d6(loops, kmax, op, threads, tpl, grid, smem, st, p, bps);
    default: return cudaErrorInvalidValue;
  }
}
bool qmc4_kernel_available(int ndim, int loops, int kmax) {
  return ndim >= 1 && ndim <= 6 && loops >= 1 && loops <= 2 && loops <= ndim && kmax >= 0 && kmax <= 2;
}
cudaError_t qmc4_kernel_prepare(int ndim, int loops, int kmax, int threads, int tpl, size_t smem, int *blocks_per_sm) {
  return ops4(ndim, loops, kmax, 0, threads, tpl, dim3(1), smem, nullptr, nullptr, blocks_per_sm);
}
cudaError_t qmc4_kernel_launch(int ndim, int loops, int kmax, int threads, int tpl, dim3 grid, size_t smem, cudaStream_t st,
                               const Qmc4Launch &p) {
  return ops4(ndim, loops, kmax, 1, threads, tpl, grid, smem, st, &p, nullptr);
}

// ---- version 5 (complex path, constant-bank tables) ----------------------------------------------------------
#define QMC5_DECL(N) \
  cudaError_t qmc5_ops_d##N(int, int, int, dim3, size_t, cudaStream_t, const Qmc5Launch *, int *);
QMC5_DECL(1) QMC5_DECL(2) QMC5_DECL(3) QMC5_DECL(4) QMC5_DECL(5) QMC5_DECL(6)

static cudaError_t ops5(int ndim, int loops, int kmax, int op, dim3 grid, size_t smem, cudaStream_t st, const Qmc5Launch *p, int *bps) {
  switch (ndim) {
    case 1: return qmc5_ops_d1(loops, kmax, op, grid, smem, st, p, bps);
    case 2: return qmc5_ops_d2(loops, kmax, op, grid, smem, st, p, bps);
    case 3: return qmc5_ops_d3(loops, kmax, op, grid, smem, st, p, bps);
    case 4: return qmc5_ops_d4(loops, kmax, op, grid, smem, st, p, bps);
    case 5: return qmc5_ops_d5(loops, kmax, op, grid, smem, st, p, bps);
    case 6: return qmc5_ops_d6(loops, kmax, op, grid, smem, st, p, bps);
    default: return cudaErrorInvalidValue;
  }
}
bool qmc5_kernel_available(int ndim, int loops, int kmax) {
  return ndim >= 1 && ndim <= 6 && loops >= 1 && loops <= 2 && loops <= ndim && kmax >= 0 && kmax <= 2;
}
cudaError_t qmc5_kernel_prepare(int ndim, int loops, int kmax, size_t smem, int *blocks_per_sm) {
  return ops5(ndim, loops, kmax, 0, dim3(1), smem, nullptr, nullptr, blocks_per_sm);
}
cudaError_t qmc5_kernel_launch(int ndim, int loops, int kmax, dim3 grid, size_t smem, cudaStream_t st, const Qmc5Launch &p) {
  return ops5(ndim, loops, kmax, 1, grid, smem, st, &p, nullptr);
}
