// Kernel parameter block and the per-dimension launch entry points (internal).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "qmc_tables.h"

#define QMC_THREADS 256

struct QmcLaunch {
  const uint8_t *image;          // device: sector blocks
  const uint32_t *secoff;        // device: [n_sectors+1] byte offsets into image
  const double *shifts;          // device: [m][ndim]
  double *partial;               // device: block partial sums
  unsigned long long *counters;  // device: [4]
  uint32_t N, count;             // lattice size; number of lattice indices evaluated
  uint32_t zeff[QMC_MAXDIM];     // (index_step * z_j) mod N
  uint32_t off[QMC_MAXDIM];      // (index_begin * z_j) mod N
  int32_t m, kmax;
  int32_t aU0, aU1, aF0, aF1;
  double lambda;
  int32_t transform;
  int32_t sec_begin, sec_end, sec_per_chunk;
  int32_t persec;                // 0: fused (all sectors of the chunk summed), 1: per-sector sums
  uint32_t tab_smem_bytes;       // shared-memory bytes reserved for the table chunk
};


// implemented in qmc_dispatch.cu on top of one translation unit per dimension (qmc_inst_d<N>.cu)
cudaError_t qmc_kernel_prepare(int ndim, int kmax, bool cplx, size_t smem, int *blocks_per_sm);
cudaError_t qmc_kernel_launch(int ndim, int kmax, bool cplx, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch &p);
