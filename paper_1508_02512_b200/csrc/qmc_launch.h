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


// ---- version 2 (real path) --------------------------------------------------------------------------------
struct Qmc2Work {  // one block (blockIdx.x): one slice of the lattice points of a run of sectors of one chunk
  uint32_t prog_off, prog_bytes;  // chunk header + slot program in image2
  uint32_t sec_off, sec_bytes;    // the sector blocks
  int32_t s0, nsec;               // first sector (global index), number of sectors
  int32_t out_row;                // fused: row of the partial buffer; per-sector: row of the first sector
  int32_t count_boundary;         // 1 for the blocks that tally boundary points (the first run of sectors)
  int32_t slice, nslices;         // this block takes the points slice, slice + nslices, ... (in units of blocks):
                                  // runs get slices in proportion to their modelled cost
};
struct Qmc2Launch {
  const uint8_t *image2;
  const uint32_t *secoff2;       // device: [n_sectors+1]
  const Qmc2Work *work;          // device: [gridDim.y]
  const double *logtab;          // device: 128 x {1/c, -ln(1/c)}
  const double *shifts;
  double *partial;
  unsigned long long *counters;
  uint32_t N, count;
  uint32_t zeff[QMC_MAXDIM], off[QMC_MAXDIM];
  int32_t m, transform, persec;
  uint32_t sm_prog_cap, sm_sec_cap;  // shared-memory bytes reserved for the slot program and the sector blocks
  int32_t max_nsec, max_nslots;
  int32_t max_slices;            // partial buffer: [row][shift][max_slices][order], zero-filled by the launcher
};
// ---- version 3 (complex path) ------------------------------------------------------------------------------
#define QMC3_MAXSING 2  // sectors with more singular variables go to the version-1 kernel
struct Qmc3Launch {
  Qmc2Launch b;          // image2 / secoff2 here mean image3 / secoff3; max_nslots = real slots (incl. local)
  double lambda;
  int32_t max_nslots_c;  // complex slots (incl. local)
  int32_t pad;
};
cudaError_t qmc3_kernel_prepare(int ndim, int loops, int kmax, size_t smem, int *blocks_per_sm);
cudaError_t qmc3_kernel_launch(int ndim, int loops, int kmax, dim3 grid, size_t smem, cudaStream_t st, const Qmc3Launch &p);
bool qmc3_kernel_available(int ndim, int loops, int kmax);

cudaError_t qmc2_kernel_prepare(int ndim, int loops, int kmax, size_t smem, int *blocks_per_sm);
cudaError_t qmc2_kernel_launch(int ndim, int loops, int kmax, dim3 grid, size_t smem, cudaStream_t st, const Qmc2Launch &p);
bool qmc2_kernel_available(int ndim, int loops, int kmax);

// implemented in qmc_dispatch.cu on top of one translation unit per dimension (qmc_inst_d<N>.cu)
cudaError_t qmc_kernel_prepare(int ndim, int kmax, int flavor, size_t smem, int *blocks_per_sm);
cudaError_t qmc_kernel_launch(int ndim, int kmax, int flavor, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch &p);
