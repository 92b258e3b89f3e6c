// Kernel parameter block and the per-dimension launch entry points (internal).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "qmc_tables.h"

#define QMC_THREADS 256

// The polynomial periodising transforms as data, so that S3 of the kernels has no branch between them (a branch between
// Eq. 21 and its r = 2 sibling cost the complex kernel registers in its hot loop: cfg3 25 -> 32 ms):
//   t = y^2 (tc[0] + y (tc[1] + y (tc[2] + y tc[3]))),   weight factor = q (wc[0] + q wc[1]),  q = y (1 - y)
//   transform 0 (Eq. 21): tc = {3, -2, 0, 0}, wc = {6, 0};   transform 2 (R:C20): tc = {0, 10, -15, 6}, wc = {0, 30}.
// The coefficients sit in the kernel parameters (constant bank operands of the FMAs: no registers).  transform 1 (tent)
// keeps its branch.
inline void qmc_transform_poly(int transform, double *tc, double *wc) {
  if (transform == 2) {
    tc[0] = 0.0, tc[1] = 10.0, tc[2] = -15.0, tc[3] = 6.0, wc[0] = 0.0, wc[1] = 30.0;
  } else {
    tc[0] = 3.0, tc[1] = -2.0, tc[2] = 0.0, tc[3] = 0.0, wc[0] = 6.0, wc[1] = 0.0;
  }
}

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
  double tc[4], wc[2];           // periodising transform (see qmc_transform_poly)
  int32_t transform;
  int32_t sec_begin, sec_end, sec_per_chunk;
  int32_t persec;                // 0: fused (all sectors of the chunk summed), 1: per-sector sums
  int32_t ibp;                   // 1: pole extraction by integration by parts (Eq. 13) instead of the subtraction (Taylor flavour only)
  uint32_t tab_smem_bytes;       // shared-memory bytes reserved for the table chunk
};


#define QMC3_MAXSING 2  // complex path: sectors with more singular variables go to the version-1 kernel

// implemented in qmc_dispatch.cu on top of one translation unit per dimension (qmc_inst_d<N>.cu)
cudaError_t qmc_kernel_prepare(int ndim, int kmax, int flavor, size_t smem, int *blocks_per_sm);
cudaError_t qmc_kernel_launch(int ndim, int kmax, int flavor, dim3 grid, size_t smem, cudaStream_t st, const QmcLaunch &p);

// ---- version 4 (real path, tables in the kernel-parameter constant bank) -------------------------------------
// One launch = one run of sectors of one chunk; blockIdx.x = slice of the lattice points.  The chunk's slot program and
// the sector tables travel INSIDE the kernel parameter block (constant bank 0): every table read is a uniform load
// (LDCU) into uniform registers, slot operands are addressed [thread column + uniform offset], the record loops run on
// the uniform datapath.  A monomial record is 8 bytes {u32 off0, u32 off1}: value = slot[off0] * slot[off1] (byte offsets
// into the thread's slot column; the coefficient lives in a slot, qmc_image4.cpp).  Layout of `tab` (16-byte words):
//   [prog_word ..)  slot program: nprog x {u32 a_off, u32 b_off}, 2 per word
//   [sec_word ..)   sector blocks, back to back; sector block (word offsets relative to its start):
//     w0 = {nsing | nL0 << 8 | nlocal << 16 | nfused << 24, nwords of the block, first dense position word, 0}
//     w1 = sing_ln[4]  (byte offsets of ln t_k of the singular positions)      w2 = sing_t[4]  (of t_k)
//     w3,w4 = 1/beta[4] (f64)      w5,w6 = beta[4] (f64)
//     w7 = {f64 coefficient of G0, u32 off0, u32 off1}: G0 = c * slot * slot = c_U^aU0 c_F^aF0 prod_reg t^alpha
//     w8 = {f64 constant of L0 = aU1 ln c_U + aF1 ln c_F, 0, 0}
//     w9.. = (n - nsing) x {f64 beta_j, u32 offset of ln t_j, 0} (one per regular variable), then the local program nlocal x {u32 a_off,
//     u32 b_off} padded to a word (slot[local0 + i] = slot[a] * slot[b]), then nfused x 2 words {a, b, c, d}{dst, 0, 0, 0}
//     (slot[dst] = slot[a] * slot[b] + slot[c] * slot[d]: the overflow of groups with more monomials than dense positions),
//     then the dense positions: for U^ then F^, group by group, qmc4_cap(nsing, polynomial, popcount of the group) records
//     (qmc_tables.h; an unused position is the 0.0 slot twice), padded to a word
#define QMC4_TAB_WORDS 1820  // 29 120 bytes of tables per launch (kernel parameters are limited to 32 764 bytes)
#define QMC4_MAX_SEC 160     // sectors per launch
#define QMC4_LOG_ENTRIES 64
#define QMC4_LOG_COPIES 8
struct Qmc4Launch {
  const double *logtab;          // device: 64 x {1/c, -ln(1/c)}
  const double *shifts;          // device: [m][ndim]
  double *partial;               // device: [row][shift][max_slices][NACC]
  unsigned long long *counters;  // device: [4]
  uint32_t N, count;
  uint32_t zeff[QMC_MAXDIM], off[QMC_MAXDIM];
  int32_t m, transform, pad2, max_slices;
  int32_t nsec, out_row, count_boundary, nslices;
  uint32_t nprog, prog_word, sec_word, first_prod_off;  // first_prod_off, local0_off: byte offsets in the slot column
  uint32_t local0_off, max_nslots, nconst, sync_every;  // sync_every: block barrier every that many points (0 = never)
  double tc[4], wc[2];           // periodising transform (see qmc_transform_poly)
  double dN, invN;               // (double)N and RN(1 / N): constant-bank operands of the lattice-point division (S1)
  double cval[QMC4_MAXCONST];    // values of the coefficient-constant slots 3n + 2 ..
  int32_t nsb[QMC_MAXSING + 2];  // evaluation positions [nsb[ns], nsb[ns + 1]) hold the sectors with ns singular variables
  uint16_t secw[QMC4_MAX_SEC];  // word offset of the sector blocks in tab, in evaluation order (sorted by nsing: one code
                                // path per class, no dispatch per sector)
  uint4 tab[QMC4_TAB_WORDS];
};
static_assert(sizeof(Qmc4Launch) <= 32764, "kernel parameter limit");
cudaError_t qmc4_kernel_prepare(int ndim, int loops, int kmax, int threads, int tpl, size_t smem, int *blocks_per_sm);
cudaError_t qmc4_kernel_launch(int ndim, int loops, int kmax, int threads, int tpl, dim3 grid, size_t smem, cudaStream_t st,
                               const Qmc4Launch &p);
bool qmc4_kernel_available(int ndim, int loops, int kmax);

// ---- version 5 (complex path, tables in the kernel-parameter constant bank) ---------------------------------------
// The complex-path counterpart of version 4: one launch = one run of sectors of one chunk, grid = (slices, shifts).
// Layout of `tab` (16-byte words): [prog_r_word ..) real slot program, [prog_c_word ..) complex slot program, each
// {u32 a_off, u32 b_off} byte offsets into the thread's real (8-byte entries) resp. complex (16-byte entries) column,
// two per word; then the sector blocks (word offsets relative to the block):
//   w0 = {nsing | nL0 << 8 | nlocal_r << 16 | nlocal_c << 24, nwords, first real record (G0), 0}
//   w1 = {variable index of the singular positions (u8 x 4), 0, alpha[0..3] (i8 x 4), alpha[4..7]}
//   w2 = {beta[0..3] (i8 x 4), beta[4..7], 0, 0}      w3,w4 = 1/beta of the singular positions (f64 x 4)      w5,w6 = beta (f64 x 4)
//   w7 = word offsets of the corner blocks Z = 0..3
//   w8.. = local real program, local complex program (each padded to a word), then records [G0][L0 x nL0]
//   corner block Z (npoly = n + n(n+1)/2 + 2 polynomials: F_i, F_ik (i <= k), U, F; only the monomials free of the variables of Z
//     survive): u8 countsA[npoly] (one-factor records per polynomial; padded to a word), u8 countsB[npoly] (two-factor records),
//     f64 c0[npoly] (the constant monomials, summed on the host; padded to a word), then real A: qmc5_capA FIXED positions per
//     derivative polynomial {f64 c, u32 off, 0}: c * slot (unused: c = 0; a surplus travels in B as c * slot * 1), then three
//     record streams, each closed by two sentinels:  real B {f64 c, u32 off0, u32 off1}: c * slot * slot;  complex A, complex B
//     the same over the complex slots (U^ and F^).
//   A record is duplicated into every corner block that needs it: each corner is flat streams without skips.
struct Qmc5Launch {
  const double *logtab;          // device: 64 x {1/c, -ln(1/c)}
  const double *shifts;
  double *partial;               // [row][shift][max_slices][NACC][2]
  unsigned long long *counters;
  uint32_t N, count;
  uint32_t zeff[QMC_MAXDIM], off[QMC_MAXDIM];
  int32_t m, transform, persec, max_slices;
  int32_t nsec, out_row, count_boundary, nslices;
  uint32_t nprog_r, prog_r_word, first_prod_r_off, local0_r_off;  // *_off: byte offsets in the real column
  uint32_t nprog_c, prog_c_word, first_prod_c_off, local0_c_off;  // ... in the complex column
  uint32_t max_nslots_r, max_nslots_c, pad0, pad1;
  double lambda;
  double tc[4], wc[2];           // periodising transform (see qmc_transform_poly)
  uint16_t secw[QMC4_MAX_SEC];
  uint16_t secrow[QMC4_MAX_SEC];
  uint4 tab[QMC4_TAB_WORDS];
};
static_assert(sizeof(Qmc5Launch) <= 32764, "kernel parameter limit");
cudaError_t qmc5_kernel_prepare(int ndim, int loops, int kmax, size_t smem, int *blocks_per_sm);
cudaError_t qmc5_kernel_launch(int ndim, int loops, int kmax, dim3 grid, size_t smem, cudaStream_t st, const Qmc5Launch &p);
bool qmc5_kernel_available(int ndim, int loops, int kmax);
