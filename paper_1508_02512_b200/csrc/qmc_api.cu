// C-ABI entry points (include/qmc_feynman.h), launch logic, small helper kernels.  sm_100a.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <numeric>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/qmc_feynman.h"
#include "qmc_launch.h"
#include "qmc_tables.h"

#define QMC_MAX_BLOCKS 592  // upper bound of gridDim.x used for workspace sizing (148 SMs x 4)
#define QMC_MAX_BLOCKS_BATCH 32  // the same for a batch of kinematic points (one small run per point)
#define QMC_NCAND 64        // Korobov candidates of the P_2 search
#define QMC_P2_BLOCKS 296

namespace {

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// ---- S7 (second stage): fixed-order sum of the block partials, times 1/N -----------------------------
// fused : partial [chunk][shift][block][nacc] -> out [nacc][shift]            (rows = n_chunks, summed)
// persec: partial [sector][shift][block][nacc] -> out [sector][nacc][shift]   (rows = n_sectors, kept)
__global__ void qmc_finalize_kernel(const double *partial, double *out, int rows, int m, int nblocks, int nacc,
                                    double invN, int persec) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  int total = (persec ? rows : 1) * nacc * m;
  if (idx >= total) return;
  int kap = idx % m, a = (idx / m) % nacc, row = idx / (m * nacc);
  double s = 0.0;
  if (persec) {
    const double *src = partial + (((size_t)row * m + kap) * nblocks) * nacc + a;
    for (int b = 0; b < nblocks; ++b) s += src[(size_t)b * nacc];
  } else {
    for (int c = 0; c < rows; ++c) {
      const double *src = partial + (((size_t)c * m + kap) * nblocks) * nacc + a;
      for (int b = 0; b < nblocks; ++b) s += src[(size_t)b * nacc];
    }
  }
  out[idx] = s * invN;
}

// batch of kinematic points (mode 3): partial [run][shift][block][nacc], the runs of row r are [run_begin[r], run_begin[r + 1])
// -> out [row][nacc][shift]
__global__ void qmc_finalize_rows_kernel(const double *partial, double *out, const int *run_begin, int nrows, int m, int nblocks,
                                         int nacc, double invN) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nrows * nacc * m) return;
  int kap = idx % m, a = (idx / m) % nacc, row = idx / (m * nacc);
  double s = 0.0;
  for (int c = run_begin[row]; c < run_begin[row + 1]; ++c) {
    const double *src = partial + (((size_t)c * m + kap) * nblocks) * nacc + a;
    for (int b = 0; b < nblocks; ++b) s += src[(size_t)b * nacc];
  }
  out[idx] = s * invN;
}

// ---- generating vector: P_2 figure of merit of Korobov candidates (R:C13) ----------------------------
// P2(z) = -1 + (1/N) sum_i prod_j (1 + 2 pi^2 B_2({i z_j / N})),  B_2(x) = x^2 - x + 1/6
__global__ void qmc_p2_kernel(const uint32_t *zc /*[ncand][8]*/, double *partial /*[ncand][gridDim.x]*/, uint32_t N,
                              int dim) {
  const int cand = blockIdx.y;
  const uint32_t *z = zc + cand * QMC_MAXDIM;
  const double invN = 1.0 / (double)N;
  const double c2 = 2.0 * 9.86960440108935861883;
  double s = 0.0;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += stride) {
    double prod = 1.0;
    for (int j = 0; j < dim; ++j) {
      uint32_t r = (uint32_t)(((uint64_t)i * z[j]) % N);
      double x = (double)r * invN;
      prod *= 1.0 + c2 * (x * x - x + 1.0 / 6.0);
    }
    s += prod;
  }
  __shared__ double sh[8];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += sh[w];
    partial[(size_t)cand * gridDim.x + blockIdx.x] = t;
  }
}

// ---- FP64 FMA peak: 8 independent register-resident DFMA chains per thread ---------------------------
__global__ void __launch_bounds__(256) qmc_dfma_peak_kernel(double *sink, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
  if (s == 12345.678) sink[0] = s;  // never true; keeps the chains alive
}

// ---- S8: statistics over the shifts (Eqs. 19-20), Re and Im separately (R:C15) ------------
// in : out [row][nacc*nc][m] (row = sector in per-sector mode, a single row in fused mode)
// stat (doubles): totals [K][m][2] | coeff [K][2] | err [K][2] | sector_coeff [nrows][K][2] | sector_err [nrows][K][2]
//                 | shift_sums [nrows][K][m][2]           (nrows = 0 in fused mode)
// One thread per (row or total, order, Re/Im); sums run in a fixed order.
struct StatLayout {
  size_t totals, coeff, err, sector_coeff, sector_err, shift_sums, total;
};
__host__ __device__ inline StatLayout stat_layout(int nrows, int K, int m) {
  StatLayout S;
  size_t o = 0;
  S.totals = o; o += (size_t)K * m * 2;
  S.coeff = o; o += (size_t)K * 2;
  S.err = o; o += (size_t)K * 2;
  S.sector_coeff = o; o += (size_t)nrows * K * 2;
  S.sector_err = o; o += (size_t)nrows * K * 2;
  S.shift_sums = o; o += (size_t)nrows * K * m * 2;
  S.total = o;
  return S;
}
__global__ void qmc_stats_kernel(const double *out, double *stat, int nrows, int K, int m, int nacc, int nc, int acc0) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (nrows + 1) * K * 2) return;
  const int c = idx & 1, k = (idx >> 1) % K, row = (idx >> 1) / K;
  const StatLayout S = stat_layout(nrows, K, m);
  const int a = (acc0 + k) * nc + c;  // accumulator of order k_min + k
  const bool total = row == nrows;
  const int r0 = total ? 0 : row, r1 = total ? (nrows ? nrows : 1) : row + 1;
  double *v = total ? stat + S.totals + (size_t)k * m * 2 + c : stat + S.shift_sums + ((size_t)row * K + k) * m * 2 + c;
  double s = 0.0;
  for (int kap = 0; kap < m; ++kap) {
    double x = 0.0;
    if (c < nc)
      for (int r = r0; r < r1; ++r) x += out[((size_t)r * nacc * nc + a) * m + kap];
    v[2 * kap] = x;
    s += x;
  }
  const double q = s / m;
  double d2 = 0.0;
  for (int kap = 0; kap < m; ++kap) {
    double d = v[2 * kap] - q;
    d2 += d * d;
  }
  const double e = sqrt(d2 / ((double)m * (m - 1)));
  if (total) {
    stat[S.coeff + 2 * k + c] = q;
    stat[S.err + 2 * k + c] = e;
  } else {
    stat[S.sector_coeff + ((size_t)row * K + k) * 2 + c] = q;
    stat[S.sector_err + ((size_t)row * K + k) * 2 + c] = e;
  }
}

uint64_t splitmix64(uint64_t &state) {
  state += 0x9E3779B97F4A7C15ull;
  uint64_t x = state;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}

uint64_t mulmod(uint64_t a, uint64_t b, uint64_t n) { return (uint64_t)(((unsigned __int128)a * b) % n); }

struct DevLayout {
  size_t image, secoff, logtab4, shifts, counters, out, stat, partial, p2z, p2partial, runbegin, total;
};

DevLayout layout(const qmc_tables *t, int m) {
  DevLayout L;
  size_t nsec = t->sectors.size();
  size_t o = 0;
  L.image = o; o += align256(t->image.size());
  L.secoff = o; o += align256((nsec + 1) * 4);
  L.logtab4 = o; o += align256(sizeof t->logtab4);
  L.shifts = o; o += align256((size_t)m * QMC_MAXDIM * 8);
  L.counters = o; o += 256;
  L.out = o; o += align256(nsec * QMC_NACC_MAX * 2 * (size_t)m * 8);
  L.stat = o; o += align256(stat_layout((int)nsec, QMC_MAXK, m).total * 8);
  L.partial = o; o += align256(nsec * (size_t)m * (t->n_rows > 1 ? QMC_MAX_BLOCKS_BATCH : QMC_MAX_BLOCKS) * QMC_NACC_MAX * 2 * 8);
  L.p2z = o; o += align256((size_t)QMC_NCAND * QMC_MAXDIM * 4);
  L.p2partial = o; o += align256((size_t)QMC_NCAND * QMC_P2_BLOCKS * 8);
  L.runbegin = o; o += align256((nsec + 2) * 4);
  L.total = o;
  return L;
}

#define CUDA_OK(x)                      \
  do {                                  \
    if ((x) != cudaSuccess) {           \
      cudaGetLastError();               \
      return QMC_ECUDA;                 \
    }                                   \
  } while (0)

// ---- allocation-free variant of the P_2 search (qmc_generating_vector_noalloc) ------------------------------------------
// Its scratch (candidate vectors + per-block partial sums of qmc_p2_kernel) lives in a file-scope device array of FIXED
// size: 2 048 + 64 x 296 x 8 = 153 600 bytes, held by every GPU that loads the library until the process exits.  In host
// code the array's name is a host-side stand-in, NOT a device address: the address is fetched once per device with
// cudaGetSymbolAddress (that device current) and handed to the kernel.
#define QMC_NOALLOC_P2Z_BYTES 2048u
#define QMC_NOALLOC_BYTES (QMC_NOALLOC_P2Z_BYTES + (size_t)QMC_NCAND * QMC_P2_BLOCKS * 8)
static_assert((size_t)QMC_NCAND * QMC_MAXDIM * 4 <= QMC_NOALLOC_P2Z_BYTES, "candidate block of the P_2 search");
static __device__ __align__(256) unsigned char qmc_noalloc_scratch[QMC_NOALLOC_BYTES];
#define QMC_NOALLOC_MAXDEV 64
unsigned char *noalloc_addr[QMC_NOALLOC_MAXDEV] = {nullptr};  // device address of qmc_noalloc_scratch, per device

int korobov_search(uint64_t N, int dim, cudaStream_t st, unsigned char *ws, size_t p2z_off, size_t p2p_off,
                   uint64_t *z_out) {
  if (dim == 1) {
    z_out[0] = 1;
    return QMC_OK;
  }
  std::vector<uint32_t> zc((size_t)QMC_NCAND * QMC_MAXDIM, 0);
  std::vector<uint64_t> cand;
  uint64_t state = N;
  int guard = 0;
  while ((int)cand.size() < QMC_NCAND && guard++ < 100000) {
    uint64_t a = 2 + splitmix64(state) % (N - 3);
    if (std::gcd(a, N) != 1) continue;
    cand.push_back(a);
  }
  if (cand.empty()) return QMC_EINVAL;
  int nc = (int)cand.size();
  for (int c = 0; c < nc; ++c) {
    uint64_t v = 1;
    for (int j = 0; j < dim; ++j) {
      zc[(size_t)c * QMC_MAXDIM + j] = (uint32_t)v;
      v = mulmod(v, cand[c], N);
    }
  }
  uint32_t *dz = reinterpret_cast<uint32_t *>(ws + p2z_off);
  double *dp = reinterpret_cast<double *>(ws + p2p_off);
  CUDA_OK(cudaMemcpyAsync(dz, zc.data(), zc.size() * 4, cudaMemcpyHostToDevice, st));
  qmc_p2_kernel<<<dim3(QMC_P2_BLOCKS, nc), 256, 0, st>>>(dz, dp, (uint32_t)N, dim);
  CUDA_OK(cudaGetLastError());
  std::vector<double> part((size_t)nc * QMC_P2_BLOCKS);
  CUDA_OK(cudaMemcpyAsync(part.data(), dp, part.size() * 8, cudaMemcpyDeviceToHost, st));
  CUDA_OK(cudaStreamSynchronize(st));
  int best = 0;
  double bestv = 0.0;
  for (int c = 0; c < nc; ++c) {
    double s = 0.0;
    for (int b = 0; b < QMC_P2_BLOCKS; ++b) s += part[(size_t)c * QMC_P2_BLOCKS + b];
    double p2 = s / (double)N - 1.0;
    if (c == 0 || p2 < bestv || (p2 == bestv && cand[c] < cand[best])) {
      best = c;
      bestv = p2;
    }
  }
  for (int j = 0; j < dim; ++j) z_out[j] = zc[(size_t)best * QMC_MAXDIM + j];
  return QMC_OK;
}

// Eqs. 19-20 on per-shift values v[kap] (stride in doubles)
void mean_err(const double *v, size_t stride, int m, double *mean, double *err) {
  double s = 0.0;
  for (int k = 0; k < m; ++k) s += v[k * stride];
  double q = s / m, d2 = 0.0;
  for (int k = 0; k < m; ++k) {
    double d = v[k * stride] - q;
    d2 += d * d;
  }
  *mean = q;
  *err = std::sqrt(d2 / ((double)m * (m - 1)));
}

// ---- version-4 launch (real path): one launch per run of sectors, tables in the kernel parameters ------------------
// Runs = maximal pieces of a chunk whose tables fit QMC4_TAB_WORDS (and, in per-sector mode, whose accumulators fit
// the shared memory).  grid = (point slices, shift vectors); slices in proportion to the modelled cost of the run.
// The launches are independent (disjoint rows of the partial buffer): they are spread over side streams forked from
// and joined back into the caller's stream, so that the tail of one launch overlaps the next ones.
int launch_v4(qmc_tables *t, const DevLayout &L, unsigned char *ws, cudaStream_t st, uint64_t N, int m, int sb, int se,
              bool persec, uint64_t ibeg, uint64_t istep, uint64_t icount, const uint64_t *z, int sms, int smem_optin,
              int waves_opt, int streams_opt, const uint8_t *mask, const int *rowmap, std::vector<int> *row_of_run, int *gx_out,
              int *rows_out, int *launches_out, size_t *h2d, cudaError_t *ce_out) {
  const int n = t->n, nacc = QMC_MAXSING + t->kmax + 1, T = t->threads_real;
  const size_t budget = (size_t)smem_optin - 1024;
  // shared memory of a launch: logarithm table, shift vectors, reduction scratch, the chunk's slot columns.
  // Per-sector mode = one launch per sector (its accumulators are then registers like in the fused mode).
  auto fixed_of = [&](const Qmc2Chunk &c) {
    return (size_t)QMC4_LOG_ENTRIES * QMC4_LOG_COPIES * 16 + (((size_t)m * n * 8 + 15) & ~(size_t)15) + (T / 32) * 8 +
           (size_t)(c.nslots + c.max_local) * T * 8;
  };
  struct Run { int chunk, a, b; double cost; size_t smem; };
  std::vector<Run> runs;
  double total_cost = 0.0;
  size_t smem = 0;
  for (size_t ci = 0; ci < t->chunks.size(); ++ci) {
    const Qmc2Chunk &c = t->chunks[ci];
    int a = std::max(sb, c.sec_begin);
    const int e = std::min(se, c.sec_end);
    const size_t prog_words = t->prog4[ci].size() / 4;
    const size_t fixed = fixed_of(c);
    if (a < e && fixed > budget) return QMC_ENOMEM;
    while (a < e) {
      int b = a;
      while (b < e) {
        const size_t words = prog_words + (t->secoff4[b + 1] - t->secoff4[a]);
        if (words > QMC4_TAB_WORDS || b + 1 - a > QMC4_MAX_SEC || (persec && b > a)) break;
        if (rowmap && b > a && rowmap[b] != rowmap[a]) break;  // a run never mixes kinematic points
        ++b;
      }
      if (b == a) return QMC_ENOMEM;
      Run r = {(int)ci, a, b, 0.0, fixed};
      for (int s = a; s < b; ++s)
        if (!mask || mask[s]) r.cost += t->sec_cost[s];
      total_cost += r.cost;
      smem = std::max(smem, r.smem);
      runs.push_back(r);
      a = b;
    }
  }
  const int nitems = (int)runs.size();
  int bps = 0;
  CUDA_OK(qmc4_kernel_prepare(n, t->L, t->kmax, T, t->tpl_real, smem, &bps));
  if (bps < 1) return QMC_ECUDA;
  const int waves = waves_opt > 0 ? waves_opt : 16;
  const long long max_slices_pts = std::max<long long>(1, (long long)((icount + T - 1) / T));
  const double nblocks_target = (double)waves * sms * bps / (double)m;  // a block serves ONE shift vector
  std::vector<int> nsl(nitems);
  int max_slices = 1;
  for (int i = 0; i < nitems; ++i) {
    long long ns = total_cost > 0.0 ? (long long)(nblocks_target * runs[i].cost / total_cost + 0.5) : 1;
    if (persec) ns = std::max<long long>(ns, (sms + 4 * m - 1) / (4 * m));  // one small launch per sector: a quarter wave each
    if (rowmap) ns = std::max<long long>(ns, (2LL * sms * bps + (long long)m * 4 - 1) / ((long long)m * 4));  // one small launch per point
    ns = std::max<long long>(1, std::min<long long>({ns, (long long)(rowmap ? QMC_MAX_BLOCKS_BATCH : QMC_MAX_BLOCKS), max_slices_pts}));
    nsl[i] = (int)ns;
    max_slices = std::max(max_slices, (int)ns);
  }
  const int rows_partial = persec ? (se - sb) : nitems;
  CUDA_OK(cudaMemsetAsync(ws + L.partial, 0, (size_t)rows_partial * m * max_slices * nacc * 8, st));
  // side streams
  int nstreams = streams_opt < 0 ? 0 : (streams_opt == 0 ? 4 : std::min(8, streams_opt));
  nstreams = std::min(nstreams, nitems);
  if (nstreams < 2) nstreams = 0;
  for (int q = 0; q < nstreams; ++q)
    if (!t->side_streams[q]) {
      CUDA_OK(cudaStreamCreateWithFlags(reinterpret_cast<cudaStream_t *>(&t->side_streams[q]), cudaStreamNonBlocking));
    }
  for (int q = 0; q < nstreams + 1; ++q)
    if (!t->side_events[q]) {
      CUDA_OK(cudaEventCreateWithFlags(reinterpret_cast<cudaEvent_t *>(&t->side_events[q]), cudaEventDisableTiming));
    }
  static thread_local Qmc4Launch p;  // 30 KB: not on the stack
  std::memset(&p, 0, offsetof(Qmc4Launch, tab));
  p.logtab = reinterpret_cast<const double *>(ws + L.logtab4);
  p.shifts = reinterpret_cast<const double *>(ws + L.shifts);
  p.partial = reinterpret_cast<double *>(ws + L.partial);
  p.counters = reinterpret_cast<unsigned long long *>(ws + L.counters);
  p.N = (uint32_t)N;
  p.count = (uint32_t)icount;
  for (int j = 0; j < n; ++j) {
    p.zeff[j] = (uint32_t)mulmod(istep % N, z[j], N);
    p.off[j] = (uint32_t)mulmod(ibeg, z[j], N);
  }
  p.m = m;
  p.transform = t->transform;
  qmc_transform_poly(t->transform, p.tc, p.wc);
  p.max_slices = max_slices;
  p.dN = (double)N;
  p.invN = 1.0 / (double)N;
  p.sync_every = 4;  // measured on B200 (kernels): a block barrier every fourth point
  cudaEventRecord(static_cast<cudaEvent_t>(t->ev0), st);
  if (nstreams) {
    cudaEventRecord(static_cast<cudaEvent_t>(t->side_events[nstreams]), st);
    for (int q = 0; q < nstreams; ++q)
      cudaStreamWaitEvent(static_cast<cudaStream_t>(t->side_streams[q]), static_cast<cudaEvent_t>(t->side_events[nstreams]), 0);
  }
  cudaError_t ce = cudaSuccess;
  for (int i = 0; i < nitems && ce == cudaSuccess; ++i) {
    const Run &r = runs[i];
    const Qmc2Chunk &c = t->chunks[r.chunk];
    const std::vector<uint32_t> &pg = t->prog4[r.chunk];
    p.nsec = r.b - r.a;
    p.out_row = persec ? r.a - sb : i;
    p.count_boundary = i == 0 ? 1 : 0;
    p.nslices = nsl[i];
    p.max_nslots = (uint32_t)(c.nslots + c.max_local);
    p.nconst = (uint32_t)c.nconst;
    for (int q = 0; q < c.nconst; ++q) p.cval[q] = t->const4[r.chunk][q];
    p.nprog = (uint32_t)(c.nslots - (2 * n + 2 + c.nconst));
    p.prog_word = 0;
    p.sec_word = (uint32_t)(pg.size() / 4);
    p.first_prod_off = (uint32_t)(2 * n + 2 + c.nconst) * T * 8u;
    p.local0_off = (uint32_t)c.nslots * T * 8u;
    uint32_t *tw = reinterpret_cast<uint32_t *>(p.tab);
    std::memcpy(tw, pg.data(), pg.size() * 4);
    const size_t w0 = t->secoff4[r.a], w1 = t->secoff4[r.b];
    std::memcpy(tw + pg.size(), t->tab4.data() + w0 * 4, (w1 - w0) * 16);
    {  // evaluation order: by number of singular variables (stable)
      int k = 0;
      for (int ns = 0; ns <= QMC_MAXSING; ++ns) {
        p.nsb[ns] = k;
        for (int s = r.a; s < r.b; ++s)
          if (t->sectors[s].nsing == ns && (!mask || mask[s])) p.secw[k++] = (uint16_t)(p.sec_word + (t->secoff4[s] - w0));
      }
      p.nsb[QMC_MAXSING + 1] = k;
      if (k == 0) continue;  // no sector of this run is selected (qmc_run.sector_mask): its row of partials stays zero
    }
    cudaStream_t ls = nstreams ? static_cast<cudaStream_t>(t->side_streams[i % nstreams]) : st;
    ce = qmc4_kernel_launch(n, t->L, t->kmax, T, t->tpl_real, dim3((unsigned)nsl[i], (unsigned)m), r.smem, ls, p);
    *h2d += offsetof(Qmc4Launch, tab) + pg.size() * 4 + (w1 - w0) * 16;  // the tables travel with the launch
  }
  if (nstreams)
    for (int q = 0; q < nstreams; ++q) {
      cudaEventRecord(static_cast<cudaEvent_t>(t->side_events[q]), static_cast<cudaStream_t>(t->side_streams[q]));
      cudaStreamWaitEvent(st, static_cast<cudaEvent_t>(t->side_events[q]), 0);
    }
  cudaEventRecord(static_cast<cudaEvent_t>(t->evm), st);
  if (rowmap && row_of_run) {
    row_of_run->clear();
    for (const Run &r : runs) row_of_run->push_back(rowmap[r.a]);
  }
  *ce_out = ce;
  *gx_out = max_slices;
  *rows_out = nitems;
  *launches_out = nitems;
  return QMC_OK;
}

// ---- version-5 launch (complex path): as version 4, two slot tables per thread ------------------------------------------
int launch_v5(qmc_tables *t, const DevLayout &L, unsigned char *ws, cudaStream_t st, uint64_t N, int m, int sb, int se,
              bool persec, uint64_t ibeg, uint64_t istep, uint64_t icount, const uint64_t *z, int sms, int smem_optin,
              int waves_opt, int streams_opt, const uint8_t *mask, const int *rowmap, std::vector<int> *row_of_run, int *gx_out,
              int *rows_out, int *launches_out, size_t *h2d, cudaError_t *ce_out) {
  const int n = t->n, nacc = 2 * (QMC_MAXSING + t->kmax + 1), T = QMC3_THREADS;  // accumulators: (Re, Im) per order
  int max_r = 0, max_c = 0;
  for (size_t ci = 0; ci < t->chunks3.size(); ++ci) {
    const Qmc2Chunk &c = t->chunks3[ci];
    if (c.sec_end > sb && c.sec_begin < se) {
      max_r = std::max(max_r, c.nslots + c.max_local);
      max_c = std::max(max_c, t->chunk3_nslots_c[ci] + t->chunk3_max_local_c[ci]);
    }
  }
  const size_t budget = (size_t)smem_optin - 1024;
  const size_t fixed = (size_t)QMC4_LOG_ENTRIES * QMC4_LOG_COPIES * 16 + (((size_t)m * n * 8 + 15) & ~(size_t)15) + (T / 32) * 8 +
                       (size_t)max_r * T * 8 + (size_t)max_c * T * 16;
  const size_t accbytes = persec ? (size_t)nacc * T * 8 : 0;
  if (fixed + accbytes > budget) return QMC_ENOMEM;
  struct Run { int chunk, a, b; double cost; };
  std::vector<Run> runs;
  double total_cost = 0.0;
  int max_nsec = 0;
  for (size_t ci = 0; ci < t->chunks3.size(); ++ci) {
    const Qmc2Chunk &c = t->chunks3[ci];
    int a = std::max(sb, c.sec_begin);
    const int e = std::min(se, c.sec_end);
    const size_t prog_words = (t->prog5r[ci].size() + t->prog5c[ci].size()) / 4;
    while (a < e) {
      int b = a;
      while (b < e) {
        const size_t words = prog_words + (t->secoff5[b + 1] - t->secoff5[a]);
        if (words > QMC4_TAB_WORDS || b + 1 - a > QMC4_MAX_SEC || fixed + accbytes * (b + 1 - a) > budget) break;
        if (rowmap && b > a && rowmap[b] != rowmap[a]) break;  // a run never mixes kinematic points
        ++b;
      }
      if (b == a) return QMC_ENOMEM;
      Run r = {(int)ci, a, b, 0.0};
      for (int s = a; s < b; ++s)
        if (!mask || mask[s]) r.cost += t->sec_cost[s];
      total_cost += r.cost;
      max_nsec = std::max(max_nsec, b - a);
      runs.push_back(r);
      a = b;
    }
  }
  const int nitems = (int)runs.size();
  const size_t smem = fixed + accbytes * max_nsec;
  int bps = 0;
  CUDA_OK(qmc5_kernel_prepare(n, t->L, t->kmax, smem, &bps));
  if (bps < 1) return QMC_ECUDA;
  const int waves = waves_opt > 0 ? waves_opt : 16;
  const long long max_slices_pts = std::max<long long>(1, (long long)((icount + T - 1) / T));
  const double nblocks_target = (double)waves * sms * bps / (double)m;
  std::vector<int> nsl(nitems);
  int max_slices = 1;
  for (int i = 0; i < nitems; ++i) {
    long long ns = total_cost > 0.0 ? (long long)(nblocks_target * runs[i].cost / total_cost + 0.5) : 1;
    if (rowmap) ns = std::max<long long>(ns, (2LL * sms * bps + (long long)m * 4 - 1) / ((long long)m * 4));  // one small launch per point
    ns = std::max<long long>(1, std::min<long long>({ns, (long long)(rowmap ? QMC_MAX_BLOCKS_BATCH : QMC_MAX_BLOCKS), max_slices_pts}));
    nsl[i] = (int)ns;
    max_slices = std::max(max_slices, (int)ns);
  }
  const int rows_partial = persec ? (se - sb) : nitems;
  CUDA_OK(cudaMemsetAsync(ws + L.partial, 0, (size_t)rows_partial * m * max_slices * nacc * 8, st));
  int nstreams = streams_opt < 0 ? 0 : (streams_opt == 0 ? 4 : std::min(8, streams_opt));
  nstreams = std::min(nstreams, nitems);
  if (nstreams < 2) nstreams = 0;
  for (int q = 0; q < nstreams; ++q)
    if (!t->side_streams[q]) {
      CUDA_OK(cudaStreamCreateWithFlags(reinterpret_cast<cudaStream_t *>(&t->side_streams[q]), cudaStreamNonBlocking));
    }
  for (int q = 0; q < nstreams + 1; ++q)
    if (!t->side_events[q]) {
      CUDA_OK(cudaEventCreateWithFlags(reinterpret_cast<cudaEvent_t *>(&t->side_events[q]), cudaEventDisableTiming));
    }
  static thread_local Qmc5Launch p;
  std::memset(&p, 0, offsetof(Qmc5Launch, tab));
  p.logtab = reinterpret_cast<const double *>(ws + L.logtab4);
  p.shifts = reinterpret_cast<const double *>(ws + L.shifts);
  p.partial = reinterpret_cast<double *>(ws + L.partial);
  p.counters = reinterpret_cast<unsigned long long *>(ws + L.counters);
  p.N = (uint32_t)N;
  p.count = (uint32_t)icount;
  for (int j = 0; j < n; ++j) {
    p.zeff[j] = (uint32_t)mulmod(istep % N, z[j], N);
    p.off[j] = (uint32_t)mulmod(ibeg, z[j], N);
  }
  p.m = m;
  p.transform = t->transform;
  qmc_transform_poly(t->transform, p.tc, p.wc);
  p.persec = persec ? 1 : 0;
  p.max_slices = max_slices;
  p.max_nslots_r = (uint32_t)max_r;
  p.max_nslots_c = (uint32_t)max_c;
  p.lambda = t->lambda;
  cudaEventRecord(static_cast<cudaEvent_t>(t->ev0), st);
  if (nstreams) {
    cudaEventRecord(static_cast<cudaEvent_t>(t->side_events[nstreams]), st);
    for (int q = 0; q < nstreams; ++q)
      cudaStreamWaitEvent(static_cast<cudaStream_t>(t->side_streams[q]), static_cast<cudaEvent_t>(t->side_events[nstreams]), 0);
  }
  cudaError_t ce = cudaSuccess;
  for (int i = 0; i < nitems && ce == cudaSuccess; ++i) {
    const Run &r = runs[i];
    const Qmc2Chunk &c = t->chunks3[r.chunk];
    const std::vector<uint32_t> &pgr = t->prog5r[r.chunk], &pgc = t->prog5c[r.chunk];
    const int nslots_c = t->chunk3_nslots_c[r.chunk];
    p.nsec = r.b - r.a;
    p.out_row = persec ? r.a - sb : i;
    p.count_boundary = i == 0 ? 1 : 0;
    p.nslices = nsl[i];
    p.nprog_r = (uint32_t)(c.nslots - (2 * n + 1));
    p.prog_r_word = 0;
    p.first_prod_r_off = (uint32_t)(2 * n + 1) * T * 8u;
    p.local0_r_off = (uint32_t)c.nslots * T * 8u;
    p.nprog_c = (uint32_t)(nslots_c - (n + 1));
    p.prog_c_word = (uint32_t)(pgr.size() / 4);
    p.first_prod_c_off = (uint32_t)(n + 1) * T * 16u;
    p.local0_c_off = (uint32_t)nslots_c * T * 16u;
    const uint32_t sec_word = (uint32_t)((pgr.size() + pgc.size()) / 4);
    uint32_t *tw = reinterpret_cast<uint32_t *>(p.tab);
    std::memcpy(tw, pgr.data(), pgr.size() * 4);
    std::memcpy(tw + pgr.size(), pgc.data(), pgc.size() * 4);
    const size_t w0 = t->secoff5[r.a], w1 = t->secoff5[r.b];
    std::memcpy(tw + pgr.size() + pgc.size(), t->tab5.data() + w0 * 4, (w1 - w0) * 16);
    {
      int k = 0;
      for (int ns = 0; ns <= QMC_MAXSING; ++ns)
        for (int s = r.a; s < r.b; ++s)
          if (t->sectors[s].nsing == ns && (!mask || mask[s])) {
            p.secw[k] = (uint16_t)(sec_word + (t->secoff5[s] - w0));
            p.secrow[k] = (uint16_t)(s - r.a);
            ++k;
          }
      p.nsec = k;
      if (k == 0) continue;  // no sector of this run is selected (qmc_run.sector_mask)
    }
    cudaStream_t ls = nstreams ? static_cast<cudaStream_t>(t->side_streams[i % nstreams]) : st;
    ce = qmc5_kernel_launch(n, t->L, t->kmax, dim3((unsigned)nsl[i], (unsigned)m), smem, ls, p);
    *h2d += offsetof(Qmc5Launch, tab) + (pgr.size() + pgc.size()) * 4 + (w1 - w0) * 16;
  }
  if (nstreams)
    for (int q = 0; q < nstreams; ++q) {
      cudaEventRecord(static_cast<cudaEvent_t>(t->side_events[q]), static_cast<cudaStream_t>(t->side_streams[q]));
      cudaStreamWaitEvent(st, static_cast<cudaEvent_t>(t->side_events[q]), 0);
    }
  cudaEventRecord(static_cast<cudaEvent_t>(t->evm), st);
  if (rowmap && row_of_run) {
    row_of_run->clear();
    for (const Run &r : runs) row_of_run->push_back(rowmap[r.a]);
  }
  *ce_out = ce;
  *gx_out = max_slices;
  *rows_out = nitems;
  *launches_out = nitems;
  return QMC_OK;
}

}  // namespace

// =====================================================================================================
extern "C" {

int qmc_prepare(const qmc_graph *graph, const qmc_kinematics *kin, int32_t eps_order, const qmc_options *options,
                qmc_tables **out) {
  if (!out) return QMC_EINVAL;
  *out = nullptr;
  qmc_tables *t = new (std::nothrow) qmc_tables;
  if (!t) return QMC_ENOMEM;
  int rc;
  try {
    rc = qmc_build_tables(graph, kin, eps_order, options, t);
  } catch (...) {
    rc = QMC_ENOMEM;
  }
  if (rc != QMC_OK) {
    delete t;
    return rc;
  }
  *out = t;
  return QMC_OK;
}

int qmc_prepare_batch(const qmc_graph *graph, const qmc_kinematics *kinematics, int32_t n_points, int32_t eps_order,
                      const qmc_options *options, qmc_tables **out) {
  if (!out) return QMC_EINVAL;
  *out = nullptr;
  qmc_tables *t = new (std::nothrow) qmc_tables;
  if (!t) return QMC_ENOMEM;
  int rc;
  try {
    rc = qmc_build_tables_batch(graph, kinematics, n_points, eps_order, options, t);
  } catch (...) {
    rc = QMC_ENOMEM;
  }
  if (rc != QMC_OK) {
    delete t;
    return rc;
  }
  *out = t;
  return QMC_OK;
}

int qmc_tables_batch_info(const qmc_tables *t, int32_t *n_points, int32_t *sectors_per_point) {
  if (!t) return QMC_EINVAL;
  if (n_points) *n_points = t->n_rows;
  if (sectors_per_point) *sectors_per_point = t->n_rows > 0 ? (int32_t)(t->sectors.size() / t->n_rows) : 0;
  return QMC_OK;
}

void qmc_tables_free(qmc_tables *t) {
  if (t && t->ev0) {
    cudaEventDestroy(static_cast<cudaEvent_t>(t->ev0));
    cudaEventDestroy(static_cast<cudaEvent_t>(t->ev1));
    cudaEventDestroy(static_cast<cudaEvent_t>(t->evm));
  }
  if (t) {
    for (void *&q : t->side_streams)
      if (q) cudaStreamDestroy(static_cast<cudaStream_t>(q));
    for (void *&q : t->side_events)
      if (q) cudaEventDestroy(static_cast<cudaEvent_t>(q));
  }
  delete t;
}

int qmc_tables_info(const qmc_tables *t, int32_t *n_sectors, int32_t *dim, int32_t *k_min, int32_t *k_max,
                    int32_t *is_complex) {
  if (!t) return QMC_EINVAL;
  if (n_sectors) *n_sectors = (int32_t)t->sectors.size();
  if (dim) *dim = t->n;
  if (k_min) *k_min = t->kmin;
  if (k_max) *k_max = t->kmax;
  if (is_complex) *is_complex = t->lambda > 0.0 ? 1 : 0;
  return QMC_OK;
}

int qmc_tables_export(const qmc_tables *t, void *buf, size_t *len) {
  if (!t || !len) return QMC_EINVAL;
  size_t words = 12;
  for (const QmcSector &s : t->sectors) words += 1 + 2 * (size_t)t->n + 2 + (s.U.size() + s.F.size()) * (1 + (size_t)t->n);
  size_t need = words * 8;
  if (!buf) {
    *len = need;
    return QMC_OK;
  }
  if (*len < need) {
    *len = need;
    return QMC_ENOMEM;
  }
  int64_t *w = static_cast<int64_t *>(buf);
  double *d = static_cast<double *>(buf);
  size_t p = 0;
  w[p++] = 0x514D4346;
  w[p++] = 1;
  w[p++] = (int64_t)t->sectors.size();
  w[p++] = t->n;
  w[p++] = t->kmin;
  w[p++] = t->kmax;
  w[p++] = (t->lambda > 0.0 ? 1 : 0) + (t->ibp ? 2 : 0);
  w[p++] = t->aU0;
  w[p++] = t->aU1;
  w[p++] = t->aF0;
  w[p++] = t->aF1;
  d[p++] = t->lambda;
  for (const QmcSector &s : t->sectors) {
    w[p++] = s.primary;
    for (int j = 0; j < t->n; ++j) w[p++] = s.alpha[j];
    for (int j = 0; j < t->n; ++j) w[p++] = s.beta[j];
    w[p++] = (int64_t)s.U.size();
    w[p++] = (int64_t)s.F.size();
    for (int which = 0; which < 2; ++which)
      for (const QmcMono &m : (which ? s.F : s.U)) {
        d[p++] = m.c;
        for (int j = 0; j < t->n; ++j) w[p++] = m.e[j];
      }
  }
  *len = need;
  return QMC_OK;
}

size_t qmc_workspace_bytes(const qmc_tables *t, uint64_t, int32_t m) {
  if (!t || m < 1) return 0;
  return layout(t, m).total;
}

int qmc_shifts(uint64_t seed, int32_t m, int32_t dim, double *shifts_out) {
  if (m < 1 || dim < 1 || !shifts_out) return QMC_EINVAL;
  uint64_t state = seed;
  for (int k = 0; k < m; ++k)
    for (int j = 0; j < dim; ++j) shifts_out[(size_t)k * dim + j] = (double)(splitmix64(state) >> 11) * (1.0 / 9007199254740992.0);
  return QMC_OK;
}

int qmc_generating_vector(uint64_t N, int32_t dim, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                          uint64_t *z_out) {
  if (N < 5 || N >= (1ull << 31) || dim < 1 || dim > QMC_MAXDIM || !z_out) return QMC_EINVAL;
  size_t p2z = 0, p2p = align256((size_t)QMC_NCAND * QMC_MAXDIM * 4);
  if (dim > 1 && (!dev_workspace || dev_workspace_bytes < p2p + (size_t)QMC_NCAND * QMC_P2_BLOCKS * 8)) return QMC_ENOMEM;
  return korobov_search(N, dim, static_cast<cudaStream_t>(cuda_stream), static_cast<unsigned char *>(dev_workspace), p2z,
                        p2p, z_out);
}

int qmc_generating_vector_noalloc(uint64_t N, int32_t dim, void *cuda_stream, uint64_t *z_out) {
  if (N < 5 || N >= (1ull << 31) || dim < 1 || !z_out) return QMC_EINVAL;
  if (dim > QMC_MAXDIM) return QMC_ENOMEM;  // beyond what the fixed scratch (and the kernels) are sized for
  if (dim == 1) {
    z_out[0] = 1;
    return QMC_OK;
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0;
  CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= QMC_NOALLOC_MAXDEV) return QMC_EINVAL;
  if (!noalloc_addr[dev]) {  // set-up, once per device, with that device current
    unsigned char *ptr = nullptr;
    CUDA_OK(cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), qmc_noalloc_scratch));
    if (!ptr) return QMC_ECUDA;
    noalloc_addr[dev] = ptr;
  }
  unsigned char *ws = noalloc_addr[dev];
  // host side: fixed-size staging (no heap): candidates, their vectors, the partial sums coming back
  static thread_local uint32_t zc[QMC_NCAND * QMC_MAXDIM];
  static thread_local uint64_t cand[QMC_NCAND];
  static thread_local double part[QMC_NCAND * QMC_P2_BLOCKS];
  std::memset(zc, 0, sizeof zc);
  int nc = 0, guard = 0;
  uint64_t state = N;  // the candidate list of korobov_search (R:C13): the same vectors, hence the same answer
  while (nc < QMC_NCAND && guard++ < 100000) {
    const uint64_t a = 2 + splitmix64(state) % (N - 3);
    if (std::gcd(a, N) != 1) continue;
    cand[nc++] = a;
  }
  if (nc == 0) return QMC_EINVAL;
  for (int c = 0; c < nc; ++c) {
    uint64_t v = 1;
    for (int j = 0; j < dim; ++j) {
      zc[(size_t)c * QMC_MAXDIM + j] = (uint32_t)v;
      v = mulmod(v, cand[c], N);
    }
  }
  uint32_t *dz = reinterpret_cast<uint32_t *>(ws);
  double *dp = reinterpret_cast<double *>(ws + QMC_NOALLOC_P2Z_BYTES);
  // the array keeps the last call's contents: everything read below is written first (candidates by the copy, every
  // partial [cand][block] by its block), nothing has to start at zero
  CUDA_OK(cudaMemcpyAsync(dz, zc, sizeof zc, cudaMemcpyHostToDevice, st));
  qmc_p2_kernel<<<dim3(QMC_P2_BLOCKS, nc), 256, 0, st>>>(dz, dp, (uint32_t)N, dim);
  CUDA_OK(cudaGetLastError());
  CUDA_OK(cudaMemcpyAsync(part, dp, (size_t)nc * QMC_P2_BLOCKS * 8, cudaMemcpyDeviceToHost, st));
  CUDA_OK(cudaStreamSynchronize(st));
  int best = 0;
  double bestv = 0.0;
  for (int c = 0; c < nc; ++c) {
    double sum = 0.0;
    for (int b = 0; b < QMC_P2_BLOCKS; ++b) sum += part[(size_t)c * QMC_P2_BLOCKS + b];
    const double p2 = sum / (double)N - 1.0;
    if (c == 0 || p2 < bestv || (p2 == bestv && cand[c] < cand[best])) {
      best = c;
      bestv = p2;
    }
  }
  for (int j = 0; j < dim; ++j) z_out[j] = zc[(size_t)best * QMC_MAXDIM + j];
  return QMC_OK;
}

// ---- embedded lattice sequence (R:C26) --------------------------------------------------------------
// N = 2^k with ODD generating-vector components: the even indices of level k + 1 are the lattice of level k
// ({2i z / 2^(k+1)} = {i z / 2^k}), so raising N re-uses every point already evaluated and only the odd indices are new.
int qmc_embedded_vector(int32_t k_min, int32_t k_max, int32_t dim, void *cuda_stream, void *dev_workspace,
                        size_t dev_workspace_bytes, uint64_t *z_out) {
  if (k_min < 3 || k_max < k_min || k_max > 30 || dim < 1 || dim > QMC_MAXDIM || !z_out) return QMC_EINVAL;
  if (dim == 1) {
    z_out[0] = 1;
    return QMC_OK;
  }
  const size_t p2z = 0, p2p = align256((size_t)QMC_NCAND * QMC_MAXDIM * 4);
  if (!dev_workspace || dev_workspace_bytes < p2p + (size_t)QMC_NCAND * QMC_P2_BLOCKS * 8) return QMC_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  unsigned char *ws = static_cast<unsigned char *>(dev_workspace);
  const uint64_t Nmax = 1ull << k_max;
  // candidates: Korobov form z = (1, a, a^2, ...) mod 2^k_max with odd a from a SplitMix64 stream keyed by (k_max, dim)
  std::vector<uint64_t> cand;
  uint64_t state = ((uint64_t)k_max << 8) | (uint64_t)dim;
  while ((int)cand.size() < QMC_NCAND) cand.push_back((splitmix64(state) % Nmax) | 1ull);
  std::vector<uint64_t> zfull((size_t)QMC_NCAND * QMC_MAXDIM, 0);
  for (int c = 0; c < QMC_NCAND; ++c) {
    uint64_t v = 1;
    for (int j = 0; j < dim; ++j) {
      zfull[(size_t)c * QMC_MAXDIM + j] = v;
      v = mulmod(v, cand[c], Nmax);
    }
  }
  // criterion: the worst level of P_2(z mod 2^k; 2^k) relative to the reference rate (k ln 2)^dim / 4^k
  std::vector<double> worst(QMC_NCAND, 0.0), part((size_t)QMC_NCAND * QMC_P2_BLOCKS);
  std::vector<uint32_t> zc((size_t)QMC_NCAND * QMC_MAXDIM);
  uint32_t *dz = reinterpret_cast<uint32_t *>(ws + p2z);
  double *dp = reinterpret_cast<double *>(ws + p2p);
  for (int k = k_min; k <= k_max; ++k) {
    const uint64_t N = 1ull << k;
    for (size_t i = 0; i < zc.size(); ++i) zc[i] = (uint32_t)(zfull[i] & (N - 1));
    CUDA_OK(cudaMemcpyAsync(dz, zc.data(), zc.size() * 4, cudaMemcpyHostToDevice, st));
    qmc_p2_kernel<<<dim3(QMC_P2_BLOCKS, QMC_NCAND), 256, 0, st>>>(dz, dp, (uint32_t)N, dim);
    CUDA_OK(cudaGetLastError());
    CUDA_OK(cudaMemcpyAsync(part.data(), dp, part.size() * 8, cudaMemcpyDeviceToHost, st));
    CUDA_OK(cudaStreamSynchronize(st));
    const double ref = std::pow((double)k * 0.6931471805599453, (double)dim) / ((double)N * (double)N);
    for (int c = 0; c < QMC_NCAND; ++c) {
      double sum = 0.0;
      for (int b = 0; b < QMC_P2_BLOCKS; ++b) sum += part[(size_t)c * QMC_P2_BLOCKS + b];
      worst[c] = std::max(worst[c], (sum / (double)N - 1.0) / ref);
    }
  }
  int best = 0;
  for (int c = 1; c < QMC_NCAND; ++c)
    if (worst[c] < worst[best] || (worst[c] == worst[best] && cand[c] < cand[best])) best = c;
  for (int j = 0; j < dim; ++j) z_out[j] = zfull[(size_t)best * QMC_MAXDIM + j];
  return QMC_OK;
}

int qmc_integrate_embedded(const qmc_tables *t, int32_t k_min, int32_t k_max, double target_rel_err, int32_t m, uint64_t seed,
                           const uint64_t *z, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                           qmc_result *out, int32_t *k_reached, int64_t *points_evaluated) {
  if (!t || !out || !z || k_min < 3 || k_max < k_min || k_max > 30 || m < 2) return QMC_EINVAL;
  if (out->sector_coeff || out->sector_err || out->shift_sums) return QMC_EINVAL;  // totals only
  const int n = t->n, K = t->kmax - t->kmin + 1;
  for (int j = 0; j < n; ++j)
    if (!(z[j] & 1ull)) return QMC_EINVAL;  // odd components: coprime to every 2^k
  std::vector<double> T((size_t)K * m * 2, 0.0), part((size_t)K * m * 2), coeff((size_t)K * 2), err((size_t)K * 2);
  int64_t npts = 0, counters[4] = {0, 0, 0, 0};
  double kms = 0.0, ems = 0.0;
  int64_t h2d = 0, d2h = 0;
  int launches = 0, kr = k_min;
  for (int k = k_min; k <= k_max; ++k) {
    const uint64_t N = 1ull << k;
    uint64_t zk[QMC_MAXDIM] = {0};
    for (int j = 0; j < n; ++j) zk[j] = z[j] & (N - 1);
    qmc_run run;
    std::memset(&run, 0, sizeof run);
    run.z = zk;
    run.mode = 1;
    run.tables_resident = k > k_min ? 2 : 0;  // the logarithm table and the shift vectors of the first level stay in the workspace
    if (k > k_min) {  // only the odd indices are new
      run.index_begin = 1;
      run.index_step = 2;
      run.index_count = N / 2;
    }
    qmc_result r;
    std::memset(&r, 0, sizeof r);
    r.shift_totals = part.data();
    const int rc = qmc_integrate_ex(t, N, m, seed, &run, cuda_stream, dev_workspace, dev_workspace_bytes, &r);
    if (rc != QMC_OK) return rc;
    // Eq. 18 at level k: (1/N) sum over all indices = half of the level below + the odd part (both already carry their 1/N)
    for (size_t i = 0; i < T.size(); ++i) T[i] = (k > k_min ? 0.5 * T[i] : 0.0) + part[i];
    npts += (int64_t)(k > k_min ? N / 2 : N);
    for (int q = 0; q < 4; ++q) counters[q] += r.counters[q];
    kms += r.kernel_ms; ems += r.eval_kernel_ms; h2d += r.h2d_bytes; d2h += r.d2h_bytes; launches += r.kernel_launches;
    qmc_statistics(T.data(), K, m, coeff.data(), err.data());
    kr = k;
    if (target_rel_err > 0.0) {  // reading C17 on the highest order kept (eps^k_max)
      const double re = coeff[2 * (K - 1)], im = coeff[2 * (K - 1) + 1];
      const double mod = std::sqrt(re * re + im * im);
      if (mod > 0.0 && std::max(err[2 * (K - 1)], err[2 * (K - 1) + 1]) <= target_rel_err * mod) break;
    }
  }
  if (out->coeff) std::memcpy(out->coeff, coeff.data(), coeff.size() * 8);
  if (out->err) std::memcpy(out->err, err.data(), err.size() * 8);
  if (out->shift_totals) std::memcpy(out->shift_totals, T.data(), T.size() * 8);
  for (int q = 0; q < 4; ++q) out->counters[q] = counters[q];
  out->kernel_ms = kms; out->eval_kernel_ms = ems; out->h2d_bytes = h2d; out->d2h_bytes = d2h;
  out->kernel_launches = launches; out->mode_used = 1;
  if (k_reached) *k_reached = kr;
  if (points_evaluated) *points_evaluated = npts;
  return QMC_OK;
}

// ---- per-sector lattice sizes by variance (R:C27) ----------------------------------------------------
int qmc_integrate_allocated(const qmc_tables *t, int32_t k0, int32_t k_max, double target_rel_err, int32_t m, uint64_t seed,
                            const uint64_t *z, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                            qmc_result *out, int32_t *levels_out, int64_t *evals_per_shift) {
  if (!t || !out || !z || k0 < 3 || k_max < k0 || k_max > 30 || m < 2 || !(target_rel_err > 0.0)) return QMC_EINVAL;
  if (out->sector_coeff || out->sector_err || out->shift_sums) return QMC_EINVAL;  // totals only
  const int n = t->n, K = t->kmax - t->kmin + 1, nsec = (int)t->sectors.size();
  for (int j = 0; j < n; ++j)
    if (!(z[j] & 1ull)) return QMC_EINVAL;
  const size_t TS = (size_t)K * m * 2;
  auto zmod = [&](int k, uint64_t *zk) {
    for (int j = 0; j < n; ++j) zk[j] = z[j] & ((1ull << k) - 1);
  };
  int64_t counters[4] = {0, 0, 0, 0}, evals = 0, h2d = 0, d2h = 0;
  double kms = 0.0, ems = 0.0;
  int launches = 0;
  auto book = [&](const qmc_result &r) {
    for (int q = 0; q < 4; ++q) counters[q] += r.counters[q];
    kms += r.kernel_ms; ems += r.eval_kernel_ms; h2d += r.h2d_bytes; d2h += r.d2h_bytes; launches += r.kernel_launches;
  };
  // ---- stage 1: every sector at level k0, per-sector mode: S[sector][order][shift]
  std::vector<double> S((size_t)nsec * TS), T0(TS), coeff((size_t)K * 2), err((size_t)K * 2);
  {
    uint64_t zk[QMC_MAXDIM] = {0};
    zmod(k0, zk);
    qmc_run run;
    std::memset(&run, 0, sizeof run);
    run.z = zk;
    run.mode = 2;
    qmc_result r;
    std::memset(&r, 0, sizeof r);
    r.shift_sums = S.data();
    r.shift_totals = T0.data();
    const int rc = qmc_integrate_ex(t, 1ull << k0, m, seed, &run, cuda_stream, dev_workspace, dev_workspace_bytes, &r);
    if (rc != QMC_OK) return rc;
    book(r);
    evals += (int64_t)nsec << k0;
  }
  qmc_statistics(T0.data(), K, m, coeff.data(), err.data());
  const double c0 = std::hypot(coeff[2 * (K - 1)], coeff[2 * (K - 1) + 1]);
  const double tau = target_rel_err * c0;
  // ---- stage 2: lattice size per sector.  With error ~ e_s N0 / N (the O(1/n) rate the paper quotes) and cost c_s N the
  // cheapest sizes that meet sum_s e_s(N_s)^2 <= tau^2 are  N_s = (a_s / c_s)^(1/3) (sum_r a_r^(1/3) c_r^(2/3))^(1/2) / tau,
  // a_s = e_s^2 N0^2 (Lagrange multiplier); rounded up to a power of two in [2^k0, 2^k_max]
  std::vector<int> lev(nsec, k0);
  {
    std::vector<double> a(nsec, 0.0);
    double sum = 0.0;
    const double N0 = (double)(1ull << k0);
    for (int s = 0; s < nsec; ++s) {
      double e2 = 0.0;
      for (int c = 0; c < 2; ++c) {  // Re and Im separately (R:C15): the larger of the two
        double mean, e;
        mean_err(S.data() + (size_t)s * TS + (size_t)(K - 1) * m * 2 + c, 2, m, &mean, &e);
        e2 = std::max(e2, e * e);
      }
      a[s] = e2 * N0 * N0;
      sum += std::cbrt(a[s]) * std::pow(t->sec_cost[s], 2.0 / 3.0);
    }
    for (int s = 0; s < nsec && tau > 0.0; ++s) {
      const double Ns = std::cbrt(a[s] / t->sec_cost[s]) * std::sqrt(sum) / tau;
      int k = k0;
      while (k < k_max && (double)(1ull << k) < Ns) ++k;
      lev[s] = k;
    }
  }
  // ---- stage 3: one CLASS per lattice size, evaluated in fused mode through qmc_run.sector_mask (a launch then serves the
  // class's sectors of a chunk wherever they sit: the per-point work S1-S3 is shared by all of them); per-class per-shift totals.
  // Kernels without mask support (the generic one): classes = maximal runs of neighbouring sectors of one size instead.
  struct Run { int a, b, k; std::vector<double> T; std::vector<uint8_t> mask; };
  std::vector<Run> runs;
  {
    std::vector<uint8_t> probe(nsec, 0);
    uint64_t zk[QMC_MAXDIM] = {0};
    zmod(k0, zk);
    qmc_run run;
    std::memset(&run, 0, sizeof run);
    run.z = zk;
    run.mode = 1;
    run.sector_mask = probe.data();
    const bool masks = qmc_integrate_async(t, 1ull << k0, m, seed, &run, cuda_stream, dev_workspace, dev_workspace_bytes) == QMC_OK;
    if (masks) {
      for (int k = k0; k <= k_max; ++k) {
        Run R = {0, nsec, k, std::vector<double>(TS, 0.0), std::vector<uint8_t>(nsec, 0)};
        bool any = false;
        for (int s = 0; s < nsec; ++s)
          if (lev[s] == k) R.mask[s] = 1, any = true;
        if (any) runs.push_back(R);
      }
    } else {
      for (int s = 0; s < nsec;) {
        int e = s;
        while (e < nsec && lev[e] == lev[s]) ++e;
        runs.push_back({s, e, lev[s], std::vector<double>(TS, 0.0), std::vector<uint8_t>()});
        s = e;
      }
    }
  }
  std::vector<double> part(TS), T(TS);
  auto integrate_run = [&](Run &R, int k, bool odd_only) -> int {
    uint64_t zk[QMC_MAXDIM] = {0};
    zmod(k, zk);
    qmc_run run;
    std::memset(&run, 0, sizeof run);
    run.z = zk;
    run.mode = 1;
    run.sector_begin = R.a;
    run.sector_end = R.b;
    run.sector_mask = R.mask.empty() ? nullptr : R.mask.data();
    if (odd_only) {
      run.index_begin = 1;
      run.index_step = 2;
      run.index_count = (1ull << k) / 2;
    }
    qmc_result r;
    std::memset(&r, 0, sizeof r);
    r.shift_totals = part.data();
    const int rc = qmc_integrate_ex(t, 1ull << k, m, seed, &run, cuda_stream, dev_workspace, dev_workspace_bytes, &r);
    if (rc != QMC_OK) return rc;
    book(r);
    for (size_t i = 0; i < TS; ++i) R.T[i] = (odd_only ? 0.5 * R.T[i] : 0.0) + part[i];
    int64_t nsel = R.b - R.a;
    if (!R.mask.empty()) {
      nsel = 0;
      for (uint8_t v : R.mask) nsel += v != 0;
    }
    evals += nsel * (int64_t)((1ull << k) / (odd_only ? 2 : 1));
    return QMC_OK;
  };
  for (Run &R : runs) {
    if (R.k == k0) {  // stage 1 already holds these sectors at their level
      for (int s = R.a; s < R.b; ++s)
        if (R.mask.empty() || R.mask[s])
          for (size_t i = 0; i < TS; ++i) R.T[i] += S[(size_t)s * TS + i];
    } else {
      const int rc = integrate_run(R, R.k, false);
      if (rc != QMC_OK) return rc;
    }
  }
  // ---- stage 4: Eqs. 19-20 on the per-shift totals over all runs; while the error is above the target every run climbs one
  // level of the embedded sequence (only its odd indices are new)
  for (;;) {
    std::fill(T.begin(), T.end(), 0.0);
    for (const Run &R : runs)
      for (size_t i = 0; i < TS; ++i) T[i] += R.T[i];
    qmc_statistics(T.data(), K, m, coeff.data(), err.data());
    const double mod = std::hypot(coeff[2 * (K - 1)], coeff[2 * (K - 1) + 1]);
    if (mod > 0.0 && std::max(err[2 * (K - 1)], err[2 * (K - 1) + 1]) <= target_rel_err * mod) break;
    bool any = false;
    for (Run &R : runs)
      if (R.k < k_max) {
        const int rc = integrate_run(R, R.k + 1, true);
        if (rc != QMC_OK) return rc;
        ++R.k;
        any = true;
      }
    if (!any) break;
  }
  if (out->coeff) std::memcpy(out->coeff, coeff.data(), coeff.size() * 8);
  if (out->err) std::memcpy(out->err, err.data(), err.size() * 8);
  if (out->shift_totals) std::memcpy(out->shift_totals, T.data(), TS * 8);
  for (int q = 0; q < 4; ++q) out->counters[q] = counters[q];
  out->kernel_ms = kms; out->eval_kernel_ms = ems; out->h2d_bytes = h2d; out->d2h_bytes = d2h;
  out->kernel_launches = launches; out->mode_used = 1;
  if (levels_out)
    for (const Run &R : runs)
      for (int s = R.a; s < R.b; ++s)
        if (R.mask.empty() || R.mask[s]) levels_out[s] = R.k;
  if (evals_per_shift) *evals_per_shift = evals;
  return QMC_OK;
}

int qmc_fp64_peak(void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes, double *flops_out, double *ms_out) {
  if (!dev_workspace || dev_workspace_bytes < 8 || !flops_out) return QMC_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 0;
  CUDA_OK(cudaGetDevice(&dev));
  CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int iters = 4096, blocks = sms * 8;
  cudaEvent_t e0, e1;
  CUDA_OK(cudaEventCreate(&e0));
  CUDA_OK(cudaEventCreate(&e1));
  double best = 0.0, best_ms = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0, st);
    qmc_dfma_peak_kernel<<<blocks, 256, 0, st>>>(static_cast<double *>(dev_workspace), iters, 1.0000001, 1e-9);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) {
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      cudaGetLastError();
      return QMC_ECUDA;
    }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    double fl = (double)blocks * 256.0 * iters * 64.0 * 2.0 / (ms * 1e-3);
    if (rep > 0 && fl > best) {
      best = fl;
      best_ms = ms;
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *flops_out = best;
  if (ms_out) *ms_out = best_ms;
  return QMC_OK;
}

int qmc_integrate_async(const qmc_tables *tc, uint64_t N, int32_t m, uint64_t seed, const qmc_run *run, void *cuda_stream,
                        void *dev_workspace, size_t dev_workspace_bytes) {
  if (!tc) return QMC_EINVAL;
  qmc_tables *t = const_cast<qmc_tables *>(tc);  // launcher caches (resident image, generating vector, last launch)
  t->last.valid = false;
  const int n = t->n, nsec_all = (int)t->sectors.size();
  if (N < 5 || N >= (1ull << 31) || m < 2) return QMC_EINVAL;  // Eq. 20 needs m >= 2
  qmc_run r;
  std::memset(&r, 0, sizeof r);
  if (run) r = *run;
  const int sb = r.sector_begin, se = r.sector_end > 0 ? r.sector_end : nsec_all;
  if (sb < 0 || se > nsec_all || sb >= se) return QMC_EINVAL;
  const uint64_t ibeg = r.index_begin, istep = r.index_count ? r.index_step : 1, icount = r.index_count ? r.index_count : N;
  if (istep < 1 || ibeg >= N || icount > N) return QMC_EINVAL;
  const bool cplx = t->lambda > 0.0;
  const int mode = r.mode ? r.mode : 1;
  if (mode != 1 && mode != 2 && mode != 3) return QMC_EINVAL;
  const bool persec = mode == 2;
  const bool batch = mode == 3;  // fused within a kinematic point, one row of results per point (qmc_prepare_batch)
  if (batch && (t->row_of_sector.size() != t->sectors.size() || sb != 0 || se != nsec_all || r.sector_mask)) return QMC_EINVAL;

  int devcount = 0;
  if (cudaGetDeviceCount(&devcount) != cudaSuccess || devcount < 1) {
    cudaGetLastError();
    return QMC_ECUDA;  // no CPU fallback
  }
  DevLayout L = layout(t, m);
  if (!dev_workspace || dev_workspace_bytes < L.total) return QMC_ENOMEM;
  unsigned char *ws = static_cast<unsigned char *>(dev_workspace);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const bool image_resident_ws = r.tables_resident >= 1 && t->resident_ws == dev_workspace;
  // resident shift vectors are reused only if they are the ones this call asks for: the same count and -- unless they were
  // passed explicitly by the call that left them -- the same seed (a different seed re-generates and re-uploads them)
  const bool shifts_resident = r.tables_resident >= 2 && image_resident_ws && t->resident_m == m && !r.shifts &&
                               (t->resident_explicit || t->resident_seed == seed);

  // ---- generating vector and shifts ---------------------------------------------------------------------
  uint64_t z[QMC_MAXDIM] = {0};
  if (r.z) {
    for (int j = 0; j < n; ++j) z[j] = r.z[j];
  } else {
    if (t->cached_N != N) {
      int rc = t->lattice == 1 ? qmc_cbc_vector(N, n, t->cached_z, nullptr)
                               : korobov_search(N, n, st, ws, L.p2z, L.p2partial, t->cached_z);
      if (rc != QMC_OK) return rc;
      t->cached_N = N;
    }
    for (int j = 0; j < n; ++j) z[j] = t->cached_z[j];
  }
  for (int j = 0; j < n; ++j)
    if (z[j] == 0 || z[j] >= N || std::gcd(z[j], N) != 1) return QMC_EINVAL;
  if (!shifts_resident) {
    t->shifts_host.resize((size_t)m * n);
    if (r.shifts) {
      std::memcpy(t->shifts_host.data(), r.shifts, t->shifts_host.size() * 8);
      for (double v : t->shifts_host)
        if (!(v >= 0.0 && v < 1.0)) return QMC_EINVAL;
    } else {
      qmc_shifts(seed, m, n, t->shifts_host.data());
    }
  }

  // ---- launch geometry ----------------------------------------------------------------------------------
  int dev = 0, sms = 0, smem_optin = 0;
  CUDA_OK(cudaGetDevice(&dev));
  CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  CUDA_OK(cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  const int nacc = QMC_MAXSING + t->kmax + 1, nc = cplx ? 2 : 1;
  if (!t->ev0) {
    CUDA_OK(cudaEventCreate(reinterpret_cast<cudaEvent_t *>(&t->ev0)));
    CUDA_OK(cudaEventCreate(reinterpret_cast<cudaEvent_t *>(&t->ev1)));
    CUDA_OK(cudaEventCreate(reinterpret_cast<cudaEvent_t *>(&t->evm)));
  }
  size_t h2d = 0;
  int gx = 1, nchunks = 1;
  cudaError_t ce = cudaSuccess;
  double *partial = reinterpret_cast<double *>(ws + L.partial);
  if (r.kernel != 0 && r.kernel != 1) return QMC_EINVAL;
  if (n > 6) return QMC_EUNSUPPORTED;  // every kernel family is instantiated for 1..6 integration variables
  const bool use_v4 = !cplx && !t->tab4.empty() && qmc4_kernel_available(n, t->L, t->kmax) && r.kernel == 0;
  const bool use_v5 = cplx && !t->tab5.empty() && -t->kmin <= QMC3_MAXSING && qmc5_kernel_available(n, t->L, t->kmax) &&
                      r.kernel == 0;
  int eval_launches = 1;
  if ((r.sector_mask || batch) && (persec || !(use_v4 || use_v5))) return QMC_EUNSUPPORTED;  // fused mode of the table-driven kernels only
  std::vector<int> row_of_run;
  const int *rowmap = batch ? t->row_of_sector.data() : nullptr;
  // ---- uploads (skipped when resident).  Versions 4 and 5 carry their tables in the kernel parameters: only the
  // logarithm table lives in the workspace; the version-1 image is uploaded for the generic fallback kernel only.
  const int kind = (use_v4 || use_v5) ? 4 : 1;  // what has to be in the workspace: the logarithm table, or the version-1 image
  if (!(image_resident_ws && t->resident_kind == kind)) {
    if (use_v4 || use_v5) {
      CUDA_OK(cudaMemcpyAsync(ws + L.logtab4, t->logtab4, sizeof t->logtab4, cudaMemcpyHostToDevice, st));
      h2d += sizeof t->logtab4;
    } else {
      h2d += t->image.size() + t->secoff.size() * 4;
      CUDA_OK(cudaMemcpyAsync(ws + L.image, t->image.data(), t->image.size(), cudaMemcpyHostToDevice, st));
      CUDA_OK(cudaMemcpyAsync(ws + L.secoff, t->secoff.data(), t->secoff.size() * 4, cudaMemcpyHostToDevice, st));
    }
    t->resident_ws = dev_workspace;
    t->resident_kind = kind;
    if (!shifts_resident) t->resident_m = 0;
  }
  if (!shifts_resident) {
    h2d += t->shifts_host.size() * 8;
    CUDA_OK(cudaMemcpyAsync(ws + L.shifts, t->shifts_host.data(), t->shifts_host.size() * 8, cudaMemcpyHostToDevice, st));
    t->resident_m = m;
    t->resident_seed = seed;
    t->resident_explicit = r.shifts != nullptr;
  }
  CUDA_OK(cudaMemsetAsync(ws + L.counters, 0, 32, st));

  if (use_v5) {
    int rc = launch_v5(t, L, ws, st, N, m, sb, se, persec, ibeg, istep, icount, z, sms, smem_optin, r.waves, r.streams, r.sector_mask, rowmap, &row_of_run, &gx, &nchunks, &eval_launches, &h2d, &ce);
    if (rc != QMC_OK) return rc;
  } else if (use_v4) {
    int rc = launch_v4(t, L, ws, st, N, m, sb, se, persec, ibeg, istep, icount, z, sms, smem_optin, r.waves, r.streams, r.sector_mask, rowmap, &row_of_run, &gx, &nchunks, &eval_launches, &h2d, &ce);
    if (rc != QMC_OK) return rc;
  } else {
  const size_t fixed_smem = 16 + (((size_t)m * n * 8 + 15) & ~(size_t)15) + (QMC_THREADS / 32) * 8 + (size_t)3 * n * QMC_THREADS * 8;
  const size_t per_sector_acc = persec ? (size_t)nacc * nc * QMC_THREADS * 8 : 0;
  // sectors per chunk: as many as fit the shared-memory budget (tables + per-sector accumulators)
  int spc = 0;
  uint32_t tab_bytes = 0;
  {
    const size_t budget = (size_t)smem_optin - 1024;
    auto fits = [&](int cnt, uint32_t &tb) {
      // worst-case table bytes over all chunks of `cnt` sectors
      uint32_t worst = 0;
      for (int s0 = sb; s0 < se; s0 += cnt) {
        int s1 = std::min(s0 + cnt, se);
        worst = std::max(worst, t->secoff[s1] - t->secoff[s0]);
      }
      tb = worst;
      size_t need = worst + (((size_t)(cnt + 1) * 4 + 15) & ~(size_t)15) + fixed_smem + per_sector_acc * cnt;
      return need <= budget;
    };
    int lo = 1, hi = se - sb;
    uint32_t tb;
    if (!fits(1, tb)) return QMC_ENOMEM;
    if (fits(hi, tb)) {
      spc = hi;
    } else {
      while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (fits(mid, tb)) lo = mid; else hi = mid;
      }
      spc = lo;
    }
    fits(spc, tab_bytes);
  }
  nchunks = (se - sb + spc - 1) / spc;
  const size_t smem = tab_bytes + (((size_t)(spc + 1) * 4 + 15) & ~(size_t)15) + fixed_smem + per_sector_acc * spc;
  int bps = 0;
  const int flavor = !cplx ? (t->has_taylor ? 3 : 0) : (-t->kmin <= 1 ? 2 : 1);  // kmin = -(largest number of singular variables)
  CUDA_OK(qmc_kernel_prepare(n, t->kmax, flavor, smem, &bps));
  if (bps < 1) return QMC_ECUDA;
  gx = std::min<long long>({(long long)sms * bps, (long long)QMC_MAX_BLOCKS, (long long)((icount + QMC_THREADS - 1) / QMC_THREADS)});
  gx = std::max(gx, 1);

  QmcLaunch p;
  std::memset(&p, 0, sizeof p);
  p.image = ws + L.image;
  p.secoff = reinterpret_cast<const uint32_t *>(ws + L.secoff);
  p.shifts = reinterpret_cast<const double *>(ws + L.shifts);
  p.partial = reinterpret_cast<double *>(ws + L.partial);
  p.counters = reinterpret_cast<unsigned long long *>(ws + L.counters);
  p.N = (uint32_t)N;
  p.count = (uint32_t)icount;
  for (int j = 0; j < n; ++j) {
    p.zeff[j] = (uint32_t)mulmod(istep % N, z[j], N);
    p.off[j] = (uint32_t)mulmod(ibeg, z[j], N);
  }
  p.m = m;
  p.kmax = t->kmax;
  p.aU0 = t->aU0; p.aU1 = t->aU1; p.aF0 = t->aF0; p.aF1 = t->aF1;
  p.lambda = t->lambda;
  p.transform = t->transform;
  p.ibp = t->ibp ? 1 : 0;
  qmc_transform_poly(t->transform, p.tc, p.wc);
  p.sec_begin = sb; p.sec_end = se; p.sec_per_chunk = spc;
  p.persec = persec ? 1 : 0;
  p.tab_smem_bytes = (tab_bytes + 15) & ~15u;

  cudaEventRecord(static_cast<cudaEvent_t>(t->ev0), st);
  ce = qmc_kernel_launch(n, t->kmax, flavor, dim3(gx, nchunks), smem, st, p);
  cudaEventRecord(static_cast<cudaEvent_t>(t->evm), st);
  }
  const int rows = persec ? (se - sb) : nchunks;
  const int nrows = persec ? (se - sb) : (batch ? t->n_rows : 0);  // rows of the statistics block: sectors, or kinematic points
  const int nout = (nrows ? nrows : 1) * nacc * nc * m;
  const int K = t->kmax - t->kmin + 1;
  double *dout = reinterpret_cast<double *>(ws + L.out);
  if (ce == cudaSuccess && batch) {
    // runs are in sector order, hence in row order: row r owns the runs [run_begin[r], run_begin[r + 1])
    t->run_begin_host.assign(t->n_rows + 1, 0);
    for (int rr : row_of_run) ++t->run_begin_host[rr + 1];
    for (int q = 0; q < t->n_rows; ++q) t->run_begin_host[q + 1] += t->run_begin_host[q];
    int *drb = reinterpret_cast<int *>(ws + L.runbegin);
    ce = cudaMemcpyAsync(drb, t->run_begin_host.data(), t->run_begin_host.size() * 4, cudaMemcpyHostToDevice, st);
    h2d += t->run_begin_host.size() * 4;
    if (ce == cudaSuccess) {
      qmc_finalize_rows_kernel<<<(nout + 127) / 128, 128, 0, st>>>(partial, dout, drb, nrows, m, gx, nacc * nc, 1.0 / (double)N);
      ce = cudaGetLastError();
    }
  } else if (ce == cudaSuccess) {
    qmc_finalize_kernel<<<(nout + 127) / 128, 128, 0, st>>>(partial, dout, rows, m, gx, nacc * nc, 1.0 / (double)N, persec ? 1 : 0);
    ce = cudaGetLastError();
  }
  if (ce == cudaSuccess) {
    const int nthreads = (nrows + 1) * K * 2;
    qmc_stats_kernel<<<(nthreads + 63) / 64, 64, 0, st>>>(dout, reinterpret_cast<double *>(ws + L.stat), nrows, K, m, nacc, nc,
                                                          t->kmin + QMC_MAXSING);
    ce = cudaGetLastError();
  }
  cudaEventRecord(static_cast<cudaEvent_t>(t->ev1), st);
  if (ce != cudaSuccess) {
    cudaGetLastError();
    t->resident_ws = nullptr;
    return QMC_ECUDA;
  }
  t->last.valid = true;
  t->last.ws = dev_workspace;
  t->last.m = m;
  t->last.mode = mode;
  t->last.nrows = nrows;
  t->last.h2d = h2d;
  t->last.launches = eval_launches + 2;
  return QMC_OK;
}

int qmc_result_fetch(const qmc_tables *tc, void *cuda_stream, void *dev_workspace, size_t dev_workspace_bytes,
                     qmc_result *out) {
  if (!tc || !out) return QMC_EINVAL;
  qmc_tables *t = const_cast<qmc_tables *>(tc);
  if (!t->last.valid || t->last.ws != dev_workspace) return QMC_EINVAL;
  const int m = t->last.m, nrows = t->last.nrows, K = t->kmax - t->kmin + 1;
  DevLayout L = layout(t, m);
  if (dev_workspace_bytes < L.total) return QMC_ENOMEM;
  if ((out->sector_coeff || out->sector_err || out->shift_sums) && t->last.mode != 2 && t->last.mode != 3) return QMC_EINVAL;
  unsigned char *ws = static_cast<unsigned char *>(dev_workspace);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const StatLayout S = stat_layout(nrows, K, m);
  t->stat_host.resize(S.total);
  unsigned long long hc[4] = {0, 0, 0, 0};
  // totals always; the per-sector block only when wanted
  const size_t ncopy = (out->sector_coeff || out->sector_err || out->shift_sums) ? S.total : S.sector_coeff;
  cudaError_t ce = cudaMemcpyAsync(t->stat_host.data(), ws + L.stat, ncopy * 8, cudaMemcpyDeviceToHost, st);
  if (ce == cudaSuccess) ce = cudaMemcpyAsync(hc, ws + L.counters, 32, cudaMemcpyDeviceToHost, st);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
  float ms = 0.f, ms_eval = 0.f;
  if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, static_cast<cudaEvent_t>(t->ev0), static_cast<cudaEvent_t>(t->ev1));
  if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms_eval, static_cast<cudaEvent_t>(t->ev0), static_cast<cudaEvent_t>(t->evm));
  if (ce != cudaSuccess) {
    cudaGetLastError();
    t->resident_ws = nullptr;
    return QMC_ECUDA;
  }
  out->kernel_ms = ms;
  out->eval_kernel_ms = ms_eval;
  out->h2d_bytes = (int64_t)t->last.h2d;
  out->d2h_bytes = (int64_t)(ncopy * 8 + 32);
  out->kernel_launches = t->last.launches;
  out->mode_used = t->last.mode;
  for (int q = 0; q < 4; ++q) out->counters[q] = (int64_t)hc[q];
  const double *h = t->stat_host.data();
  if (out->shift_totals) std::memcpy(out->shift_totals, h + S.totals, (size_t)K * m * 2 * 8);
  if (out->coeff) std::memcpy(out->coeff, h + S.coeff, (size_t)K * 2 * 8);
  if (out->err) std::memcpy(out->err, h + S.err, (size_t)K * 2 * 8);
  if (out->sector_coeff) std::memcpy(out->sector_coeff, h + S.sector_coeff, (size_t)nrows * K * 2 * 8);
  if (out->sector_err) std::memcpy(out->sector_err, h + S.sector_err, (size_t)nrows * K * 2 * 8);
  if (out->shift_sums) std::memcpy(out->shift_sums, h + S.shift_sums, (size_t)nrows * K * m * 2 * 8);
  return QMC_OK;
}

int qmc_result_device_totals(const qmc_tables *t, void *dev_workspace, size_t dev_workspace_bytes, void **totals_out) {
  if (!t || !totals_out || !t->last.valid || t->last.ws != dev_workspace) return QMC_EINVAL;
  DevLayout L = layout(t, t->last.m);
  if (dev_workspace_bytes < L.total) return QMC_ENOMEM;
  const StatLayout S = stat_layout(t->last.nrows, t->kmax - t->kmin + 1, t->last.m);
  *totals_out = static_cast<unsigned char *>(dev_workspace) + L.stat + S.totals * 8;
  return QMC_OK;
}

int qmc_integrate_ex(const qmc_tables *t, uint64_t N, int32_t m, uint64_t seed, const qmc_run *run, void *cuda_stream,
                     void *dev_workspace, size_t dev_workspace_bytes, qmc_result *out) {
  if (!t || !out) return QMC_EINVAL;
  qmc_run r;
  std::memset(&r, 0, sizeof r);
  if (run) r = *run;
  const bool want_persec = out->sector_coeff || out->sector_err || out->shift_sums;
  if (r.mode == 0) r.mode = want_persec ? 2 : 1;
  if (r.mode == 1 && want_persec) return QMC_EINVAL;
  if (r.mode == 3 && !want_persec) return QMC_EINVAL;  // a batch returns its results per kinematic point (the sector_* outputs)
  int rc = qmc_integrate_async(t, N, m, seed, &r, cuda_stream, dev_workspace, dev_workspace_bytes);
  if (rc != QMC_OK) return rc;
  return qmc_result_fetch(t, cuda_stream, dev_workspace, dev_workspace_bytes, out);
}

int qmc_integrate(const qmc_tables *t, uint64_t N, int32_t m, uint64_t seed, void *cuda_stream, void *dev_workspace,
                  size_t dev_workspace_bytes, qmc_result *out) {
  return qmc_integrate_ex(t, N, m, seed, nullptr, cuda_stream, dev_workspace, dev_workspace_bytes, out);
}

int qmc_statistics(const double *shift_totals, int32_t K, int32_t m, double *coeff, double *err) {
  if (!shift_totals || K < 1 || m < 2) return QMC_EINVAL;
  for (int k = 0; k < K; ++k)
    for (int c = 0; c < 2; ++c) {
      double mean, e;
      mean_err(shift_totals + (size_t)k * m * 2 + c, 2, m, &mean, &e);
      if (coeff) coeff[2 * k + c] = mean;
      if (err) err[2 * k + c] = e;
    }
  return QMC_OK;
}

// Laurent series of e^{eg eps gammaE} base^{p0+p1 eps} Gamma(g0 + g1 eps)
int qmc_prefactor_series(double eg, double base, double p0, double p1, int32_t g0, double g1, int32_t n_out,
                         double *series_out, int32_t *lowest_order) {
  if (n_out < 1 || n_out > 16 || g0 < 0 || !series_out || !(base > 0.0)) return QMC_EINVAL;
  static const double zeta[17] = {0, 0, 1.6449340668482264365, 1.2020569031595942854, 1.0823232337111381915,
                                  1.0369277551433699263, 1.0173430619844491397, 1.0083492773819228268,
                                  1.0040773561979443394, 1.0020083928260822144, 1.0009945751278180853,
                                  1.0004941886041194646, 1.0002460865533080483, 1.0001227133475784891,
                                  1.0000612481350587048, 1.0000305882363070205, 1.0000152822594086519};
  const double gammaE = 0.57721566490153286061;
  const int n = n_out;
  // exponent series E(eps) with exp(E) = e^{eg eps gE} base^{p1 eps} Gamma(1 + g1 eps)
  std::vector<double> E(n, 0.0), S(n, 0.0);
  if (n > 1) E[1] = eg * gammaE + p1 * std::log(base) - gammaE * g1;
  double gp = g1;
  for (int k = 2; k < n; ++k) {
    gp *= g1;
    E[k] = ((k & 1) ? -1.0 : 1.0) * zeta[k] * gp / k;
  }
  // S = exp(E): S' = E' S
  S[0] = 1.0;
  for (int k = 1; k < n; ++k) {
    double s = 0.0;
    for (int j = 1; j <= k; ++j) s += j * E[j] * S[k - j];
    S[k] = s / k;
  }
  // Gamma(g0 + x) = Gamma(1 + x) prod_{q=1}^{g0-1} (q + x);  g0 = 0: Gamma(x) = Gamma(1+x)/x
  for (int q = 1; q < g0; ++q) {
    for (int k = n - 1; k >= 1; --k) S[k] = q * S[k] + g1 * S[k - 1];
    S[0] *= q;
  }
  double scale = std::pow(base, p0);
  int lo = 0;
  if (g0 == 0) {
    if (g1 == 0.0) return QMC_EINVAL;
    scale /= g1;
    lo = -1;
  }
  for (int k = 0; k < n; ++k) series_out[k] = S[k] * scale;
  if (lowest_order) *lowest_order = lo;
  return QMC_OK;
}

int qmc_tables_describe(const qmc_tables *t, char *buf, size_t len) {
  if (!t || !buf || len < 1) return QMC_EINVAL;
  std::string o;
  char line[256];
  int ntaylor = 0;
  for (const QmcSector &s : t->sectors) ntaylor += s.ndeep > 0;
  std::snprintf(line, sizeof line, "sectors %d dim %d loops %d orders %d..%d lambda %g generic image %zu B real-path tables %zu B chunks %zu threads %d template %d",
                (int)t->sectors.size(), t->n, t->L, t->kmin, t->kmax, t->lambda, t->image.size(), t->tab4.size() * 4, t->chunks.size(),
                t->threads_real, t->tpl_real);
  o += line;
  if (t->generic_only) {  // propagator powers, sectors with alpha <= -2, integration by parts: the generic kernel only
    std::snprintf(line, sizeof line, " generic kernel only (exponents U^%d%+deps F^%d%+deps, sectors with Taylor terms %d, pole extraction %s)",
                  t->aU0, t->aU1, t->aF0, t->aF1, ntaylor, t->ibp ? "by parts" : "subtraction");
    o += line;
  }
  o += "\n";
  for (size_t c = 0; c < t->chunks.size(); ++c) {
    const Qmc2Chunk &ch = t->chunks[c];
    std::snprintf(line, sizeof line, "chunk %zu: sectors [%d,%d) slots %d (constants %d, products %d) tables %u B records %d (one-factor %d, beyond the dense positions %d) local products %d (max local slots %d) cost %.0f\n", c,
                  ch.sec_begin, ch.sec_end, ch.nslots, ch.nconst, ch.nslots - (2 * t->n + 2 + ch.nconst), ch.tab_words * 16u, ch.nrec,
                  ch.nsingle, ch.noverflow, ch.nlocal, ch.max_local, ch.cost);
    o += line;
  }
  for (size_t c = 0; c < t->chunks3.size(); ++c) {  // complex path
    const Qmc2Chunk &ch = t->chunks3[c];
    std::snprintf(line, sizeof line,
                  "complex chunk %zu: sectors [%d,%d) real slots %d (+%d local) complex slots %d (+%d local) tables %u B (version 5: %u B) cost %.0f\n",
                  c, ch.sec_begin, ch.sec_end, ch.nslots, ch.max_local, t->chunk3_nslots_c[c], t->chunk3_max_local_c[c],
                  t->secend3[ch.sec_end - 1] - t->secoff3[ch.sec_begin],
                  t->secoff5.empty() ? 0u : (t->secoff5[ch.sec_end] - t->secoff5[ch.sec_begin]) * 16u, ch.cost);
    o += line;
  }
  std::snprintf(buf, len, "%s", o.c_str());
  return QMC_OK;
}

const char *qmc_strerror(int status) {
  switch (status) {
    case QMC_OK: return "ok";
    case QMC_EINVAL: return "invalid argument (graph, kinematics, N, z, m or shifts)";
    case QMC_EDEPTH: return "sector decomposition did not terminate within max_depth";
    case QMC_EUNSUPPORTED: return "unsupported: alpha <= -2, beta = 0 on a singular variable, > 4 singular variables, nu != 1 or eps_order > 2";
    case QMC_ECUDA: return "CUDA error or no CUDA device (there is no CPU fallback)";
    case QMC_ENOMEM: return "workspace or buffer too small";
    case QMC_ECONTOUR: return "contour deformation on the wrong side";
    default: return "unknown status";
  }
}

}  // extern "C"
