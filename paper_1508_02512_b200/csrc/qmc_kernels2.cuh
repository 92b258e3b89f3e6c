// Evaluation kernel, version 2 (real / Euclidean path), sm_100a.  Steps S1-S7 of DESIGN.md.
//
// One thread = one lattice point at a time (grid-stride over the points of one shift).  A block works on one WORK
// ITEM = a run of sectors of one chunk, whose tables (chunk slot program + sector blocks, qmc_tables.h "version 2")
// it stages in shared memory with TMA bulk copies.  Per point the thread fills its column of the shared-memory slot
// table (t_j, ln t_j, 1/t_j, 1, then the chunk's product slots); a monomial of U^ or F^ is then ONE 16-byte record
// c * slot[s0] * slot[s1] (two LDS + DMUL + DFMA).  Per sector with s singular variables:
//   1. partial sums of U^, F^ per group (= set of singular variables a monomial depends on), subset sums -> the values
//      at all 2^s corners t^Z of the subtraction (Eqs. 11-12) from one pass over the records;
//   2. per corner: W_Z = G0 U^aU0 F^aF0 with one reciprocal, Lambda_Z = ln(U^aU1 F^aF1) + L0 with ONE table-driven
//      logarithm (exponents are compile-time: they depend only on the dimension and the loop number, Eq. 6);
//   3. the product form of the eps-expanded subtracted integrand, folded one singular variable at a time with series
//      windows of exactly the needed length (see Fold2).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "qmc_kernels.cuh"  // TMA / mbarrier helpers, block_sum
#include "qmc_launch.h"
#include "qmc_tables.h"

namespace qmc2 {

using qmcdev::mbar_expect_tx;
using qmcdev::mbar_init;
using qmcdev::mbar_wait;
using qmcdev::tma_bulk_g2s;

// 1/x to ~1 ulp: MUFU.RCP64H seed + two Newton steps (x normal, which U^ and F^ are: sums of O(1) terms)
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

// ln x, absolute error ~1e-16: x = 2^e * z, z in [0.6875, 1.375), 128 sub-intervals with centre c_i;
// tab[i] = {1/c_i rounded, -ln(that) in extended precision}; r = z/c_i - 1 (one FMA, |r| < 2^-8), degree-6 log1p.
// Arguments that are not positive normal numbers give NaN (the evaluation is then dropped and counted as non-finite).
__constant__ double qmc2_logc[6] = {0.693147180559945309417, -1.0 / 6.0, 0.2, -0.25, 1.0 / 3.0, -0.5};
__device__ __forceinline__ double fast_log(double x, const double2 *__restrict__ tab) {
  const int hi = __double2hiint(x), lo = __double2loint(x);
  const bool ok = (unsigned)(hi - 0x00100000) < 0x7fe00000u;  // positive, normal
  const int tmp = hi - 0x3fe60000;
  const int e = tmp >> 20;
  const double2 T = tab[(tmp >> 13) & 127];
  const double z = __hiloint2double(hi - (tmp & 0xfff00000), lo);
  const double r = fma(z, T.x, -1.0);
  const double y0 = fma((double)e, qmc2_logc[0], T.y);
  double q = fma(r, qmc2_logc[1], qmc2_logc[2]);
  q = fma(r, q, qmc2_logc[3]);
  q = fma(r, q, qmc2_logc[4]);
  q = fma(r, q, qmc2_logc[5]);
  const double v = fma(r * r, q, r) + y0;
  return ok ? v : __longlong_as_double(0x7ff8000000000000ll);
}

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

// sum of n records: c * slot[s0] * slot[s1]
// (sl = this thread's column of the slot table as a byte pointer; record offsets are byte offsets slot * T * 8)
__device__ __forceinline__ double rec_sum(const uint4 *__restrict__ &rec, int n, const unsigned char *__restrict__ sl) {
  double acc = 0.0;
#pragma unroll 1
  for (int i = 0; i < n; ++i) {
    const uint4 r = *rec++;
    const double c = __hiloint2double((int)r.y, (int)r.x);
    acc = fma(c, *reinterpret_cast<const double *>(sl + r.z) * *reinterpret_cast<const double *>(sl + r.w), acc);
  }
  return acc;
}

// per-sector state shared by the fold
template <int NS, int K>
struct Ctx2 {
  double invt[NS > 0 ? NS : 1], invbeta[NS > 0 ? NS : 1];
  double cL[NS > 0 ? NS : 1][K > 1 ? K - 1 : 1];  // (beta_k ln t_k)^p / p!, p = 0 .. K-2
  double W[1 << NS], Lam[1 << NS];                // index X = set of singular variables NOT set to zero
};

// Fold2<LEVEL, ZMASK>: series of sum over Z' subset of {LEVEL..NS-1} of
//   g_{ZMASK u Z'} prod_{j >= LEVEL, j notin Z'} A_j prod_{j in Z'} (B_j - A_j),  A_j = t_j^-1 e^{eps beta_j ln t_j}, B_j = 1/(beta_j eps)
// window: orders -(NS-LEVEL) .. KMAX + popcount(ZMASK)  (what the remaining factors of levels < LEVEL can still use).
template <int NS, int KMAX, int K, int LEVEL, int ZMASK>
struct Fold2 {
  static constexpr int LEN = NS - LEVEL + KMAX + __builtin_popcount(ZMASK) + 1;
  static __device__ __forceinline__ void eval(const Ctx2<NS, K> &c, double (&out)[LEN]) {
    double a[LEN - 1], b[LEN];
    Fold2<NS, KMAX, K, LEVEL + 1, ZMASK>::eval(c, a);
    Fold2<NS, KMAX, K, LEVEL + 1, ZMASK | (1 << LEVEL)>::eval(c, b);
    const double it = c.invt[LEVEL], ib = c.invbeta[LEVEL];
    double d[LEN - 1];
#pragma unroll
    for (int i = 0; i < LEN - 1; ++i) d[i] = it * (a[i] - b[i]);
    out[0] = ib * b[0];
#pragma unroll
    for (int i = 1; i < LEN; ++i) {
      double s = fma(ib, b[i], d[i - 1]);
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
    for (int p = 1; p < LEN; ++p) out[p] = out[p - 1] * c.Lam[X] * (1.0 / p);
  }
};

// one sector at one point: out[i] = coefficient of eps^(i - NS) of the subtracted integrand (without the weight w)
template <int NDIM, int L, int NS, int KMAX>
__device__ __forceinline__ void sector2(const Qmc2SectorHdr *__restrict__ h, double *__restrict__ sl, int local0,
                                        const double2 *__restrict__ logtab, double (&out)[KMAX + NS + 1]) {
  constexpr int K = KMAX + NS + 1, NC = 1 << NS, FULL = NC - 1;
  typedef Expo<NDIM, L> E;
  const int nlocal = h->nlocal;
  {  // sector-local products: slot[local0 + i] = slot[a] * slot[b]
    const uint32_t *lp = reinterpret_cast<const uint32_t *>(h + 1);
#pragma unroll 1
    for (int i = 0; i < nlocal; ++i) {
      const uint32_t pw = lp[i];
      sl[local0 + i * QMC2_THREADS] = sl[pw & 0xffffu] * sl[pw >> 16];
    }
  }
  const uint4 *rec = reinterpret_cast<const uint4 *>(reinterpret_cast<const unsigned char *>(h + 1) + ((nlocal * 4 + 15) & ~15));
  const unsigned char *slb = reinterpret_cast<const unsigned char *>(sl);
  const double G0 = rec_sum(rec, 1, slb);
  const double L0 = rec_sum(rec, h->nL0, slb);
  Ctx2<NS, K> c;
  {
    // group partial sums (records are sorted by group), then subset sums: P[X] = value with the singular variables
    // outside X set to zero
    double PU[NC], PF[NC];
    const uint4 cu = *reinterpret_cast<const uint4 *>(h->cntU), cf = *reinterpret_cast<const uint4 *>(h->cntF);
    const unsigned cuw[4] = {cu.x, cu.y, cu.z, cu.w}, cfw[4] = {cf.x, cf.y, cf.z, cf.w};
#pragma unroll
    for (int g = 0; g < NC; ++g) PU[g] = rec_sum(rec, (cuw[g >> 2] >> (8 * (g & 3))) & 255u, slb);
#pragma unroll
    for (int g = 0; g < NC; ++g) PF[g] = rec_sum(rec, (cfw[g >> 2] >> (8 * (g & 3))) & 255u, slb);
#pragma unroll
    for (int b = 0; b < NS; ++b)
#pragma unroll
      for (int X = 0; X < NC; ++X)
        if (X >> b & 1) {
          PU[X] += PU[X ^ (1 << b)];
          PF[X] += PF[X ^ (1 << b)];
        }
    // corners: W = G0 U^aU0 F^aF0 (one reciprocal), Lambda = ln(U^aU1 F^aF1) + L0 (one logarithm)
#pragma unroll
    for (int X = 0; X < NC; ++X) {
      const double U = PU[X], F = PF[X];
      const double rF = fast_rcp(F);
      double W = G0;
      if (E::aU0 > 0) W *= ipow_c<(E::aU0 > 0 ? E::aU0 : 0)>(U);
      if (E::aU0 < 0) W *= ipow_c<(E::aU0 < 0 ? -E::aU0 : 0)>(fast_rcp(U));
      if (E::aF0 > 0) W *= ipow_c<(E::aF0 > 0 ? E::aF0 : 0)>(F);
      if (E::aF0 < 0) W *= ipow_c<(E::aF0 < 0 ? -E::aF0 : 0)>(rF);
      c.W[X] = W;
      if (KMAX > 0 || X != FULL) c.Lam[X] = fast_log(ipow_c<E::aU1>(U) * ipow_c<-E::aF1>(rF), logtab) + L0;
    }
  }
#pragma unroll
  for (int k = 0; k < NS; ++k) {
    c.invt[k] = sl[h->sing_inv[k]];
    c.invbeta[k] = h->invbeta[k];
    const double Lk = h->beta[k] * sl[h->sing_ln[k]];
    c.cL[k][0] = 1.0;
#pragma unroll
    for (int q = 1; q < K - 1; ++q) c.cL[k][q] = c.cL[k][q - 1] * Lk * (1.0 / q);
  }
  Fold2<NS, KMAX, K, 0, 0>::eval(c, out);
}

__device__ __forceinline__ bool finite_hi(double v) { return (__double2hiint(v) & 0x7ff00000) != 0x7ff00000; }

}  // namespace qmc2

#ifndef QMC2_MIN_BLOCKS
#define QMC2_MIN_BLOCKS 2
#endif

// partial layout: fused  : [run of sectors][shift][slice][NACC]
//                 persec : [sector row][shift][slice][NACC]        (NACC = QMC_MAXSING + KMAX + 1, index a <-> order a - QMC_MAXSING)
template <int NDIM, int L, int KMAX>
__global__ void __launch_bounds__(QMC2_THREADS, QMC2_MIN_BLOCKS) qmc2_eval_kernel(const Qmc2Launch p) {
  using namespace qmc2;
  constexpr int NACC = QMC_MAXSING + KMAX + 1;
  constexpr int SMAX = NDIM < QMC_MAXSING ? NDIM : QMC_MAXSING;
  constexpr int T = QMC2_THREADS;

  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x;
  const Qmc2Work wk = p.work[blockIdx.x];

  // shared memory carve-up (all offsets multiples of 16)
  unsigned char *sprog = smem;
  unsigned char *stab = smem + p.sm_prog_cap;
  size_t o = (size_t)p.sm_prog_cap + p.sm_sec_cap;
  uint32_t *soff = reinterpret_cast<uint32_t *>(smem + o);
  o += (((size_t)(p.max_nsec + 1) * 4) + 15) & ~(size_t)15;
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem + o);
  o += 16;
  double *shf = reinterpret_cast<double *>(smem + o);
  o += (((size_t)p.m * NDIM * 8) + 15) & ~(size_t)15;
  double *scratch = reinterpret_cast<double *>(smem + o);
  o += (T / 32) * 8;
  double2 *logtab = reinterpret_cast<double2 *>(smem + o);
  o += 128 * 16;
  double *slots = reinterpret_cast<double *>(smem + o);
  o += (size_t)p.max_nslots * T * 8;
  double *sacc = reinterpret_cast<double *>(smem + o);  // persec: [nsec][NACC][T]
  double *sl = slots + tid;

  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    mbar_expect_tx(bar, wk.prog_bytes + wk.sec_bytes);
    tma_bulk_g2s(sprog, p.image2 + wk.prog_off, wk.prog_bytes, bar);
    tma_bulk_g2s(stab, p.image2 + wk.sec_off, wk.sec_bytes, bar);
  }
  for (int i = tid; i <= wk.nsec; i += T) soff[i] = p.secoff2[wk.s0 + i] - wk.sec_off;
  for (int i = tid; i < p.m * NDIM; i += T) shf[i] = p.shifts[i];
  for (int i = tid; i < 256; i += T) reinterpret_cast<double *>(logtab)[i] = p.logtab[i];
  sl[3 * NDIM * T] = 1.0;  // the constant slot
  mbar_wait(bar, 0);
  __syncthreads();

  const Qmc2ChunkHdr *ch = reinterpret_cast<const Qmc2ChunkHdr *>(sprog);
  const uint32_t *prog = reinterpret_cast<const uint32_t *>(sprog + sizeof(Qmc2ChunkHdr));
  const int nprog = ch->nprog, first_prod = ch->first_prod, local0 = ch->nslots * T;

  const uint32_t N = p.N;
  const double dN = (double)N;
  const uint32_t stride = (uint32_t)wk.nslices * T;
  uint32_t dz[NDIM];
#pragma unroll
  for (int j = 0; j < NDIM; ++j) dz[j] = (uint32_t)(((uint64_t)stride * p.zeff[j]) % N);

  unsigned cntNonFinite = 0, cntBoundary = 0;

  for (int kap = 0; kap < p.m; ++kap) {
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;
    if (p.persec)
      for (int i = 0; i < wk.nsec * NACC; ++i) sacc[(size_t)i * T + tid] = 0.0;

    uint32_t cidx = (uint32_t)wk.slice * T + tid;
    uint32_t r[NDIM];
#pragma unroll
    for (int j = 0; j < NDIM; ++j) r[j] = (uint32_t)((p.off[j] + (uint64_t)cidx * p.zeff[j]) % N);

    for (; cidx < p.count; cidx += stride) {
      // S1-S3: lattice point (Eq. 17), shift + wrap (Eq. 18), periodising transform (Eq. 21), per-point slot table
      double w = 1.0;
      bool inside = true;
#pragma unroll
      for (int j = 0; j < NDIM; ++j) {
        double u = (double)r[j] / dN;
        double y = u + shf[kap * NDIM + j];
        if (y >= 1.0) y -= 1.0;
        double tj;
        if (p.transform == 0) {
          tj = y * y * (3.0 - 2.0 * y);
          w *= 6.0 * y * (1.0 - y);
        } else {
          tj = 1.0 - fabs(2.0 * y - 1.0);
        }
        if (!(y > 0.0) || !(tj > 0.0)) inside = false;
        sl[j * T] = tj;
        sl[(NDIM + j) * T] = fast_log(tj, logtab);   // t >= 3.7e-32 for y >= 2^-53: always a normal number
        sl[(2 * NDIM + j) * T] = fast_rcp(tj);
        uint32_t rn = r[j] + dz[j];
        r[j] = rn >= N ? rn - N : rn;
      }
      if (!inside) {
        if (wk.count_boundary) ++cntBoundary;
        continue;
      }
      for (int i = 0; i < nprog; ++i) {
        const uint32_t pw = prog[i];
        sl[(first_prod + i) * T] = sl[pw & 0xffffu] * sl[pw >> 16];
      }
      // S4-S6: all sectors of the work item at this point
      for (int si = 0; si < wk.nsec; ++si) {
        const Qmc2SectorHdr *h = reinterpret_cast<const Qmc2SectorHdr *>(stab + soff[si]);
#define QMC2_CASE(NS_)                                                                                       \
  case NS_: {                                                                                                \
    if (NS_ <= SMAX) {                                                                                       \
      constexpr int NSC = NS_ <= SMAX ? NS_ : 0, KK = KMAX + NSC + 1;                                        \
      double res[KK];                                                                                        \
      sector2<NDIM, L, NSC, KMAX>(h, sl, local0, logtab, res);                                                       \
      bool fin = true;                                                                                       \
      _Pragma("unroll") for (int i = 0; i < KK; ++i) fin = fin && finite_hi(res[i]);                         \
      if (!fin) {                                                                                            \
        ++cntNonFinite;                                                                                      \
      } else if (!p.persec) {                                                                                \
        _Pragma("unroll") for (int i = 0; i < KK; ++i) acc[QMC_MAXSING - NSC + i] = fma(w, res[i], acc[QMC_MAXSING - NSC + i]); \
      } else {                                                                                               \
        double *sa = sacc + ((size_t)si * NACC + (QMC_MAXSING - NSC)) * T + tid;                             \
        _Pragma("unroll") for (int i = 0; i < KK; ++i) sa[(size_t)i * T] += w * res[i];                      \
      }                                                                                                      \
    }                                                                                                        \
  } break;
        switch (h->nsing) {
          QMC2_CASE(0)
          QMC2_CASE(1)
          QMC2_CASE(2)
          QMC2_CASE(3)
          QMC2_CASE(4)
          default:
            break;
        }
#undef QMC2_CASE
      }
    }

    // S7: block reduction -> one partial per (work item | sector, shift, block)
    if (!p.persec) {
      double *dst = p.partial + (((size_t)wk.out_row * p.m + kap) * p.max_slices + wk.slice) * NACC;
#pragma unroll
      for (int a = 0; a < NACC; ++a) {
        double sr = qmcdev::block_sum(acc[a], scratch);
        if (tid == 0) dst[a] = sr;
      }
    } else {
      for (int si = 0; si < wk.nsec; ++si) {
        double *dst = p.partial + (((size_t)(wk.out_row + si) * p.m + kap) * p.max_slices + wk.slice) * NACC;
        for (int a = 0; a < NACC; ++a) {
          double v = qmcdev::block_sum(sacc[((size_t)si * NACC + a) * T + tid], scratch);
          if (tid == 0) dst[a] = v;
        }
      }
    }
  }

  unsigned c2[2] = {cntNonFinite, cntBoundary};
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    unsigned v = c2[q];
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) v += __shfl_down_sync(0xffffffffu, v, o2);
    if ((tid & 31) == 0 && v) atomicAdd(p.counters + 2 + q, (unsigned long long)v);
  }
}
