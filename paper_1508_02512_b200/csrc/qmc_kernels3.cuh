// Evaluation kernel, version 3 (complex path: physical region, contour deformation), sm_100a.  Steps S1-S7 of DESIGN.md.
//
// Same organisation as version 2 (qmc_kernels2.cuh): one thread = one lattice point, a block = one slice of the points
// of a run of sectors of one chunk, tables staged by TMA, monomials as 16-byte records over per-thread slot tables in
// shared memory.  Per corner Z of a sector (real point tau = t with the variables of Z set to 0):
//   S4  F^_i(tau), F^_ik(tau) from the record lists of the derivative polynomials (groups meeting Z are skipped);
//       rho_i = 1 - i lambda (1 - tau_i) F^_i,  z_i = tau_i rho_i,
//       J_ik = delta_ik [1 - i lambda (1 - 2 tau_i) F^_i] - i lambda tau_i (1 - tau_i) F^_ik   (Eq. 14; R:C12),
//       det J by LU with row pivoting;
//   S5  the complex slot table is refilled with z_j and the chunk's products, U^(z), F^(z) are sums of complex records;
//       G_Z = G0 det J prod_{j notin Z} rho_j^alpha_j U^aU0 F^aF0,
//       Lambda_Z = aU1 ln U + aF1 ln F + sum_j beta_j ln rho_j + L0   (principal logs; -i pi on the negative real axis, R:C11);
//   S6  product form folded one singular variable at a time with exact series windows (as Fold2, complex).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "qmc_kernels2.cuh"

namespace qmc3 {

using qmcdev::cd;
using qmcdev::cinv;
using qmcdev::cnorm2;
using qmcdev::mbar_expect_tx;
using qmcdev::mbar_init;
using qmcdev::mbar_wait;
using qmcdev::tma_bulk_g2s;
using qmc2::Expo;
using qmc2::fast_log;
using qmc2::fast_rcp;

// Shared-memory accesses by 32-bit shared address: corner3 is an out-of-line function, and through generic pointers
// kept in a struct the compiler emits generic loads with 64-bit address arithmetic (measured: 10 % LD, 13 % R2UR).
__device__ __forceinline__ uint32_t saddr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ double lds_f64(uint32_t a) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ double2 lds_f64x2(uint32_t a) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
  return v;
}
__device__ __forceinline__ uint4 lds_u32x4(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t lds_u8(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts_f64x2(uint32_t a, double x, double y) {
  asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(x), "d"(y) : "memory");
}
// qmc2::fast_log with the table given by shared address
__device__ __forceinline__ double fast_log_s(double x, uint32_t tab) {
  const int hi = __double2hiint(x), lo = __double2loint(x);
  const bool ok = (unsigned)(hi - 0x00100000) < 0x7fe00000u;
  const int tmp = hi - 0x3fe60000;
  const int e = tmp >> 20;
  const double2 T = lds_f64x2(tab + (((unsigned)tmp >> 13) & 127u) * 16u);
  const double z = __hiloint2double(hi - (tmp & 0xfff00000), lo);
  const double r = fma(z, T.x, -1.0);
  const double y0 = fma((double)e, qmc2::qmc2_logc[0], T.y);
  double q = fma(r, qmc2::qmc2_logc[1], qmc2::qmc2_logc[2]);
  q = fma(r, q, qmc2::qmc2_logc[3]);
  q = fma(r, q, qmc2::qmc2_logc[4]);
  q = fma(r, q, qmc2::qmc2_logc[5]);
  const double v = fma(r * r, q, r) + y0;
  return ok ? v : __longlong_as_double(0x7ff8000000000000ll);
}

static __device__ __noinline__ double atan2_lib(double y, double x) { return atan2(y, x); }
// principal log; a negative real argument carries the -i0 of F -> F - i0: arg = -pi (R:C11)
__device__ __forceinline__ cd clog3(cd a, uint32_t logtab) {
  const double arg = (a.im == 0.0 && a.re < 0.0) ? -3.14159265358979323846 : atan2_lib(a.im, a.re);
  return cd{0.5 * fast_log_s(cnorm2(a), logtab), arg};
}
template <int E>
__device__ __forceinline__ cd cpow_c(cd x) {  // x^E, E >= 0 compile time
  if (E == 0) return cd{1.0, 0.0};
  if (E == 1) return x;
  cd h = cpow_c<E / 2>(x);
  h = h * h;
  return (E & 1) ? h * x : h;
}

// sum of n real records c * slot[s0] * slot[s1] (rec, sl: shared addresses of the records and of the thread's column)
__device__ __forceinline__ double rsum(uint32_t &rec, int n, uint32_t sl) {
  double acc = 0.0;
#pragma unroll 1
  for (int i = 0; i < n; ++i) {
    const uint4 r = lds_u32x4(rec);
    rec += 16;
    acc = fma(__hiloint2double((int)r.y, (int)r.x), lds_f64(sl + r.z) * lds_f64(sl + r.w), acc);
  }
  return acc;
}
// sum of n complex records (16 bytes per column entry)
__device__ __forceinline__ cd csum(uint32_t &rec, int n, uint32_t sl) {
  cd acc = cd{0.0, 0.0};
#pragma unroll 1
  for (int i = 0; i < n; ++i) {
    const uint4 r = lds_u32x4(rec);
    rec += 16;
    const double c = __hiloint2double((int)r.y, (int)r.x);
    const double2 a = lds_f64x2(sl + r.z), b = lds_f64x2(sl + r.w);
    acc.re = fma(c, a.x * b.x - a.y * b.y, acc.re);
    acc.im = fma(c, a.x * b.y + a.y * b.x, acc.im);
  }
  return acc;
}

template <int NDIM, int NS, int K>
struct Ctx3 {
  double invt[NS > 0 ? NS : 1], invbeta[NS > 0 ? NS : 1];
  double cL[NS > 0 ? NS : 1][K > 1 ? K - 1 : 1];
  // everything below: 32-bit shared-memory addresses
  uint32_t counts;                  // u8 [npoly][1 << NS]
  uint32_t rec_deriv, rec_c;        // first record of F_1, first complex record
  uint32_t locprog_c, prog_c;       // sector-local / chunk complex products {u16 a, u16 b}
  int nprog_c, first_prod_c, local0_c, nlocal_c;
  uint32_t slr;                     // this thread's real column; slot s at slr + s * T * 8
  uint32_t slc;                     // this thread's complex column; slot s at slc + s * T * 16
  uint32_t logtab;
  unsigned zvar[NS > 0 ? NS : 1];   // variable index of singular position k
  int alpha[NDIM], beta[NDIM];
  double G0, L0, lambda;
  unsigned cntImF, cntReU;
};

// W_Z and Lambda_Z of one corner (Z = bit mask over the singular positions)
template <int NDIM, int L, int NS, int K>
__device__ __noinline__ void corner3(Ctx3<NDIM, NS, K> &c, const int Z, cd &Wout, cd &Lout) {
  constexpr int NG = 1 << NS, T = QMC3_THREADS, NDERIV = NDIM + NDIM * (NDIM + 1) / 2;
  typedef Expo<NDIM, L> E;
  unsigned zv = 0;  // variables set to zero
#pragma unroll
  for (int k = 0; k < NS; ++k)
    if (Z >> k & 1) zv |= 1u << c.zvar[k];
  // ---- S4: gradient and Hessian of F^ at tau -------------------------------------------------------------------
  double grad[NDIM], hess[NDIM][NDIM];
  {
    uint32_t rec = c.rec_deriv, cnt = c.counts;
#pragma unroll
    for (int i = 0; i < NDIM; ++i) {
      double s = 0.0;
#pragma unroll
      for (int g = 0; g < NG; ++g) {
        const int n = (int)lds_u8(cnt++);
        if (g & Z) rec += 16 * n; else s += rsum(rec, n, c.slr);
      }
      grad[i] = s;
    }
#pragma unroll
    for (int i = 0; i < NDIM; ++i)
#pragma unroll
      for (int k = i; k < NDIM; ++k) {
        double s = 0.0;
#pragma unroll
        for (int g = 0; g < NG; ++g) {
          const int n = (int)lds_u8(cnt++);
          if (g & Z) rec += 16 * n; else s += rsum(rec, n, c.slr);
        }
        hess[i][k] = s;
      }
  }
  // rho_i, z_i, J = 1 + i B
  cd rho[NDIM], J[NDIM][NDIM];
#pragma unroll
  for (int i = 0; i < NDIM; ++i) {
    const bool inZ = (zv >> i & 1u) != 0;
    const double tau = inZ ? 0.0 : lds_f64(c.slr + i * T * 8);
    rho[i] = cd{1.0, -c.lambda * (1.0 - tau) * grad[i]};
    sts_f64x2(c.slc + i * T * 16, tau, tau * rho[i].im);  // z_i = tau rho_i
#pragma unroll
    for (int k = 0; k < NDIM; ++k) {
      const bool kinZ = (zv >> k & 1u) != 0;
      if (inZ || kinZ) {
        J[i][k] = cd{(i == k) ? 1.0 : 0.0, 0.0};  // row / column of a Z variable: its rho cancels rho^-1 (alpha = -1)
      } else {
        const double hik = (k >= i) ? hess[i][k] : hess[k][i];
        double b = -c.lambda * tau * (1.0 - tau) * hik;
        if (i == k) b += -c.lambda * (1.0 - 2.0 * tau) * grad[i];
        J[i][k] = cd{(i == k) ? 1.0 : 0.0, b};
      }
    }
  }
  cd det = cd{1.0, 0.0};
#pragma unroll
  for (int col = 0; col < NDIM; ++col) {
#pragma unroll
    for (int r = col + 1; r < NDIM; ++r) {
      if (cnorm2(J[r][col]) > cnorm2(J[col][col])) {
#pragma unroll
        for (int k = col; k < NDIM; ++k) {
          cd tmp = J[r][k];
          J[r][k] = J[col][k];
          J[col][k] = tmp;
        }
        det = cd{-det.re, -det.im};
      }
    }
    det = det * J[col][col];
    if (col + 1 < NDIM) {
      const cd ip = cinv(J[col][col]);
#pragma unroll
      for (int r = col + 1; r < NDIM; ++r) {
        const cd f = J[r][col] * ip;
#pragma unroll
        for (int k = col + 1; k < NDIM; ++k) J[r][k] = J[r][k] - f * J[col][k];
      }
    }
  }
  // ---- S5: complex slot table over z, U^(z), F^(z) -----------------------------------------------------------------
#pragma unroll 1
  for (int i = 0; i < c.nprog_c; ++i) {
    const uint32_t w = lds_u32(c.prog_c + 4 * i);
    const double2 a = lds_f64x2(c.slc + (w & 0xffffu) * (T * 16)), b = lds_f64x2(c.slc + (w >> 16) * (T * 16));
    sts_f64x2(c.slc + (c.first_prod_c + i) * (T * 16), a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
  }
#pragma unroll 1
  for (int i = 0; i < c.nlocal_c; ++i) {
    const uint32_t w = lds_u32(c.locprog_c + 4 * i);
    const double2 a = lds_f64x2(c.slc + (w & 0xffffu) * (T * 16)), b = lds_f64x2(c.slc + (w >> 16) * (T * 16));
    sts_f64x2(c.slc + (c.local0_c + i) * (T * 16), a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
  }
  cd Uv = cd{0.0, 0.0}, Fv = cd{0.0, 0.0};
  {
    uint32_t rec = c.rec_c, cnt = c.counts + NDERIV * NG;
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      const int n = (int)lds_u8(cnt++);
      if (g & Z) rec += 16 * n; else Uv = Uv + csum(rec, n, c.slc);
    }
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      const int n = (int)lds_u8(cnt++);
      if (g & Z) rec += 16 * n; else Fv = Fv + csum(rec, n, c.slc);
    }
  }
  if (Fv.im > 0.0) ++c.cntImF;
  if (!(Uv.re > 0.0)) ++c.cntReU;
  // G_Z = G0 det J prod_{j notin Z} rho_j^alpha_j U^aU0 F^aF0 ;  Lambda_Z = aU1 ln U + aF1 ln F + sum_j beta_j ln rho_j + L0
  cd num = cd{c.G0 * det.re, c.G0 * det.im}, den = cd{1.0, 0.0};
  cd Lam = (double)E::aU1 * clog3(Uv, c.logtab) + (double)E::aF1 * clog3(Fv, c.logtab);
  Lam.re += c.L0;
#pragma unroll
  for (int j = 0; j < NDIM; ++j) {
    const bool inZ = (zv >> j & 1u) != 0;
    const int a = c.alpha[j], b = c.beta[j];
    if (!inZ) {
      if (a < 0) den = den * rho[j];
      for (int q = 0; q < a; ++q) num = num * rho[j];
    }
    if (b) Lam = Lam + (double)b * clog3(rho[j], c.logtab);
  }
  if (E::aU0 > 0) num = num * cpow_c<(E::aU0 > 0 ? E::aU0 : 0)>(Uv);
  if (E::aU0 < 0) den = den * cpow_c<(E::aU0 < 0 ? -E::aU0 : 0)>(Uv);
  if (E::aF0 > 0) num = num * cpow_c<(E::aF0 > 0 ? E::aF0 : 0)>(Fv);
  if (E::aF0 < 0) den = den * cpow_c<(E::aF0 < 0 ? -E::aF0 : 0)>(Fv);
  Wout = num * cinv(den);
  Lout = Lam;
}

// fold of the singular variables with exact series windows (see qmc2::Fold2), complex
template <int NDIM, int L, int NS, int KMAX, int K, int LEVEL, int ZMASK>
struct Fold3 {
  static constexpr int LEN = NS - LEVEL + KMAX + __builtin_popcount(ZMASK) + 1;
  static __device__ __forceinline__ void eval(Ctx3<NDIM, NS, K> &c, cd (&out)[LEN]) {
    cd a[LEN - 1], b[LEN];
    Fold3<NDIM, L, NS, KMAX, K, LEVEL + 1, ZMASK>::eval(c, a);
    Fold3<NDIM, L, NS, KMAX, K, LEVEL + 1, ZMASK | (1 << LEVEL)>::eval(c, b);
    const double it = c.invt[LEVEL], ib = c.invbeta[LEVEL];
    cd d[LEN - 1];
#pragma unroll
    for (int i = 0; i < LEN - 1; ++i) d[i] = it * (a[i] - b[i]);
    out[0] = ib * b[0];
#pragma unroll
    for (int i = 1; i < LEN; ++i) {
      cd s = ib * b[i] + d[i - 1];
#pragma unroll
      for (int p = 1; p < i; ++p) s = s + c.cL[LEVEL][p] * d[i - 1 - p];
      out[i] = s;
    }
  }
};
template <int NDIM, int L, int NS, int KMAX, int K, int ZMASK>
struct Fold3<NDIM, L, NS, KMAX, K, NS, ZMASK> {
  static constexpr int LEN = KMAX + __builtin_popcount(ZMASK) + 1;
  static __device__ __forceinline__ void eval(Ctx3<NDIM, NS, K> &c, cd (&out)[LEN]) {
    cd W, Lam;
    corner3<NDIM, L, NS, K>(c, ZMASK, W, Lam);
    out[0] = W;
#pragma unroll
    for (int p = 1; p < LEN; ++p) out[p] = (1.0 / p) * (out[p - 1] * Lam);
  }
};

// one sector at one point: out[i] = coefficient of eps^(i - NS)
template <int NDIM, int L, int NS, int KMAX>
__device__ __forceinline__ void sector3(const Qmc3SectorHdr *__restrict__ h, double *__restrict__ slr_d, double2 *__restrict__ slc,
                                        int local0_r, const uint32_t *prog_c, int nprog_c, int first_prod_c, int local0_c,
                                        double lambda, const double2 *__restrict__ logtab, cd (&out)[KMAX + NS + 1],
                                        unsigned &cntImF, unsigned &cntReU) {
  constexpr int K = KMAX + NS + 1, NG = 1 << NS, T = QMC3_THREADS, NPOLY = NDIM + NDIM * (NDIM + 1) / 2 + 2;
  Ctx3<NDIM, NS, K> c;
  const unsigned char *p = reinterpret_cast<const unsigned char *>(h + 1);
  c.counts = saddr(p);
  p += (NPOLY * NG + 15) & ~15;
  const uint32_t *locprog_r = reinterpret_cast<const uint32_t *>(p);
  p += (h->nlocal_r * 4 + 15) & ~15;
  c.locprog_c = saddr(p);
  p += (h->nlocal_c * 4 + 15) & ~15;
  uint32_t rec = saddr(p);
  c.rec_c = rec + 16u * h->nrec_r;
  c.prog_c = saddr(prog_c); c.nprog_c = nprog_c; c.first_prod_c = first_prod_c; c.local0_c = local0_c;
  c.nlocal_c = h->nlocal_c;
  c.slr = saddr(slr_d);
  c.slc = saddr(slc);
  c.logtab = saddr(logtab);
  c.lambda = lambda;
  c.cntImF = 0; c.cntReU = 0;
#pragma unroll
  for (int j = 0; j < NDIM; ++j) {
    c.alpha[j] = h->alpha[j];
    c.beta[j] = h->beta[j];
  }
  {  // sector-local real products
    const int nl = h->nlocal_r;
#pragma unroll 1
    for (int i = 0; i < nl; ++i) {
      const uint32_t w = locprog_r[i];
      slr_d[(local0_r + i) * T] = slr_d[(w & 0xffffu) * T] * slr_d[(w >> 16) * T];
    }
  }
  c.G0 = rsum(rec, 1, c.slr);
  c.L0 = rsum(rec, h->nL0, c.slr);
  c.rec_deriv = rec;
#pragma unroll
  for (int k = 0; k < NS; ++k) {
    const int j = h->sing_var[k];
    c.zvar[k] = j;
    c.invt[k] = slr_d[(2 * NDIM + j) * T];
    c.invbeta[k] = h->invbeta[k];
    const double Lk = h->betas[k] * slr_d[(NDIM + j) * T];
    c.cL[k][0] = 1.0;
#pragma unroll
    for (int q = 1; q < K - 1; ++q) c.cL[k][q] = c.cL[k][q - 1] * Lk * (1.0 / q);
  }
  Fold3<NDIM, L, NS, KMAX, K, 0, 0>::eval(c, out);
  cntImF += c.cntImF;
  cntReU += c.cntReU;
}

__device__ __forceinline__ bool finite_hi(cd v) {
  return (__double2hiint(v.re) & 0x7ff00000) != 0x7ff00000 && (__double2hiint(v.im) & 0x7ff00000) != 0x7ff00000;
}

}  // namespace qmc3

// partial layout: fused [run][shift][slice][NACC][2], persec [sector row][shift][slice][NACC][2]
template <int NDIM, int L, int KMAX>
__global__ void __launch_bounds__(QMC3_THREADS, (NDIM <= 4 ? 2 : 1)) qmc3_eval_kernel(const Qmc3Launch q) {
  using namespace qmc3;
  const Qmc2Launch &p = q.b;
  constexpr int NACC = QMC_MAXSING + KMAX + 1;
  constexpr int SMAX = NDIM < QMC3_MAXSING ? NDIM : QMC3_MAXSING;
  constexpr int T = QMC3_THREADS;

  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x;
  const Qmc2Work wk = p.work[blockIdx.x];

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
  double *slots_r = reinterpret_cast<double *>(smem + o);
  o += (size_t)p.max_nslots * T * 8;
  double2 *slots_c = reinterpret_cast<double2 *>(smem + o);
  o += (size_t)q.max_nslots_c * T * 16;
  double *sacc = reinterpret_cast<double *>(smem + o);  // persec: [nsec][NACC*2][T]
  double *slr = slots_r + tid;
  double2 *slc = slots_c + tid;

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
  slr[3 * NDIM * T] = 1.0;
  slc[NDIM * T] = make_double2(1.0, 0.0);
  mbar_wait(bar, 0);
  __syncthreads();

  const Qmc3ChunkHdr *ch = reinterpret_cast<const Qmc3ChunkHdr *>(sprog);
  const uint32_t *prog_r = reinterpret_cast<const uint32_t *>(sprog + sizeof(Qmc3ChunkHdr));
  const int nprog_r = ch->nprog_r, first_prod_r = ch->first_prod_r, local0_r = ch->nslots_r;
  const uint32_t *prog_c = prog_r + ((nprog_r + 3) & ~3);
  const int nprog_c = ch->nprog_c, first_prod_c = ch->first_prod_c, local0_c = ch->nslots_c;

  const uint32_t N = p.N;
  const double dN = (double)N;
  const uint32_t stride = (uint32_t)wk.nslices * T;
  uint32_t dz[NDIM];
#pragma unroll
  for (int j = 0; j < NDIM; ++j) dz[j] = (uint32_t)(((uint64_t)stride * p.zeff[j]) % N);

  unsigned cntImF = 0, cntReU = 0, cntNonFinite = 0, cntBoundary = 0;

  for (int kap = 0; kap < p.m; ++kap) {
    cd acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = cd{0.0, 0.0};
    if (p.persec)
      for (int i = 0; i < wk.nsec * NACC * 2; ++i) sacc[(size_t)i * T + tid] = 0.0;

    uint32_t cidx = (uint32_t)wk.slice * T + tid;
    uint32_t r[NDIM];
#pragma unroll
    for (int j = 0; j < NDIM; ++j) r[j] = (uint32_t)((p.off[j] + (uint64_t)cidx * p.zeff[j]) % N);

    for (; cidx < p.count; cidx += stride) {
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
        slr[j * T] = tj;
        slr[(NDIM + j) * T] = fast_log(tj, logtab);
        slr[(2 * NDIM + j) * T] = fast_rcp(tj);
        uint32_t rn = r[j] + dz[j];
        r[j] = rn >= N ? rn - N : rn;
      }
      if (!inside) {
        if (wk.count_boundary) ++cntBoundary;
        continue;
      }
      for (int i = 0; i < nprog_r; ++i) {
        const uint32_t pw = prog_r[i];
        slr[(first_prod_r + i) * T] = slr[(pw & 0xffffu) * T] * slr[(pw >> 16) * T];
      }
      for (int si = 0; si < wk.nsec; ++si) {
        const Qmc3SectorHdr *h = reinterpret_cast<const Qmc3SectorHdr *>(stab + soff[si]);
#define QMC3_CASE(NS_)                                                                                       \
  case NS_: {                                                                                                \
    if (NS_ <= SMAX) {                                                                                       \
      constexpr int NSC = NS_ <= SMAX ? NS_ : 0, KK = KMAX + NSC + 1;                                        \
      cd res[KK];                                                                                            \
      sector3<NDIM, L, NSC, KMAX>(h, slr, slc, local0_r, prog_c, nprog_c, first_prod_c, local0_c, q.lambda,  \
                                  logtab, res, cntImF, cntReU);                                              \
      bool fin = true;                                                                                       \
      _Pragma("unroll") for (int i = 0; i < KK; ++i) fin = fin && finite_hi(res[i]);                         \
      if (!fin) {                                                                                            \
        ++cntNonFinite;                                                                                      \
      } else if (!p.persec) {                                                                                \
        _Pragma("unroll") for (int i = 0; i < KK; ++i) {                                                     \
          acc[QMC_MAXSING - NSC + i].re = fma(w, res[i].re, acc[QMC_MAXSING - NSC + i].re);                  \
          acc[QMC_MAXSING - NSC + i].im = fma(w, res[i].im, acc[QMC_MAXSING - NSC + i].im);                  \
        }                                                                                                    \
      } else {                                                                                               \
        double *sa = sacc + ((size_t)si * NACC + (QMC_MAXSING - NSC)) * 2 * T + tid;                         \
        _Pragma("unroll") for (int i = 0; i < KK; ++i) {                                                     \
          sa[(size_t)(2 * i) * T] += w * res[i].re;                                                          \
          sa[(size_t)(2 * i + 1) * T] += w * res[i].im;                                                      \
        }                                                                                                    \
      }                                                                                                      \
    }                                                                                                        \
  } break;
        switch (h->nsing) {
          QMC3_CASE(0)
          QMC3_CASE(1)
          QMC3_CASE(2)
          default:
            break;
        }
#undef QMC3_CASE
      }
    }

    if (!p.persec) {
      double *dst = p.partial + (((size_t)wk.out_row * p.m + kap) * p.max_slices + wk.slice) * (NACC * 2);
#pragma unroll
      for (int a = 0; a < NACC; ++a) {
        double sr = qmcdev::block_sum(acc[a].re, scratch);
        double si = qmcdev::block_sum(acc[a].im, scratch);
        if (tid == 0) {
          dst[2 * a] = sr;
          dst[2 * a + 1] = si;
        }
      }
    } else {
      for (int si = 0; si < wk.nsec; ++si) {
        double *dst = p.partial + (((size_t)(wk.out_row + si) * p.m + kap) * p.max_slices + wk.slice) * (NACC * 2);
        for (int a = 0; a < NACC * 2; ++a) {
          double v = qmcdev::block_sum(sacc[((size_t)si * NACC * 2 + a) * T + tid], scratch);
          if (tid == 0) dst[a] = v;
        }
      }
    }
  }

  unsigned c4[4] = {cntImF, cntReU, cntNonFinite, cntBoundary};
#pragma unroll
  for (int qq = 0; qq < 4; ++qq) {
    unsigned v = c4[qq];
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) v += __shfl_down_sync(0xffffffffu, v, o2);
    if ((tid & 31) == 0 && v) atomicAdd(p.counters + qq, (unsigned long long)v);
  }
}
