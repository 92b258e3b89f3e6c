// Evaluation kernel of the complex path (physical region, contour deformation), "version 5", sm_100a.  Steps S1-S7.
//
// One thread = one lattice point; two slot tables per thread in shared memory: a REAL one at the lattice point (t_j,
// ln t_j, 1, products) that serves the gradient and Hessian polynomials of F^ -- emitted by qmc_prepare as record
// lists of their own -- and a COMPLEX one over the deformed variables z_j, refilled at every corner, that serves U^(z),
// F^(z).  Per corner Z of a sector (real point tau = t with the variables of Z set to 0):
//   S4  F^_i(tau), F^_ik(tau) from the record lists of the derivative polynomials;
//       rho_i = 1 - i lambda (1 - tau_i) F^_i,  z_i = tau_i rho_i,
//       J_ik = delta_ik [1 - i lambda (1 - 2 tau_i) F^_i] - i lambda tau_i (1 - tau_i) F^_ik   (Eq. 14; R:C12),
//       det J by elimination in the natural order (no pivoting: see corner5);
//   S5  U^(z), F^(z) as sums of complex records;  G_Z = G0 det J prod_{j notin Z} rho_j^alpha_j U^aU0 F^aF0,
//       Lambda_Z = aU1 ln U + aF1 ln F + sum_j beta_j ln rho_j + L0   (principal logs; -i pi on the negative real axis, R:C11);
//   S6  product form folded one singular variable at a time with exact series windows (as qmc_fold.cuh, complex).
// The tables are in the kernel parameter block (constant bank 0; layout in qmc_launch.h) like those of the real path:
// every table read is a uniform load, the record loops run on the uniform datapath, and every corner of a sector owns a
// flat record stream (records needed by several corners are duplicated by the table builder), walked with the next
// record's slot operands in flight.  The corner is inlined inside a `for Z` loop with a uniform trip count (one copy of
// the corner code per number of singular variables); its results go to compile-time registers through a uniform
// `if (Z == q)` chain.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "qmc_kernels4.cuh"  // fast_log (64 x 8 table), fast_rcp, slot_at, u2d

#ifndef QMC5_MINB
// resident 128-thread blocks per SM the register budget is sized for: n <= 4: 4 (128 registers); n = 5: 3 (168 registers,
// 92 bytes of spills; needs <= 75 KB of shared memory per block: the slot budgets of qmc_image3.cpp); n = 6: 2 (255)
#define QMC5_MINB(NDIM) ((NDIM) <= 4 ? 4 : (NDIM) == 5 ? 3 : 2)
#endif

namespace qmc5 {

using qmc2::Expo;
using qmc4::fast_log;
using qmc4::fast_rcp;
using qmc4::slot_at;
using qmc4::u2d;
using qmcdev::cd;
using qmcdev::cnorm2;

// 1 / a with the MUFU.RCP64H + cubic-step reciprocal of the real path (|a|^2 is a normal number: pivots of 1 + iS have
// modulus >= 1, U^, F^, rho_j are O(1)) instead of the IEEE division routine: six of them per corner
__device__ __forceinline__ cd cinv5(cd a) {
  const double d = fast_rcp(a.re * a.re + a.im * a.im);
  return cd{a.re * d, -a.im * d};
}
__device__ __forceinline__ double2 cslot_at(const unsigned char *__restrict__ sl, uint32_t off) {
  return *reinterpret_cast<const double2 *>(sl + off);
}
static __device__ __noinline__ double atan2_lib(double y, double x) { return atan2(y, x); }
// principal log; a negative real argument carries the -i0 of F -> F - i0: arg = -pi (R:C11)
__device__ __forceinline__ cd clog5(cd a, const double2 *__restrict__ tabq) {
  const double arg = (a.im == 0.0 && a.re < 0.0) ? -3.14159265358979323846 : atan2_lib(a.im, a.re);
  return cd{0.5 * fast_log(cnorm2(a), tabq), arg};
}
// phase of a to about 1e-5 in single precision, with the convention of clog5 on the negative real axis; only ever used to
// fix a winding number (|values| of U^, F^, rho_j are far inside the single-precision range; outside it the estimate falls
// back to the double-precision routine)
__device__ __forceinline__ float arg_estimate(cd a) {
  if (a.im == 0.0 && a.re < 0.0) return -3.14159265f;
  const float x = (float)a.re, y = (float)a.im;
  const float ax = fabsf(x), ay = fabsf(y), mx = fmaxf(ax, ay), mn = fminf(ax, ay);
  if (!(mx > 1e-30f && mx < 1e30f)) return (float)atan2_lib(a.im, a.re);
  const float t = mn * __frcp_rn(mx), s = t * t;
  float p = t * (0.99997726f + s * (-0.33262347f + s * (0.19354346f + s * (-0.11643287f + s * (0.05265332f + s * -0.01172120f)))));
  if (ay > ax) p = 1.57079633f - p;
  if (x < 0.0f) p = 3.14159265f - p;
  return y < 0.0f ? -p : p;
}
template <int E>
__device__ __forceinline__ cd cpow_c(cd x) {  // x^E, E >= 0 compile time
  if (E == 0) return cd{1.0, 0.0};
  if (E == 1) return x;
  cd h = cpow_c<E / 2>(x);
  h = h * h;
  return (E & 1) ? h * x : h;
}
__device__ __forceinline__ int sext8(uint32_t w, int k) { return (int)(int8_t)((w >> (8 * k)) & 255u); }

// W_Z and Lambda_Z of one corner.  Z (bit mask over the singular positions) is warp-uniform; `cw` = word offset of the
// corner block in p.tab.
template <int NDIM, int L, int NS>
__device__ __forceinline__ void corner5(const Qmc5Launch &p, const uint32_t cw, const int Z, const uint32_t singvar,
                                        const uint32_t alo, const uint32_t ahi, const uint32_t blo, const uint32_t bhi,
                                        const uint32_t lcw, const uint32_t nlocal_c,
                                        const double G0, const double L0, unsigned char *__restrict__ slr,
                                        unsigned char *__restrict__ slc, const double2 *__restrict__ tabq, cd &Wout, cd &Lout,
                                        unsigned &cntImF, unsigned &cntReU, const bool need_lambda) {
  constexpr int T = QMC3_THREADS, NDERIV = NDIM + NDIM * (NDIM + 1) / 2, NPOLY = NDERIV + 2, CW = (NPOLY + 15) / 16;
  typedef Expo<NDIM, L> E;
  uint32_t zv = 0;  // variables set to zero
#pragma unroll
  for (int k = 0; k < NS; ++k)
    if (Z >> k & 1) zv |= 1u << ((singvar >> (8 * k)) & 255u);
  // corner block: counts of stream A (one-factor records) and of stream B (two-factor records) per polynomial, the constant
  // terms c0[NPOLY], then the four streams (real A, real B, complex A, complex B), each closed by two sentinels
  constexpr int C0W = (NPOLY + 1) / 2;
  uint32_t cntA[CW * 4], cntB[CW * 4];
#pragma unroll
  for (int q = 0; q < CW; ++q) {
    const uint4 w = p.tab[cw + q], x = p.tab[cw + CW + q];
    cntA[4 * q] = w.x; cntA[4 * q + 1] = w.y; cntA[4 * q + 2] = w.z; cntA[4 * q + 3] = w.w;
    cntB[4 * q] = x.x; cntB[4 * q + 1] = x.y; cntB[4 * q + 2] = x.z; cntB[4 * q + 3] = x.w;
  }
  const unsigned char *tb = reinterpret_cast<const unsigned char *>(p.tab);
  const unsigned char *c0p = tb + (cw + 2 * CW) * 16u;  // c0[NPOLY] (f64)
  uint32_t rwb = (cw + 2 * CW + C0W) * 16u;              // byte offset of the current record
  // ---- S4: gradient and Hessian of F^ at tau.  Pass A: constant + one-factor records c * slot (one load, one FMA) at fixed
  // positions; pass B: two-factor records c * slot * slot, ONE software-pipelined stream over all polynomials: the slot operands
  // of the next record are requested before the current one is accumulated (operands one record ahead, table words two).
  double dv[NDERIV];
  {  // pass A: fixed positions per polynomial (qmc_tables.h: qmc5_capA), straight-line code with compile-time record offsets
    const unsigned char *ra = tb + rwb;
#pragma unroll
    for (int q = 0; q < NDERIV; ++q) {
      double acc = *reinterpret_cast<const double *>(c0p + q * 8);
#pragma unroll
      for (int k = 0; k < qmc5_capA(NDIM, L, q); ++k) {
        const uint4 r = *reinterpret_cast<const uint4 *>(ra + (qmc5_posA(NDIM, L, q) + k) * 16);
        acc = fma(u2d(r.x, r.y), slot_at(slr, r.z), acc);
      }
      dv[q] = acc;
    }
    rwb += (uint32_t)qmc5_posA(NDIM, L, NDERIV) * 16u;
  }
  {
    uint2 ro = *reinterpret_cast<const uint2 *>(tb + rwb + 8);
    double ra = slot_at(slr, ro.x), rb = slot_at(slr, ro.y);
    ro = *reinterpret_cast<const uint2 *>(tb + rwb + 24);
#pragma unroll
    for (int q = 0; q < NDERIV; ++q) {
      const uint32_t n = (cntB[q >> 2] >> (8 * (q & 3))) & 255u;
      double acc = dv[q];
#pragma unroll 1
      for (uint32_t i = 0; i < n; ++i) {
        const uint2 rc = *reinterpret_cast<const uint2 *>(tb + rwb);
        const double v = ra * rb;
        rwb += 16u;
        ra = slot_at(slr, ro.x);
        rb = slot_at(slr, ro.y);
        ro = *reinterpret_cast<const uint2 *>(tb + rwb + 24);
        acc = fma(u2d(rc.x, rc.y), v, acc);
      }
      dv[q] = acc;
    }
    rwb += 32u;  // the two sentinels of stream B
  }
  // rho_i, z_i, J = 1 + i B
  cd rho[NDIM], J[NDIM][NDIM];
#pragma unroll
  for (int i = 0; i < NDIM; ++i) {
    const bool inZ = (zv >> i & 1u) != 0;
    const double tau = inZ ? 0.0 : slot_at(slr, i * T * 8);
    rho[i] = cd{1.0, -p.lambda * (1.0 - tau) * dv[i]};
    *reinterpret_cast<double2 *>(slc + i * T * 16) = make_double2(tau, tau * rho[i].im);  // z_i = tau rho_i
#pragma unroll
    for (int k = 0; k < NDIM; ++k) {
      const bool kinZ = (zv >> k & 1u) != 0;
      if (inZ || kinZ) {
        J[i][k] = cd{(i == k) ? 1.0 : 0.0, 0.0};  // row / column of a Z variable: its rho cancels rho^-1 (alpha = -1)
      } else {
        const int a = i < k ? i : k, b = i < k ? k : i;  // Hessian entry (a <= b) in emission order
        const double hik = dv[NDIM + a * NDIM - a * (a - 1) / 2 + (b - a)];
        double bb = -p.lambda * tau * (1.0 - tau) * hik;
        if (i == k) bb += -p.lambda * (1.0 - 2.0 * tau) * dv[i];
        J[i][k] = cd{(i == k) ? 1.0 : 0.0, bb};
      }
    }
  }
  // det J by elimination WITHOUT pivoting.  J = 1 + i (E + D H) with E, D real diagonal, D = diag(tau (1 - tau)) >= 0 and H
  // the real symmetric Hessian: J is diagonally similar to 1 + i S, S real symmetric, whose Hermitian part is the identity --
  // every leading principal minor has modulus >= 1 and elimination in the natural order is stable (no growth beyond that of
  // S), with the same pivots.  Row exchanges in registers had cost a fifth of the kernel's instructions in moves and selects
  // (profiles/r02a_final.md).  The oracle pivots; the determinants agree to rounding.
  cd det = cd{1.0, 0.0};
#pragma unroll
  for (int col = 0; col < NDIM; ++col) {
    det = det * J[col][col];
    if (col + 1 < NDIM) {
      const cd ip = cinv5(J[col][col]);
#pragma unroll
      for (int r = col + 1; r < NDIM; ++r) {
        const cd f = J[r][col] * ip;
#pragma unroll
        for (int k = col + 1; k < NDIM; ++k) J[r][k] = J[r][k] - f * J[col][k];
      }
    }
  }
  // ---- S5: complex slot table over z, U^(z), F^(z) -----------------------------------------------------------------
  for (uint32_t i = 0; i < p.nprog_c; i += 2) {
    const uint4 pw = p.tab[p.prog_c_word + (i >> 1)];
    {
      const double2 a = cslot_at(slc, pw.x), b = cslot_at(slc, pw.y);
      *reinterpret_cast<double2 *>(slc + p.first_prod_c_off + i * (T * 16)) = make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
    }
    if (i + 1 < p.nprog_c) {
      const double2 a = cslot_at(slc, pw.z), b = cslot_at(slc, pw.w);
      *reinterpret_cast<double2 *>(slc + p.first_prod_c_off + (i + 1) * (T * 16)) = make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
    }
  }
  for (uint32_t i = 0; i < nlocal_c; i += 2) {  // sector-local complex products
    const uint4 pw = p.tab[lcw + (i >> 1)];
    {
      const double2 a = cslot_at(slc, pw.x), b = cslot_at(slc, pw.y);
      *reinterpret_cast<double2 *>(slc + p.local0_c_off + i * (T * 16)) = make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
    }
    if (i + 1 < nlocal_c) {
      const double2 a = cslot_at(slc, pw.z), b = cslot_at(slc, pw.w);
      *reinterpret_cast<double2 *>(slc + p.local0_c_off + (i + 1) * (T * 16)) = make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
    }
  }
  cd UF[2];
  {  // pass A: constant + one-factor complex records c * slot
    uint32_t ro = *reinterpret_cast<const uint32_t *>(tb + rwb + 8);
    double2 ra = cslot_at(slc, ro);
    ro = *reinterpret_cast<const uint32_t *>(tb + rwb + 24);
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const uint32_t n = (cntA[(NDERIV + q) >> 2] >> (8 * ((NDERIV + q) & 3))) & 255u;
      cd acc = cd{*reinterpret_cast<const double *>(c0p + (NDERIV + q) * 8), 0.0};
#pragma unroll 1
      for (uint32_t i = 0; i < n; ++i) {
        const uint2 rc = *reinterpret_cast<const uint2 *>(tb + rwb);
        const double2 v = ra;
        rwb += 16u;
        ra = cslot_at(slc, ro);
        ro = *reinterpret_cast<const uint32_t *>(tb + rwb + 24);
        const double c = u2d(rc.x, rc.y);
        acc.re = fma(c, v.x, acc.re);
        acc.im = fma(c, v.y, acc.im);
      }
      UF[q] = acc;
    }
    rwb += 32u;
  }
  {  // pass B: two-factor complex records c * slot * slot
    uint2 ro = *reinterpret_cast<const uint2 *>(tb + rwb + 8);
    double2 ra = cslot_at(slc, ro.x), rb = cslot_at(slc, ro.y);
    ro = *reinterpret_cast<const uint2 *>(tb + rwb + 24);
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const uint32_t n = (cntB[(NDERIV + q) >> 2] >> (8 * ((NDERIV + q) & 3))) & 255u;
      cd acc = UF[q];
#pragma unroll 1
      for (uint32_t i = 0; i < n; ++i) {
        const uint2 rc = *reinterpret_cast<const uint2 *>(tb + rwb);
        const double vr = ra.x * rb.x - ra.y * rb.y, vi = ra.x * rb.y + ra.y * rb.x;
        rwb += 16u;
        ra = cslot_at(slc, ro.x);
        rb = cslot_at(slc, ro.y);
        ro = *reinterpret_cast<const uint2 *>(tb + rwb + 24);
        const double c = u2d(rc.x, rc.y);
        acc.re = fma(c, vr, acc.re);
        acc.im = fma(c, vi, acc.im);
      }
      UF[q] = acc;
    }
  }
  const cd Uv = UF[0], Fv = UF[1];
  if (Fv.im > 0.0) ++cntImF;
  if (!(Uv.re > 0.0)) ++cntReU;
  // G_Z = G0 det J prod_{j notin Z} rho_j^alpha_j U^aU0 F^aF0 ;  Lambda_Z = aU1 ln U + aF1 ln F + sum_j beta_j ln rho_j + L0.
  // The 2 + n principal logarithms are taken as ONE: Lambda_Z - L0 = ln Q + 2 pi i k with Q = U^aU1 F^aF1 prod_j rho_j^beta_j
  // (complex products) and the winding number k fixed by single-precision estimates of the same phases: the sum of the
  // principal phases, known to 1e-3, differs from the principal phase of Q by an exact multiple of 2 pi.
  // Lambda_Z is needed only where the corner's eps-series has more than one term (need_lambda, warp-uniform: k_max > 0 or Z
  // not empty); a corner with a one-term window -- every corner of a sector without singular variables at k_max = 0 -- skips it.
  cd num = cd{G0 * det.re, G0 * det.im}, den = cd{1.0, 0.0};
#pragma unroll
  for (int j = 0; j < NDIM; ++j) {
    const bool inZ = (zv >> j & 1u) != 0;
    const int a = sext8(j < 4 ? alo : ahi, j & 3);
    if (!inZ) {
      if (a < 0) den = den * rho[j];
      for (int q = 0; q < a; ++q) num = num * rho[j];
    }
  }
  cd Lam = cd{0.0, 0.0};
  if (need_lambda) {
    cd qn = cpow_c<(E::aU1 > 0 ? E::aU1 : 0)>(Uv), qd = cpow_c<(E::aF1 < 0 ? -E::aF1 : 0)>(Fv);
    float th = (float)E::aU1 * arg_estimate(Uv) + (float)E::aF1 * arg_estimate(Fv);
#pragma unroll
    for (int j = 0; j < NDIM; ++j) {
      const int b = sext8(j < 4 ? blo : bhi, j & 3);
      if (b) {
        th += (float)b * arg_estimate(rho[j]);
        for (int q = 0; q < b; ++q) qn = qn * rho[j];
        for (int q = 0; q < -b; ++q) qd = qd * rho[j];
      }
    }
    Lam = clog5(qn * cinv5(qd), tabq);
    Lam.im = fma((double)rintf((th - (float)Lam.im) * 0.15915494f), 6.28318530717958647692, Lam.im);
    Lam.re += L0;
  }
  if (E::aU0 > 0) num = num * cpow_c<(E::aU0 > 0 ? E::aU0 : 0)>(Uv);
  if (E::aU0 < 0) den = den * cpow_c<(E::aU0 < 0 ? -E::aU0 : 0)>(Uv);
  if (E::aF0 > 0) num = num * cpow_c<(E::aF0 > 0 ? E::aF0 : 0)>(Fv);
  if (E::aF0 < 0) den = den * cpow_c<(E::aF0 < 0 ? -E::aF0 : 0)>(Fv);
  Wout = num * cinv5(den);
  Lout = Lam;
}

template <int NS, int K>
struct Ctx5 {
  double bt[NS > 0 ? NS : 1];  // t_k / beta_k (the 1/t_k of Eq. 12 are factored out of the fold: one reciprocal onto G0)
  double cL[NS > 0 ? NS : 1][K > 1 ? K - 1 : 1];
  cd W[1 << NS], Lam[1 << NS];  // index Z = set of singular positions set to zero
};

// fold of the singular variables with exact series windows (see qmc2::Fold2), complex
template <int NS, int KMAX, int K, int LEVEL, int ZMASK>
struct Fold5 {
  static constexpr int LEN = NS - LEVEL + KMAX + __builtin_popcount(ZMASK) + 1;
  static __device__ __forceinline__ void eval(const Ctx5<NS, K> &c, cd (&out)[LEN]) {
    cd a[LEN - 1], b[LEN];
    Fold5<NS, KMAX, K, LEVEL + 1, ZMASK>::eval(c, a);
    Fold5<NS, KMAX, K, LEVEL + 1, ZMASK | (1 << LEVEL)>::eval(c, b);
    const double bt = c.bt[LEVEL];
    cd d[LEN - 1];
#pragma unroll
    for (int i = 0; i < LEN - 1; ++i) d[i] = a[i] - b[i];
    out[0] = bt * b[0];
#pragma unroll
    for (int i = 1; i < LEN; ++i) {
      cd s = bt * b[i] + d[i - 1];
#pragma unroll
      for (int p = 1; p < i; ++p) s = s + c.cL[LEVEL][p] * d[i - 1 - p];
      out[i] = s;
    }
  }
};
template <int NS, int KMAX, int K, int ZMASK>
struct Fold5<NS, KMAX, K, NS, ZMASK> {
  static constexpr int LEN = KMAX + __builtin_popcount(ZMASK) + 1;
  static __device__ __forceinline__ void eval(const Ctx5<NS, K> &c, cd (&out)[LEN]) {
    out[0] = c.W[ZMASK];
#pragma unroll
    for (int p = 1; p < LEN; ++p) out[p] = (1.0 / p) * (out[p - 1] * c.Lam[ZMASK]);
  }
};

// one sector at one point: out[i] = coefficient of eps^(i - NS).  `o` = word offset of the sector block (uniform).
template <int NDIM, int L, int NS, int KMAX>
__device__ __forceinline__ void sector5(const Qmc5Launch &p, const uint32_t o, unsigned char *__restrict__ slr,
                                        unsigned char *__restrict__ slc, const double2 *__restrict__ tabq,
                                        cd (&out)[KMAX + NS + 1], unsigned &cntImF, unsigned &cntReU) {
  constexpr int K = KMAX + NS + 1, NG = 1 << NS, T = QMC3_THREADS;
  const uint4 h0 = p.tab[o], h1 = p.tab[o + 1], h2 = p.tab[o + 2];
  const uint32_t nL0 = (h0.x >> 8) & 255u, nlocal_r = (h0.x >> 16) & 255u, nlocal_c = (h0.x >> 24) & 255u;
  const uint32_t lrw = o + 8, lcw = lrw + ((nlocal_r + 1) >> 1);
  for (uint32_t i = 0; i < nlocal_r; i += 2) {  // sector-local real products
    const uint4 pw = p.tab[lrw + (i >> 1)];
    *reinterpret_cast<double *>(slr + p.local0_r_off + i * (T * 8)) = slot_at(slr, pw.x) * slot_at(slr, pw.y);
    if (i + 1 < nlocal_r) *reinterpret_cast<double *>(slr + p.local0_r_off + (i + 1) * (T * 8)) = slot_at(slr, pw.z) * slot_at(slr, pw.w);
  }
  uint32_t rw = o + h0.z;
  double G0 = qmc4::rec_val(p.tab[rw], slr);
  if (NS > 0) {  // the 1/t_k of the singular variables (Eq. 12), factored out of the fold: one reciprocal of their product
    double pt = slot_at(slr, (h1.x & 255u) * (T * 8));
#pragma unroll
    for (int k = 1; k < NS; ++k) pt *= slot_at(slr, ((h1.x >> (8 * k)) & 255u) * (T * 8));
    G0 *= fast_rcp(pt);
  }
  ++rw;
  double L0 = 0.0;
#pragma unroll 2
  for (uint32_t i = 0; i < nL0; ++i) L0 = qmc4::rec_fma(p.tab[rw + i], slr, L0);
  Ctx5<NS, K> c;
  const uint4 cdir = p.tab[o + 7];
  const uint32_t cws[4] = {cdir.x, cdir.y, cdir.z, cdir.w};
#pragma unroll 1
  for (int Z = 0; Z < NG; ++Z) {
    cd W, Lam;
    const uint32_t cw = o + (Z == 0 ? cws[0] : Z == 1 ? cws[1] : Z == 2 ? cws[2] : cws[3]);
    corner5<NDIM, L, NS>(p, cw, Z, h1.x, h1.z, h1.w, h2.x, h2.y, lcw, nlocal_c, G0, L0, slr, slc, tabq, W, Lam, cntImF, cntReU,
                         KMAX > 0 || Z != 0);
#pragma unroll
    for (int q = 0; q < NG; ++q)
      if (Z == q) {  // warp-uniform: the results land in compile-time registers
        c.W[q] = W;
        c.Lam[q] = Lam;
      }
  }
  if (NS > 0) {
    const uint4 ib01 = p.tab[o + 3], ib23 = p.tab[o + 4], b01 = p.tab[o + 5], b23 = p.tab[o + 6];
    const double ibv[4] = {u2d(ib01.x, ib01.y), u2d(ib01.z, ib01.w), u2d(ib23.x, ib23.y), u2d(ib23.z, ib23.w)};
    const double bv[4] = {u2d(b01.x, b01.y), u2d(b01.z, b01.w), u2d(b23.x, b23.y), u2d(b23.z, b23.w)};
#pragma unroll
    for (int k = 0; k < NS; ++k) {
      const uint32_t j = (h1.x >> (8 * k)) & 255u;
      c.bt[k] = ibv[k] * slot_at(slr, j * (T * 8));
      const double Lk = bv[k] * slot_at(slr, (NDIM + j) * (T * 8));
      c.cL[k][0] = 1.0;
#pragma unroll
      for (int q = 1; q < K - 1; ++q) c.cL[k][q] = c.cL[k][q - 1] * Lk * (1.0 / q);
    }
  }
  Fold5<NS, KMAX, K, 0, 0>::eval(c, out);
}

__device__ __forceinline__ bool finite_hi(cd v) {
  return (__double2hiint(v.re) & 0x7ff00000) != 0x7ff00000 && (__double2hiint(v.im) & 0x7ff00000) != 0x7ff00000;
}

}  // namespace qmc5

// partial layout: fused [run][shift][slice][NACC][2], persec [sector row][shift][slice][NACC][2]
template <int NDIM, int L, int KMAX>
__global__ void __launch_bounds__(QMC3_THREADS, QMC5_MINB(NDIM)) qmc5_eval_kernel(const __grid_constant__ Qmc5Launch p) {
  using namespace qmc5;
  constexpr int NACC = QMC_MAXSING + KMAX + 1;
  constexpr int SMAX = NDIM < QMC3_MAXSING ? NDIM : QMC3_MAXSING;
  constexpr int T = QMC3_THREADS;

  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x;
  double2 *logtab = reinterpret_cast<double2 *>(smem);
  size_t o = (size_t)QMC4_LOG_ENTRIES * QMC4_LOG_COPIES * 16;
  double *shf = reinterpret_cast<double *>(smem + o);
  o += (((size_t)p.m * NDIM * 8) + 15) & ~(size_t)15;
  double *scratch = reinterpret_cast<double *>(smem + o);
  o += (T / 32) * 8;
  double *slots_r = reinterpret_cast<double *>(smem + o);
  o += (size_t)p.max_nslots_r * T * 8;
  double2 *slots_c = reinterpret_cast<double2 *>(smem + o);
  o += (size_t)p.max_nslots_c * T * 16;
  double *sacc = reinterpret_cast<double *>(smem + o);  // persec: [nsec][NACC*2][T]
  unsigned char *slr = reinterpret_cast<unsigned char *>(slots_r + tid);
  unsigned char *slc = reinterpret_cast<unsigned char *>(slots_c + tid);
  const double2 *tabq = logtab + (tid & (QMC4_LOG_COPIES - 1));

  for (int i = tid; i < QMC4_LOG_ENTRIES * QMC4_LOG_COPIES; i += T)
    logtab[i] = reinterpret_cast<const double2 *>(p.logtab)[i / QMC4_LOG_COPIES];
  for (int i = tid; i < p.m * NDIM; i += T) shf[i] = p.shifts[i];
  slots_r[2 * NDIM * T + tid] = 1.0;                     // the constant slots
  slots_c[NDIM * T + tid] = make_double2(1.0, 0.0);
  __syncthreads();

  const uint32_t N = p.N;
  const double dN = (double)N, invN = 1.0 / dN;
  const uint32_t stride = (uint32_t)p.nslices * T;
  uint32_t dz[NDIM];
#pragma unroll
  for (int j = 0; j < NDIM; ++j) dz[j] = (uint32_t)(((uint64_t)stride * p.zeff[j]) % N);

  unsigned cntImF = 0, cntReU = 0, cntNonFinite = 0, cntBoundary = 0;
  const int kap = blockIdx.y;  // one block = one shift vector (see qmc_kernels4.cuh)
  {
    cd acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = cd{0.0, 0.0};
    if (p.persec)
      for (int i = 0; i < p.nsec * NACC * 2; ++i) sacc[(size_t)i * T + tid] = 0.0;

    const uint32_t c0 = (uint32_t)blockIdx.x * T;
    uint32_t r[NDIM];
#pragma unroll
    for (int j = 0; j < NDIM; ++j) r[j] = (uint32_t)((p.off[j] + (uint64_t)(c0 + tid) * p.zeff[j]) % N);

    for (uint32_t cb = c0; cb < p.count; cb += stride) {  // uniform trip count; dead threads carry the weight 0
      const bool valid = cb + tid < p.count;
      double w = 1.0;
      bool inside = true;
#pragma unroll
      for (int j = 0; j < NDIM; ++j) {
        // u = r / N correctly rounded (the oracle's IEEE division) as on the real path: q = r * RN(1/N), exact remainder by
        // FMA, one correction (Markstein; r, N integers below 2^31)
        const double rd = (double)r[j], q0 = rd * invN;
        const double u = fma(fma(-q0, dN, rd), invN, q0);
        double y = u + shf[kap * NDIM + j];
        if (y >= 1.0) y -= 1.0;
        double tj;
        if (p.transform != 1) {  // Eq. 21 (3y^2 - 2y^3, weight 6y(1-y)) or its r = 2 sibling, as data: qmc_transform_poly
          const double yq = y * (1.0 - y);
          tj = (y * y) * fma(y, fma(y, fma(y, p.tc[3], p.tc[2]), p.tc[1]), p.tc[0]);
          w *= yq * fma(yq, p.wc[1], p.wc[0]);
        } else {
          tj = 1.0 - fabs(2.0 * y - 1.0);
        }
        if (!(y > 0.0) || !(tj > 0.0)) {
          inside = false;
          tj = 0.5;
        }
        reinterpret_cast<double *>(slr)[j * T] = tj;
        reinterpret_cast<double *>(slr)[(NDIM + j) * T] = fast_log(tj, tabq);
        uint32_t rn = r[j] + dz[j];
        r[j] = rn >= N ? rn - N : rn;
      }
      if (valid && !inside && p.count_boundary) ++cntBoundary;
      const bool live = valid && inside;
      if (!live) w = 0.0;
      for (uint32_t i = 0; i < p.nprog_r; i += 2) {  // chunk-wide real product slots
        const uint4 pw = p.tab[p.prog_r_word + (i >> 1)];
        *reinterpret_cast<double *>(slr + p.first_prod_r_off + i * (T * 8)) = slot_at(slr, pw.x) * slot_at(slr, pw.y);
        if (i + 1 < p.nprog_r)
          *reinterpret_cast<double *>(slr + p.first_prod_r_off + (i + 1) * (T * 8)) = slot_at(slr, pw.z) * slot_at(slr, pw.w);
      }
      for (int si = 0; si < p.nsec; ++si) {
        const uint32_t so = p.secw[si];
        const uint4 h0 = p.tab[so];
        unsigned dImF = 0, dReU = 0;
#define QMC5_CASE(NS_)                                                                                       \
  case NS_: {                                                                                                \
    if (NS_ <= SMAX) {                                                                                       \
      constexpr int NSC = NS_ <= SMAX ? NS_ : 0, KK = KMAX + NSC + 1;                                        \
      cd res[KK];                                                                                            \
      sector5<NDIM, L, NSC, KMAX>(p, so, slr, slc, tabq, res, dImF, dReU);                                   \
      bool fin = true;                                                                                       \
      _Pragma("unroll") for (int i = 0; i < KK; ++i) fin = fin && finite_hi(res[i]);                         \
      cntNonFinite += (live && !fin) ? 1u : 0u;                                                              \
      if (!p.persec) {                                                                                       \
        _Pragma("unroll") for (int i = 0; i < KK; ++i) if (fin) {                                            \
          acc[QMC_MAXSING - NSC + i].re = fma(w, res[i].re, acc[QMC_MAXSING - NSC + i].re);                  \
          acc[QMC_MAXSING - NSC + i].im = fma(w, res[i].im, acc[QMC_MAXSING - NSC + i].im);                  \
        }                                                                                                    \
      } else {                                                                                               \
        double *sa = sacc + ((size_t)si * NACC + (QMC_MAXSING - NSC)) * 2 * T + tid;                         \
        _Pragma("unroll") for (int i = 0; i < KK; ++i) if (fin) {                                            \
          sa[(size_t)(2 * i) * T] += w * res[i].re;                                                          \
          sa[(size_t)(2 * i + 1) * T] += w * res[i].im;                                                      \
        }                                                                                                    \
      }                                                                                                      \
    }                                                                                                        \
  } break;
        switch (h0.x & 255u) {
          QMC5_CASE(0)
          QMC5_CASE(1)
          QMC5_CASE(2)
          default:
            break;
        }
#undef QMC5_CASE
        if (live) {  // the contour counters tally evaluated points only
          cntImF += dImF;
          cntReU += dReU;
        }
      }
    }

    if (!p.persec) {
      double *dst = p.partial + (((size_t)p.out_row * p.m + kap) * p.max_slices + blockIdx.x) * (NACC * 2);
#pragma unroll
      for (int a = 0; a < NACC; ++a) {
        double sr = qmc4::block_sum_t<T>(acc[a].re, scratch);
        double si = qmc4::block_sum_t<T>(acc[a].im, scratch);
        if (tid == 0) {
          dst[2 * a] = sr;
          dst[2 * a + 1] = si;
        }
      }
    } else {
      for (int si = 0; si < p.nsec; ++si) {
        double *dst = p.partial + (((size_t)(p.out_row + p.secrow[si]) * p.m + kap) * p.max_slices + blockIdx.x) * (NACC * 2);
        for (int a = 0; a < NACC * 2; ++a) {
          double v = qmc4::block_sum_t<T>(sacc[((size_t)si * NACC * 2 + a) * T + tid], scratch);
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
