// Evaluation kernel of the hot path (steps S1-S7 of DESIGN.md), sm_100a.
//
// One thread = one lattice point at a time (grid-stride over the points of one shift), all sectors of the
// block's chunk evaluated for that point with the per-point quantities (t_j, ln t_j, 1/t_j) computed once.
// Sector tables are staged in shared memory with one TMA bulk copy per block (cp.async.bulk + mbarrier) and read
// with warp-uniform (broadcast) loads.  Everything else lives in registers: FP64 (complex) arithmetic,
// truncated Laurent series, the 2^s corners of the subtraction.
//
// Per sector with s singular variables (alpha = -1), the eps-expanded subtracted integrand (Eqs. 9-12,
// PAPER.md:94-114) is evaluated in product form:
//   sum_k c_k eps^k = sum_{Z subset sing} g_Z(eps) prod_{j notin Z} A_j(eps) prod_{j in Z} (B_j(eps) - A_j(eps)),
//   g_Z = G_Z exp(eps Lambda_Z),  A_j = t_j^-1 exp(eps beta_j ln t_j),  B_j = 1/(beta_j eps),
// folded one singular variable at a time:  h <- A_j (h[Z without j] - h[Z with j]) + B_j h[Z with j].
// (The oracle uses the expanded double-sum form instead.)
// Real path: U^(t^Z), F^(t^Z) for all 2^s corners come from ONE pass over the monomials (partial sums per
// "group" = set of singular variables a monomial depends on) followed by a subset-sum transform.
// Complex path: contour deformation (Eq. 14) at every corner: gradient and Hessian of F^ from
// the monomial table, z = t rho, det(dz/dt) by LU with row pivoting, complex U^(z), F^(z), complex logs.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

#include "qmc_tables.h"

#include "qmc_launch.h"

// partial layout: fused  : [chunk][shift][block][NACC*(1|2)]
//                 persec : [sector - sec_begin][shift][block][NACC*(1|2)]
// accumulator index a <-> order k = a - QMC_MAXSING  (so that a sector with s singular variables writes
// a = QMC_MAXSING - s .. QMC_MAXSING + kmax with compile-time indices).

namespace qmcdev {

struct cd {
  double re, im;
};
__device__ __forceinline__ cd operator+(cd a, cd b) { return cd{a.re + b.re, a.im + b.im}; }
__device__ __forceinline__ cd operator-(cd a, cd b) { return cd{a.re - b.re, a.im - b.im}; }
__device__ __forceinline__ cd operator*(cd a, cd b) {
  return cd{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re};
}
__device__ __forceinline__ cd operator*(double s, cd a) { return cd{s * a.re, s * a.im}; }
__device__ __forceinline__ cd cinv(cd a) {
  double d = 1.0 / (a.re * a.re + a.im * a.im);
  return cd{a.re * d, -a.im * d};
}
__device__ __forceinline__ double cnorm2(cd a) { return a.re * a.re + a.im * a.im; }
// principal log; a negative real argument carries the -i0 of F -> F - i0: arg = -pi (R:C11)
__device__ __forceinline__ cd clog_m(cd a) {
  double arg = (a.im == 0.0 && a.re < 0.0) ? -3.14159265358979323846 : atan2(a.im, a.re);
  return cd{0.5 * log(cnorm2(a)), arg};
}

template <class T>
struct Num;
template <>
struct Num<double> {
  static __device__ __forceinline__ double zero() { return 0.0; }
  static __device__ __forceinline__ double scale(double s, double a) { return s * a; }
};
template <>
struct Num<cd> {
  static __device__ __forceinline__ cd zero() { return cd{0.0, 0.0}; }
  static __device__ __forceinline__ cd scale(double s, cd a) { return cd{s * a.re, s * a.im}; }
};

__device__ __forceinline__ double ipow_pos(double x, int e) {  // e >= 0, small
  double r = 1.0;
  for (int q = 0; q < e; ++q) r *= x;
  return r;
}

// c * prod_j x_j^{e_j}; exponents are warp-uniform nibbles of w
template <int NDIM>
__device__ __forceinline__ double monomial(double c, uint32_t w, const double (&x)[NDIM]) {
  double v = c;
#pragma unroll
  for (int j = 0; j < NDIM; ++j) {
    int e = (w >> (4 * j)) & 15;
    if (e) {
      v *= x[j];
      if (e > 1) {
        v *= x[j];
        for (int q = 2; q < e; ++q) v *= x[j];
      }
    }
  }
  return v;
}

// per-sector context shared by all corners
template <int NDIM, int NS, class T>
struct Ctx {
  double t[NDIM];            // permuted variables (singular first)
  double invt[NS > 0 ? NS : 1];
  double invbeta[NS > 0 ? NS : 1];
  double cL[NS > 0 ? NS : 1][QMC_NACC_MAX];  // (beta_j ln t_j)^p / p!
  double G0, L0;             // regular-variable factor and log (common to all corners)
  int aU0, aU1, aF0, aF1;
  // real path: subset sums of U^, F^ over the groups
  double PU[1 << NS], PF[1 << NS];
  // complex path
  double lambda;
  double invt_all[NDIM];
  const QmcSectorHdr *hdr;
  const double *coef;
  const uint32_t *exps;
  unsigned cntImF, cntReU;
};

// ---- corner value g_Z(eps) = G_Z exp(eps Lambda_Z), truncated to K terms ------------------------------
template <int NDIM, int NS, int K, int ZMASK>
__device__ __forceinline__ void corner_series(Ctx<NDIM, NS, double> &c, double (&out)[K]) {
  constexpr int FULL = (1 << NS) - 1;
  double Uv = c.PU[FULL ^ ZMASK], Fv = c.PF[FULL ^ ZMASK];
  double num = c.G0, den = 1.0;
  {
    double pu = ipow_pos(Uv, c.aU0 < 0 ? -c.aU0 : c.aU0), pf = ipow_pos(Fv, c.aF0 < 0 ? -c.aF0 : c.aF0);
    if (c.aU0 >= 0) num *= pu; else den *= pu;
    if (c.aF0 >= 0) num *= pf; else den *= pf;
  }
  double W = num / den;
  double Lam = (double)c.aU1 * log(Uv) + (double)c.aF1 * log(Fv) + c.L0;
  out[0] = W;
#pragma unroll
  for (int p = 1; p < K; ++p) out[p] = out[p - 1] * Lam * (1.0 / p);
}

// ZMASK is a run-time (warp-uniform) argument here: nothing below indexes a register array with it, and one
// out-of-line copy per (NDIM, NS, K) keeps the code size and the compile time down.
template <int NDIM, int NS, int K>
__device__ __noinline__ void corner_series_cplx(Ctx<NDIM, NS, cd> &c, const int ZMASK, cd (&out)[K]) {
  // tau = t with the components in Z set to 0.  Only monomials free of Z-variables survive in U^(z), F^(z) and
  // in the derivatives w.r.t. non-Z variables; dF^/dt_a for a in Z picks the monomials linear in t_a.
  const QmcSectorHdr *h = c.hdr;
  const int nU = h->nU, nF = h->nF;
  double grad[NDIM], hess[NDIM][NDIM];
#pragma unroll
  for (int i = 0; i < NDIM; ++i) {
    grad[i] = 0.0;
#pragma unroll
    for (int k = 0; k < NDIM; ++k) hess[i][k] = 0.0;
  }
  // nibble mask of the Z positions
  uint32_t zn = 0;
#pragma unroll
  for (int b = 0; b < NS; ++b)
    if (ZMASK >> b & 1) zn |= 15u << (4 * b);
  for (int mi = 0; mi < nF; ++mi) {
    uint32_t w = c.exps[nU + mi];
    uint32_t wz = w & zn;
    double v0 = monomial<NDIM>(c.coef[nU + mi], w & ~zn, c.t);
    if (wz == 0) {
#pragma unroll
      for (int i = 0; i < NDIM; ++i) {
        if (i < NS && (ZMASK >> i & 1)) continue;
        int ei = (w >> (4 * i)) & 15;
        if (ei) {
          double gi = (double)ei * v0 * c.invt_all[i];
          grad[i] += gi;
#pragma unroll
          for (int k = i; k < NDIM; ++k) {
            if (k < NS && (ZMASK >> k & 1)) continue;
            int ek = ((w >> (4 * k)) & 15) - (k == i ? 1 : 0);
            if (ek > 0) hess[i][k] += gi * (double)ek * c.invt_all[k];
          }
        }
      }
    } else if ((wz & (wz - 1)) == 0 && (wz & 0x11111111u)) {
      // exactly one Z-variable, with exponent 1 (a single bit set, and it is the lowest bit of its nibble)
#pragma unroll
      for (int a = 0; a < NS; ++a)
        if ((ZMASK >> a & 1) && (wz >> (4 * a) & 15)) grad[a] += v0;
    }
  }
  // rho_i = 1 - i lambda (1 - tau_i) F_i ;  z_i = tau_i rho_i ;  J = 1 + i B
  cd z[NDIM], rho[NDIM];
  cd J[NDIM][NDIM];
#pragma unroll
  for (int i = 0; i < NDIM; ++i) {
    const bool inZ = (i < NS) && (ZMASK >> i & 1);
    double tau = inZ ? 0.0 : c.t[i];
    rho[i] = cd{1.0, -c.lambda * (1.0 - tau) * grad[i]};
    z[i] = cd{tau, tau * rho[i].im};
#pragma unroll
    for (int k = 0; k < NDIM; ++k) {
      const bool kinZ = (k < NS) && (ZMASK >> k & 1);
      if (inZ || kinZ) {
        J[i][k] = cd{(i == k) ? 1.0 : 0.0, 0.0};  // row/column of a Z variable: its rho_i cancels rho_i^-1 (alpha=-1)
      } else {
        double hik = (k >= i) ? hess[i][k] : hess[k][i];
        double b = -c.lambda * tau * (1.0 - tau) * hik;
        if (i == k) b += -c.lambda * (1.0 - 2.0 * tau) * grad[i];
        J[i][k] = cd{(i == k) ? 1.0 : 0.0, b};
      }
    }
  }
  // det J: Gaussian elimination with row pivoting (compare-and-swap down each column)
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
      cd ip = cinv(J[col][col]);
#pragma unroll
      for (int r = col + 1; r < NDIM; ++r) {
        cd f = J[r][col] * ip;
#pragma unroll
        for (int k = col + 1; k < NDIM; ++k) J[r][k] = J[r][k] - f * J[col][k];
      }
    }
  }
  // complex U^(z), F^(z): monomials free of Z variables
  cd Uv = cd{0.0, 0.0}, Fv = cd{0.0, 0.0};
  for (int mi = 0; mi < nU + nF; ++mi) {
    uint32_t w = c.exps[mi];
    if (w & zn) continue;
    cd v = cd{c.coef[mi], 0.0};
#pragma unroll
    for (int j = 0; j < NDIM; ++j) {
      int e = (w >> (4 * j)) & 15;
      for (int q = 0; q < e; ++q) v = v * z[j];
    }
    if (mi < nU) Uv = Uv + v; else Fv = Fv + v;
  }
  if (Fv.im > 0.0) ++c.cntImF;
  if (!(Uv.re > 0.0)) ++c.cntReU;
  // G_Z = G0 det J prod_{j notin Z} rho_j^{alpha_j} U^{aU0} F^{aF0}
  // Lambda_Z = aU1 ln U + aF1 ln F + sum_all beta_j ln rho_j + L0
  cd num = cd{c.G0, 0.0} * det, den = cd{1.0, 0.0};
  cd Lam = (double)c.aU1 * clog_m(Uv) + (double)c.aF1 * clog_m(Fv);
  Lam.re += c.L0;
#pragma unroll
  for (int j = 0; j < NDIM; ++j) {
    const bool inZ = (j < NS) && (ZMASK >> j & 1);
    int a = h->alpha[j], b = h->beta[j];
    if (!inZ) {
      for (int q = 0; q < (a < 0 ? -a : a); ++q) {
        if (a > 0) num = num * rho[j]; else den = den * rho[j];
      }
    }
    if (b) Lam = Lam + (double)b * clog_m(rho[j]);
  }
  {
    int eu = c.aU0 < 0 ? -c.aU0 : c.aU0, ef = c.aF0 < 0 ? -c.aF0 : c.aF0;
    for (int q = 0; q < eu; ++q) { if (c.aU0 > 0) num = num * Uv; else den = den * Uv; }
    for (int q = 0; q < ef; ++q) { if (c.aF0 > 0) num = num * Fv; else den = den * Fv; }
  }
  cd W = num * cinv(den);
  out[0] = W;
#pragma unroll
  for (int p = 1; p < K; ++p) out[p] = (1.0 / p) * (out[p - 1] * Lam);
}

// ---- fold the singular variables one at a time ---------------------------------------------------------
// Series windows: at depth d (d variables folded) index i <-> order i - d.  LEVEL = next variable to fold here.
template <int NDIM, int NS, int K, int LEVEL, int ZMASK, class T>
struct Fold {
  static __device__ __forceinline__ void eval(Ctx<NDIM, NS, T> &c, T (&out)[K]) {
    T a[K], b[K];
    Fold<NDIM, NS, K, LEVEL + 1, ZMASK, T>::eval(c, a);
    Fold<NDIM, NS, K, LEVEL + 1, ZMASK | (1 << LEVEL), T>::eval(c, b);
    const double it = c.invt[LEVEL], ib = c.invbeta[LEVEL];
    T d[K];
#pragma unroll
    for (int i = 0; i + 1 < K; ++i) d[i] = Num<T>::scale(it, a[i] - b[i]);
    out[0] = Num<T>::scale(ib, b[0]);
#pragma unroll
    for (int i = 1; i < K; ++i) {
      T s = Num<T>::scale(ib, b[i]) + d[i - 1];
#pragma unroll
      for (int p = 1; p < i; ++p) s = s + Num<T>::scale(c.cL[LEVEL][p], d[i - 1 - p]);
      out[i] = s;
    }
  }
};
template <int NDIM, int NS, int K, int ZMASK>
struct Fold<NDIM, NS, K, NS, ZMASK, double> {
  static __device__ __forceinline__ void eval(Ctx<NDIM, NS, double> &c, double (&out)[K]) {
    corner_series<NDIM, NS, K, ZMASK>(c, out);
  }
};
template <int NDIM, int NS, int K, int ZMASK>
struct Fold<NDIM, NS, K, NS, ZMASK, cd> {
  static __device__ __forceinline__ void eval(Ctx<NDIM, NS, cd> &c, cd (&out)[K]) {
    corner_series_cplx<NDIM, NS, K>(c, ZMASK, out);
  }
};

// ---- one sector at one point -----------------------------------------------------------------------------
// pt: this thread's per-point arrays in shared memory, element (a, j) at pt[(a*NDIM + j)*QMC_THREADS],
//     a = 0: t_j, 1: ln t_j, 2: 1/t_j.
template <int NDIM, int NS, int KMAX, class T>
__device__ __forceinline__ void sector_eval(const QmcLaunch &p, const QmcSectorHdr *h, const double *pt, T (&res)[KMAX + NS + 1],
                                            unsigned &cntImF, unsigned &cntReU) {
  constexpr int K = KMAX + NS + 1;
  constexpr bool CPLX = sizeof(T) == sizeof(cd);
  Ctx<NDIM, NS, T> c;
  c.hdr = h;
  c.coef = reinterpret_cast<const double *>(h + 1);
  c.exps = reinterpret_cast<const uint32_t *>(c.coef + (h->nU + h->nF));
  c.aU0 = p.aU0; c.aU1 = p.aU1; c.aF0 = p.aF0; c.aF1 = p.aF1;
  c.lambda = p.lambda;
  c.cntImF = 0; c.cntReU = 0;
  c.G0 = 1.0;
  c.L0 = 0.0;
#pragma unroll
  for (int k = 0; k < NDIM; ++k) {
    int j = h->perm[k];
    double tk = pt[(0 * NDIM + j) * QMC_THREADS];
    c.t[k] = tk;
    if (CPLX) c.invt_all[k] = pt[(2 * NDIM + j) * QMC_THREADS];
    if (k < NS) {
      double L = (double)h->beta[k] * pt[(1 * NDIM + j) * QMC_THREADS];
      c.invt[k] = pt[(2 * NDIM + j) * QMC_THREADS];
      c.invbeta[k] = 1.0 / (double)h->beta[k];
      c.cL[k][0] = 1.0;
#pragma unroll
      for (int q = 1; q < K; ++q) c.cL[k][q] = c.cL[k][q - 1] * L * (1.0 / q);
    } else {
      int a = h->alpha[k], b = h->beta[k];
      if (a) c.G0 *= ipow_pos(tk, a);
      if (b) c.L0 += (double)b * pt[(1 * NDIM + j) * QMC_THREADS];
    }
  }
  if (!CPLX) {
    // partial sums per group, then subset sums: PU[X] = sum of the monomials depending only on singular
    // variables inside X  =  U^(t with the singular variables outside X set to 0)
    int idx = 0;
#pragma unroll
    for (int g = 0; g < (1 << NS); ++g) {
      double s = 0.0;
      int n = h->cntU[g];
      for (int q = 0; q < n; ++q, ++idx) s += monomial<NDIM>(c.coef[idx], c.exps[idx], c.t);
      c.PU[g] = s;
    }
#pragma unroll
    for (int g = 0; g < (1 << NS); ++g) {
      double s = 0.0;
      int n = h->cntF[g];
      for (int q = 0; q < n; ++q, ++idx) s += monomial<NDIM>(c.coef[idx], c.exps[idx], c.t);
      c.PF[g] = s;
    }
#pragma unroll
    for (int b = 0; b < NS; ++b)
#pragma unroll
      for (int X = 0; X < (1 << NS); ++X)
        if (X >> b & 1) {
          c.PU[X] += c.PU[X ^ (1 << b)];
          c.PF[X] += c.PF[X ^ (1 << b)];
        }
  }
  Fold<NDIM, NS, K, 0, 0, T>::eval(c, res);
  cntImF += c.cntImF;
  cntReU += c.cntReU;
}

// ---- sectors with a variable of exponent alpha <= -2: the p >= 1 Taylor terms of Eq. 11, real path ----
// Product form over the variables V with alpha_b = -a_b <= -1 (the oracle evaluates the expanded double sum instead):
//   sum_k c_k eps^k = sum_{Z subset V}  sum_{p_b < a_b, b in Z}   [prod_{b in Z} t_b^{p_b}] g(t; eps)|_{t_Z = 0}
//                        prod_{b notin Z} t_b^{-a_b} e^{eps beta_b ln t_b}    prod_{b in Z} C_{b,p_b}(eps),
//   C_{b,p}(eps) = 1/(p + 1 - a_b + beta_b eps)  -  t_b^{p - a_b} e^{eps beta_b ln t_b}
// ([.] = Taylor coefficient; for a_b = 1 the factor C_{b,0} is B_b - A_b of the fold above).  g = G e^{eps Lambda} with
// G = G0 U^aU0 F^aF0, Lambda = aU1 ln U + aF1 ln F + L0.  Its Taylor coefficients in the variables of Z that have a_b > 1
// (at most two per sector, a_b <= QMC_MAXTAYLOR) come from truncated power-series arithmetic: U^ and F^ are polynomials, a
// power, reciprocal or logarithm of a series a0 + x is the series of the function in the nilpotent part x.
// A slow path by design (run-time loops, local arrays): such sectors come with propagator powers, not with the configs.
struct JetDims {
  int d0, d1;  // 1 + highest power kept of the first / second series variable (1 = no such variable)
};
struct Jet {
  double c[QMC_MAXTAYLOR * QMC_MAXTAYLOR];  // coefficient of x0^p0 x1^p1 at p0 + d0 * p1
};
__device__ __forceinline__ Jet jet_const(double v) {
  Jet r;
#pragma unroll
  for (int i = 0; i < QMC_MAXTAYLOR * QMC_MAXTAYLOR; ++i) r.c[i] = 0.0;
  r.c[0] = v;
  return r;
}
static __device__ __noinline__ Jet jet_mul(const JetDims d, const Jet &a, const Jet &b) {  // truncated product
  Jet r = jet_const(0.0);
  for (int p1 = 0; p1 < d.d1; ++p1)
    for (int p0 = 0; p0 < d.d0; ++p0) {
      const double av = a.c[p0 + d.d0 * p1];
      for (int q1 = 0; p1 + q1 < d.d1; ++q1)
        for (int q0 = 0; p0 + q0 < d.d0; ++q0) r.c[(p0 + q0) + d.d0 * (p1 + q1)] += av * b.c[q0 + d.d0 * q1];
    }
  return r;
}
// f(a0 + x) = sum_m co[m] x^m, co[m] = f^(m)(a0) / m!; x^m = 0 beyond m = (d0 - 1) + (d1 - 1)
static __device__ __noinline__ Jet jet_fn(const JetDims d, const Jet &a, const double (&co)[2 * QMC_MAXTAYLOR - 1]) {
  Jet x = a, xm = jet_const(1.0), r = jet_const(0.0);
  x.c[0] = 0.0;
  const int M = d.d0 + d.d1 - 2, n = d.d0 * d.d1;
  for (int m = 0; m <= M; ++m) {
    for (int i = 0; i < n; ++i) r.c[i] += co[m] * xm.c[i];
    if (m < M) xm = jet_mul(d, xm, x);
  }
  return r;
}
__device__ __forceinline__ Jet jet_recip(const JetDims d, const Jet &a) {  // sum_m (-1)^m x^m / a0^(m+1)
  double co[2 * QMC_MAXTAYLOR - 1];
  const double r0 = 1.0 / a.c[0];
  double v = r0;
#pragma unroll
  for (int m = 0; m < 2 * QMC_MAXTAYLOR - 1; ++m) {
    co[m] = v;
    v *= -r0;
  }
  return jet_fn(d, a, co);
}
__device__ __forceinline__ Jet jet_log(const JetDims d, const Jet &a) {  // ln a0 + sum_{m>=1} (-1)^(m+1) x^m / (m a0^m)
  double co[2 * QMC_MAXTAYLOR - 1];
  const double r0 = 1.0 / a.c[0];
  double v = r0;
  co[0] = log(a.c[0]);
#pragma unroll
  for (int m = 1; m < 2 * QMC_MAXTAYLOR - 1; ++m) {
    co[m] = v / (double)m;
    v *= -r0;
  }
  return jet_fn(d, a, co);
}
__device__ __forceinline__ Jet jet_ipow(const JetDims d, const Jet &a, int e) {  // integer power of either sign
  const Jet base = e >= 0 ? a : jet_recip(d, a);
  Jet r = jet_const(1.0);
  for (int q = 0; q < (e < 0 ? -e : e); ++q) r = jet_mul(d, r, base);
  return r;
}

// out[a], a = k + QMC_MAXSING: the coefficient of eps^k of the sector at this point (zero where the sector has none)
template <int NDIM, int KMAX>
__device__ __noinline__ void sector_eval_taylor(const QmcLaunch &p, const QmcSectorHdr *h, const double *pt,
                                                double (&out)[QMC_MAXSING + KMAX + 1]) {
  constexpr int KS = QMC_MAXSING + KMAX + 1;
  const double *coef = reinterpret_cast<const double *>(h + 1);
  const uint32_t *exps = reinterpret_cast<const uint32_t *>(coef + (h->nU + h->nF));
  const int nv = h->nsing, nU = h->nU, nT = h->nU + h->nF;
  double t[NDIM], lt[NDIM];
#pragma unroll
  for (int k = 0; k < NDIM; ++k) {
    const int j = h->perm[k];
    t[k] = pt[(0 * NDIM + j) * QMC_THREADS];
    lt[k] = pt[(1 * NDIM + j) * QMC_THREADS];
  }
  double G0 = 1.0, L0 = 0.0;  // regular variables
  for (int k = nv; k < NDIM; ++k) {
    G0 *= ipow_pos(t[k], h->alpha[k]);
    L0 += (double)h->beta[k] * lt[k];
  }
#pragma unroll
  for (int i = 0; i < KS; ++i) out[i] = 0.0;
  for (int Z = 0; Z < (1 << nv); ++Z) {
    int j0 = -1, j1 = -1, nz = 0;  // series variables: the members of Z with a_b > 1
    JetDims d{1, 1};
    double pref = 1.0, Lfree = L0;
    for (int b = 0; b < nv; ++b) {
      const int a = -h->alpha[b];
      if (Z >> b & 1) {
        ++nz;
        if (a > 1) {
          if (j0 < 0) {
            j0 = b;
            d.d0 = a;
          } else {
            j1 = b;
            d.d1 = a;
          }
        }
      } else {
        pref *= 1.0 / ipow_pos(t[b], a);  // untouched variable: t^-a e^{eps beta ln t}
        Lfree += (double)h->beta[b] * lt[b];
      }
    }
    // U^, F^ as series: a monomial puts  c prod_{k notin Z} t_k^{e_k}  on the coefficient of  prod_{b in Z} t_b^{e_b}
    Jet U = jet_const(0.0), F = jet_const(0.0);
    for (int mi = 0; mi < nT; ++mi) {
      const uint32_t w = exps[mi];
      double c = coef[mi];
      int idx = 0;
      bool keep = true;
#pragma unroll
      for (int k = 0; k < NDIM; ++k) {
        const int e = (w >> (4 * k)) & 15;
        if (k < nv && (Z >> k & 1)) {
          if (k == j0) {
            if (e >= d.d0) keep = false;
            idx += e;
          } else if (k == j1) {
            if (e >= d.d1) keep = false;
            idx += d.d0 * e;
          } else if (e) {
            keep = false;
          }
        } else {
          c *= ipow_pos(t[k], e);
        }
      }
      if (keep) (mi < nU ? U : F).c[idx] += c;
    }
    Jet W = jet_mul(d, jet_ipow(d, U, p.aU0), jet_ipow(d, F, p.aF0));
    const Jet lU = jet_log(d, U), lF = jet_log(d, F);
    Jet Lam;
    const int nj = d.d0 * d.d1;
    for (int i = 0; i < QMC_MAXTAYLOR * QMC_MAXTAYLOR; ++i) {
      W.c[i] *= G0;
      Lam.c[i] = i < nj ? (double)p.aU1 * lU.c[i] + (double)p.aF1 * lF.c[i] : 0.0;
    }
    Lam.c[0] += Lfree;
    // E[k] = W Lam^k / k!: the coefficient of eps^k of g times the regulators of the untouched variables
    Jet E[KS];
    E[0] = W;
    for (int k = 1; k < KS; ++k) {
      E[k] = jet_mul(d, E[k - 1], Lam);
      const double rk = 1.0 / (double)k;
      for (int i = 0; i < nj; ++i) E[k].c[i] *= rk;
    }
    for (int p1 = 0; p1 < d.d1; ++p1)
      for (int p0 = 0; p0 < d.d0; ++p0) {
        double ser[KS];  // eps^nz times the term: coefficients of eps^0 .. eps^(KS-1)
        for (int k = 0; k < KS; ++k) ser[k] = E[k].c[p0 + d.d0 * p1];
        for (int b = 0; b < nv; ++b) {
          if (!(Z >> b & 1)) continue;
          const int a = -h->alpha[b], pb = b == j0 ? p0 : (b == j1 ? p1 : 0), q = a - 1 - pb;
          const double beta = (double)h->beta[b];
          double cc[KS];  // eps C_{b,p}(eps)
          if (q == 0) {  // the pole 1/(beta eps)
            cc[0] = 1.0 / beta;
            for (int m = 1; m < KS; ++m) cc[m] = 0.0;
          } else {  // 1/(-q + beta eps) = -(1/q) sum_m (beta eps / q)^m
            cc[0] = 0.0;
            double gq = -1.0 / (double)q;
            for (int m = 1; m < KS; ++m) {
              cc[m] = gq;
              gq *= beta / (double)q;
            }
          }
          double term = 1.0 / ipow_pos(t[b], a - pb);  // - t^(p-a) e^{eps beta ln t}
          const double Lb = beta * lt[b];
          for (int m = 0; m + 1 < KS; ++m) {
            cc[m + 1] -= term;
            term *= Lb / (double)(m + 1);
          }
          double r[KS];
          for (int i = 0; i < KS; ++i) r[i] = 0.0;
          for (int i = 0; i < KS; ++i)
            for (int jx = 0; i + jx < KS; ++jx) r[i + jx] += ser[i] * cc[jx];
          for (int i = 0; i < KS; ++i) ser[i] = r[i];
        }
        for (int i = 0; i < KS; ++i) {
          const int k = i - nz;  // order of eps
          if (k <= KMAX) out[k + QMC_MAXSING] += pref * ser[i];
        }
      }
  }
}

// ---- pole extraction by integration by parts (Eq. 13; qmc_options.pole_extraction = 1), real path -----
// Eq. 13 applied a_b = -alpha_b times to every variable with alpha_b <= -1:
//   int_0^1 dt t^(-a + beta eps) f = sum_{r<a} (-1)^r f^(r)(1) / prod_{s<=r} (s+1-a + beta eps)
//                                  + (-1)^a / prod_{s<a} (s+1-a + beta eps)  int_0^1 dt t^(beta eps) f^(a)(t),
// the operators of several variables multiplied out: a variable is taken at t_b = 1 with an order r_b < a_b, or keeps its
// integral with order a_b.  f = G e^{eps Lambda}; its mixed derivatives are p! times the Taylor coefficients around the
// point, from truncated power series in ALL variables with alpha_b <= -1 (at most QMC_IBP_JET coefficients).
struct JetN {
  double c[QMC_IBP_JET];
};
struct JetNShape {
  int n, total;                                  // coefficients; sum of the orders kept
  unsigned char dig[QMC_IBP_JET][QMC_MAXSING];   // index -> power of each variable
  unsigned char dim[QMC_MAXSING], stride[QMC_MAXSING];
};
__device__ __forceinline__ JetN jetn_const(double v) {
  JetN r;
#pragma unroll
  for (int i = 0; i < QMC_IBP_JET; ++i) r.c[i] = 0.0;
  r.c[0] = v;
  return r;
}
static __device__ __noinline__ JetN jetn_mul(const JetNShape &sh, const JetN &a, const JetN &b) {
  JetN r = jetn_const(0.0);
  for (int i = 0; i < sh.n; ++i)
    for (int k = 0; k < sh.n; ++k) {
      int idx = 0;
      bool keep = true;
#pragma unroll
      for (int v = 0; v < QMC_MAXSING; ++v) {
        const int pw = sh.dig[i][v] + sh.dig[k][v];
        if (pw >= sh.dim[v]) keep = false;
        idx += pw * sh.stride[v];
      }
      if (keep) r.c[idx] += a.c[i] * b.c[k];
    }
  return r;
}
// f(a0 + x) = sum_m co[m] x^m, x^m = 0 beyond m = total (<= QMC_IBP_JET - 1 orders)
static __device__ __noinline__ JetN jetn_fn(const JetNShape &sh, const JetN &a, const double *co) {
  JetN x = a, xm = jetn_const(1.0), r = jetn_const(0.0);
  x.c[0] = 0.0;
  for (int m = 0; m <= sh.total; ++m) {
    for (int i = 0; i < sh.n; ++i) r.c[i] += co[m] * xm.c[i];
    if (m < sh.total) xm = jetn_mul(sh, xm, x);
  }
  return r;
}
__device__ __forceinline__ JetN jetn_recip(const JetNShape &sh, const JetN &a) {
  double co[QMC_IBP_JET];
  const double r0 = 1.0 / a.c[0];
  double v = r0;
  for (int m = 0; m <= sh.total; ++m) {
    co[m] = v;
    v *= -r0;
  }
  return jetn_fn(sh, a, co);
}
__device__ __forceinline__ JetN jetn_log(const JetNShape &sh, const JetN &a) {
  double co[QMC_IBP_JET];
  const double r0 = 1.0 / a.c[0];
  double v = r0;
  co[0] = log(a.c[0]);
  for (int m = 1; m <= sh.total; ++m) {
    co[m] = v / (double)m;
    v *= -r0;
  }
  return jetn_fn(sh, a, co);
}
__device__ __forceinline__ JetN jetn_ipow(const JetNShape &sh, const JetN &a, int e) {
  const JetN base = e >= 0 ? a : jetn_recip(sh, a);
  JetN r = jetn_const(1.0);
  for (int q = 0; q < (e < 0 ? -e : e); ++q) r = jetn_mul(sh, r, base);
  return r;
}

template <int NDIM, int KMAX>
__device__ __noinline__ void sector_eval_ibp(const QmcLaunch &p, const QmcSectorHdr *h, const double *pt,
                                             double (&out)[QMC_MAXSING + KMAX + 1]) {
  constexpr int KS = QMC_MAXSING + KMAX + 1;
  const double *coef = reinterpret_cast<const double *>(h + 1);
  const uint32_t *exps = reinterpret_cast<const uint32_t *>(coef + (h->nU + h->nF));
  const int nv = h->nsing, nU = h->nU, nT = h->nU + h->nF;
  double t[NDIM], lt[NDIM];
#pragma unroll
  for (int k = 0; k < NDIM; ++k) {
    const int j = h->perm[k];
    t[k] = pt[(0 * NDIM + j) * QMC_THREADS];
    lt[k] = pt[(1 * NDIM + j) * QMC_THREADS];
  }
  double G0 = 1.0, L0 = 0.0;
  for (int k = nv; k < NDIM; ++k) {
    G0 *= ipow_pos(t[k], h->alpha[k]);
    L0 += (double)h->beta[k] * lt[k];
  }
#pragma unroll
  for (int i = 0; i < KS; ++i) out[i] = 0.0;
  for (int B = 0; B < (1 << nv); ++B) {  // B: the variables taken at the boundary t_b = 1
    JetNShape sh;
    double tau[QMC_MAXSING], Lint = L0;
    sh.n = 1;
    sh.total = 0;
    for (int b = 0; b < QMC_MAXSING; ++b) {
      int ord = 0;
      tau[b] = 1.0;
      if (b < nv) {
        const int a = -h->alpha[b];
        const bool atone = B >> b & 1;
        ord = atone ? a - 1 : a;
        if (!atone) {
          tau[b] = t[b];
          Lint += (double)h->beta[b] * lt[b];  // the factor t_b^(beta_b eps) under the integral
        }
      }
      sh.dim[b] = (unsigned char)(ord + 1);
      sh.stride[b] = (unsigned char)sh.n;
      sh.n *= ord + 1;
      sh.total += ord;
    }
    for (int i = 0; i < sh.n; ++i)
      for (int b = 0; b < QMC_MAXSING; ++b) sh.dig[i][b] = (unsigned char)((i / sh.stride[b]) % sh.dim[b]);
    // U^, F^ around the point: (tau + d)^e = sum_p C(e, p) tau^(e-p) d^p
    JetN U = jetn_const(0.0), F = jetn_const(0.0);
    for (int mi = 0; mi < nT; ++mi) {
      const uint32_t w = exps[mi];
      double c0 = coef[mi];
      for (int k = nv; k < NDIM; ++k) c0 *= ipow_pos(t[k], (w >> (4 * k)) & 15);
      for (int i = 0; i < sh.n; ++i) {
        double c = c0;
        bool keep = true;
        for (int b = 0; b < nv; ++b) {
          const int e = (w >> (4 * b)) & 15, pw = sh.dig[i][b];
          if (pw > e) {
            keep = false;
            break;
          }
          double bin = 1.0;
          for (int q = 0; q < pw; ++q) bin = bin * (double)(e - q) / (double)(q + 1);
          c *= bin * ipow_pos(tau[b], e - pw);
        }
        if (keep) (mi < nU ? U : F).c[i] += c;
      }
    }
    JetN W = jetn_mul(sh, jetn_ipow(sh, U, p.aU0), jetn_ipow(sh, F, p.aF0));
    const JetN lU = jetn_log(sh, U), lF = jetn_log(sh, F);
    JetN Lam = jetn_const(0.0);
    for (int i = 0; i < sh.n; ++i) {
      W.c[i] *= G0;
      Lam.c[i] = (double)p.aU1 * lU.c[i] + (double)p.aF1 * lF.c[i];
    }
    Lam.c[0] += Lint;
    JetN E[KS];  // E[k] = W Lam^k / k!
    E[0] = W;
    for (int k = 1; k < KS; ++k) {
      E[k] = jetn_mul(sh, E[k - 1], Lam);
      const double rk = 1.0 / (double)k;
      for (int i = 0; i < sh.n; ++i) E[k].c[i] *= rk;
    }
    for (int i = 0; i < sh.n; ++i) {  // derivative orders: r_b < a_b at the boundary, exactly a_b under the integral
      bool use = true;
      for (int b = 0; b < nv; ++b)
        if (!(B >> b & 1) && sh.dig[i][b] != -h->alpha[b]) use = false;
      if (!use) continue;
      double scalar = 1.0, ser[KS];
      int npole = 0;
      for (int k = 0; k < KS; ++k) ser[k] = E[k].c[i];
      for (int b = 0; b < nv; ++b) {
        const int a = -h->alpha[b], pw = sh.dig[i][b];
        const double beta = (double)h->beta[b];
        for (int q = 2; q <= pw; ++q) scalar *= (double)q;  // derivative = Taylor coefficient times p!
        if (pw & 1) scalar = -scalar;
        const int smax = pw < a - 1 ? pw : a - 1;
        for (int sf = 0; sf <= smax; ++sf) {  // 1 / (s+1-a + beta eps)
          const int c = sf + 1 - a;
          if (c == 0) {
            scalar *= 1.0 / beta;
            ++npole;
          } else {  // (1/c) sum_m (-beta eps / c)^m
            double r[KS];
            for (int k = 0; k < KS; ++k) r[k] = 0.0;
            for (int k = 0; k < KS; ++k) {
              double gm = 1.0 / (double)c;
              for (int m = 0; k + m < KS; ++m) {
                r[k + m] += ser[k] * gm;
                gm *= -beta / (double)c;
              }
            }
            for (int k = 0; k < KS; ++k) ser[k] = r[k];
          }
        }
      }
      for (int k = 0; k < KS; ++k) {
        const int order = k - npole;
        if (order <= KMAX) out[order + QMC_MAXSING] += scalar * ser[k];
      }
    }
  }
}

__device__ __forceinline__ bool finite_all(double v) { return fabs(v) <= 1.79769313486231570e308; }
__device__ __forceinline__ bool finite_all(cd v) { return finite_all(v.re) && finite_all(v.im); }

// TMA bulk copy global -> shared, completion on an mbarrier (sm_90+; SASS: UBLKCP)
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
  unsigned d = (unsigned)__cvta_generic_to_shared(dst), b = (unsigned)__cvta_generic_to_shared(bar);
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(d),
               "l"(src), "r"(bytes), "r"(b)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
  unsigned a = (unsigned)__cvta_generic_to_shared(bar), ok = 0;
  while (!ok) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(a), "r"(parity)
        : "memory");
  }
}

// deterministic block sum: warp shuffle tree, then pairwise tree over the warp results in shared memory
__device__ __forceinline__ double block_sum(double v, double *scratch /*[QMC_THREADS/32]*/) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) scratch[wid] = v;
  __syncthreads();
  double r = 0.0;
  if (wid == 0) {
    r = (lane < QMC_THREADS / 32) ? scratch[lane] : 0.0;
#pragma unroll
    for (int o = (QMC_THREADS / 64); o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
  }
  return r;  // valid in thread 0
}

}  // namespace qmcdev

// ================================================================================================
#ifndef QMC_V1_MIN_BLOCKS
#define QMC_V1_MIN_BLOCKS 1
#endif
// NSCAP: largest number of singular variables of any sector of the tables this instantiation serves (the code of the
// larger cases is not generated: the complex instantiation with NSCAP = 1 is a fraction of the size of NSCAP = 4)
// TAYLOR: the instantiation that also serves sectors with alpha_j <= -2 (header flag 2; real path only)
template <int NDIM, int KMAX, bool CPLX, int NSCAP, bool TAYLOR = false>
__global__ void __launch_bounds__(QMC_THREADS, QMC_V1_MIN_BLOCKS) qmc_eval_kernel(const QmcLaunch p) {
  using namespace qmcdev;
  typedef typename std::conditional<CPLX, cd, double>::type T;
  constexpr int NACC = QMC_MAXSING + KMAX + 1;  // accumulator a <-> order a - QMC_MAXSING
  constexpr int NC = CPLX ? 2 : 1;
  constexpr int SMAX0 = NDIM < QMC_MAXSING ? NDIM : QMC_MAXSING;
  constexpr int SMAX = SMAX0 < NSCAP ? SMAX0 : NSCAP;

  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x;
  const int chunk = blockIdx.y;
  const int s0 = p.sec_begin + chunk * p.sec_per_chunk;
  const int s1 = min(s0 + p.sec_per_chunk, p.sec_end);
  const int nsec = s1 - s0;

  // shared memory carve-up
  unsigned char *tab = smem;                                                   // table chunk
  uint32_t *soff = reinterpret_cast<uint32_t *>(smem + p.tab_smem_bytes);     // [nsec+1] offsets
  size_t o = p.tab_smem_bytes + (((size_t)(p.sec_per_chunk + 1) * 4 + 15) & ~(size_t)15);
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem + o);
  o += 16;
  double *shf = reinterpret_cast<double *>(smem + o);                          // [m][NDIM]
  o += (((size_t)p.m * NDIM * 8) + 15) & ~(size_t)15;
  double *scratch = reinterpret_cast<double *>(smem + o);                      // [QMC_THREADS/32]
  o += (QMC_THREADS / 32) * 8;
  double *ptbase = reinterpret_cast<double *>(smem + o);                       // [3][NDIM][QMC_THREADS]
  o += (size_t)3 * NDIM * QMC_THREADS * 8;
  double *sacc = reinterpret_cast<double *>(smem + o);                         // persec: [nsec][NACC*NC][QMC_THREADS]
  double *pt = ptbase + tid;

  // stage the chunk's tables: one TMA bulk copy, completion on an mbarrier
  const uint32_t g0 = p.secoff[s0], g1 = p.secoff[s1];
  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    mbar_expect_tx(bar, g1 - g0);
    tma_bulk_g2s(tab, p.image + g0, g1 - g0, bar);
  }
  for (int i = tid; i <= nsec; i += QMC_THREADS) soff[i] = p.secoff[s0 + i] - g0;
  for (int i = tid; i < p.m * NDIM; i += QMC_THREADS) shf[i] = p.shifts[i];
  mbar_wait(bar, 0);
  __syncthreads();

  const uint32_t N = p.N;
  const double dN = (double)N;
  const uint32_t stride = gridDim.x * QMC_THREADS;
  uint32_t dz[NDIM];
#pragma unroll
  for (int j = 0; j < NDIM; ++j) dz[j] = (uint32_t)(((uint64_t)stride * p.zeff[j]) % N);

  unsigned cntImF = 0, cntReU = 0, cntNonFinite = 0, cntBoundary = 0;

  for (int kap = 0; kap < p.m; ++kap) {
    T acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = Num<T>::zero();
    if (p.persec)
      for (int i = 0; i < nsec * NACC * NC; ++i) sacc[(size_t)i * QMC_THREADS + tid] = 0.0;

    uint32_t cidx = blockIdx.x * QMC_THREADS + tid;
    uint32_t r[NDIM];
#pragma unroll
    for (int j = 0; j < NDIM; ++j) r[j] = (uint32_t)((p.off[j] + (uint64_t)cidx * p.zeff[j]) % N);

    for (; cidx < p.count; cidx += stride) {
      // S1-S3: lattice point (Eq. 17), shift + wrap (Eq. 18), periodising transform (Eq. 21)
      double w = 1.0;
      bool inside = true;
#pragma unroll
      for (int j = 0; j < NDIM; ++j) {
        double u = (double)r[j] / dN;
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
        if (!(y > 0.0) || !(tj > 0.0)) inside = false;
        pt[(0 * NDIM + j) * QMC_THREADS] = tj;
        pt[(1 * NDIM + j) * QMC_THREADS] = log(tj);
        pt[(2 * NDIM + j) * QMC_THREADS] = 1.0 / tj;
        uint32_t rn = r[j] + dz[j];  // r, dz < N < 2^31: no wrap
        r[j] = rn >= N ? rn - N : rn;
      }
      if (!inside) {
        if (chunk == 0) ++cntBoundary;
        continue;
      }
      // S4-S6: all sectors of the chunk at this point
      for (int si = 0; si < nsec; ++si) {
        const QmcSectorHdr *h = reinterpret_cast<const QmcSectorHdr *>(tab + soff[si]);
        const int ns = h->nsing;
        T contrib[NACC];
#pragma unroll
        for (int a = 0; a < NACC; ++a) contrib[a] = Num<T>::zero();
        bool fin = true;
#define QMC_CASE(NS_)                                                                   \
  case NS_: {                                                                           \
    if (NS_ <= SMAX) {                                                                  \
      constexpr int NSC = NS_ <= SMAX ? NS_ : 0;                                        \
      T res[KMAX + NSC + 1];                                                            \
      sector_eval<NDIM, NSC, KMAX, T>(p, h, pt, res, cntImF, cntReU);                   \
      _Pragma("unroll") for (int i = 0; i < KMAX + NSC + 1; ++i) {                      \
        fin = fin && finite_all(res[i]);                                                \
        contrib[QMC_MAXSING - NSC + i] = res[i];                                        \
      }                                                                                 \
    }                                                                                   \
  } break;
        if (TAYLOR && !CPLX && (p.ibp ? ns > 0 : (h->flags & 2) != 0)) {
          if constexpr (TAYLOR && !CPLX) {
            double res[NACC];
            if (p.ibp)
              sector_eval_ibp<NDIM, KMAX>(p, h, pt, res);
            else
              sector_eval_taylor<NDIM, KMAX>(p, h, pt, res);
#pragma unroll
            for (int i = 0; i < NACC; ++i) {
              fin = fin && finite_all(res[i]);
              contrib[i] = res[i];
            }
          }
        } else
        switch (ns) {
          QMC_CASE(0)
          QMC_CASE(1)
          QMC_CASE(2)
          QMC_CASE(3)
          QMC_CASE(4)
          default:
            break;
        }
#undef QMC_CASE
        if (!fin) {
          ++cntNonFinite;
          continue;
        }
        if (!p.persec) {
#pragma unroll
          for (int a = 0; a < NACC; ++a) acc[a] = acc[a] + Num<T>::scale(w, contrib[a]);
        } else {
          double *sa = sacc + ((size_t)si * NACC * NC) * QMC_THREADS + tid;
#pragma unroll
          for (int a = 0; a < NACC; ++a) {
            if (CPLX) {
              const cd *cc = reinterpret_cast<const cd *>(&contrib[a]);
              sa[(size_t)(2 * a) * QMC_THREADS] += w * cc->re;
              sa[(size_t)(2 * a + 1) * QMC_THREADS] += w * cc->im;
            } else {
              sa[(size_t)a * QMC_THREADS] += w * *reinterpret_cast<const double *>(&contrib[a]);
            }
          }
        }
      }
    }

    // S7: block reduction -> one partial per (chunk | sector, shift, block)
    if (!p.persec) {
      double *dst = p.partial + (((size_t)chunk * p.m + kap) * gridDim.x + blockIdx.x) * (NACC * NC);
#pragma unroll
      for (int a = 0; a < NACC; ++a) {
        if (CPLX) {
          const cd *cc = reinterpret_cast<const cd *>(&acc[a]);
          double sr = block_sum(cc->re, scratch);
          double si = block_sum(cc->im, scratch);
          if (tid == 0) {
            dst[2 * a] = sr;
            dst[2 * a + 1] = si;
          }
        } else {
          double sr = block_sum(*reinterpret_cast<const double *>(&acc[a]), scratch);
          if (tid == 0) dst[a] = sr;
        }
      }
    } else {
      for (int si = 0; si < nsec; ++si) {
        double *dst = p.partial + (((size_t)(s0 - p.sec_begin + si) * p.m + kap) * gridDim.x + blockIdx.x) * (NACC * NC);
        for (int a = 0; a < NACC * NC; ++a) {
          double v = block_sum(sacc[((size_t)si * NACC * NC + a) * QMC_THREADS + tid], scratch);
          if (tid == 0) dst[a] = v;
        }
      }
    }
  }

  // counters (integers: order-independent)
  unsigned c4[4] = {cntImF, cntReU, cntNonFinite, cntBoundary};
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    unsigned v = c4[q];
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) v += __shfl_down_sync(0xffffffffu, v, o2);
    if ((tid & 31) == 0 && v) atomicAdd(p.counters + q, (unsigned long long)v);
  }
}
