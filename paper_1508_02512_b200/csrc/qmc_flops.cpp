// qmc_flop_model: algorithmic FP64 operation count of the evaluation, from the sector tables (host only).
//
// This is the denominator-side bookkeeping of the roofline: the arithmetic the
// product-form evaluation of Eqs. 9-12 + 14 needs, counted at the source level of the
// scheme the kernels implement, with DFMA = 2 and DADD = DMUL = 1 and fixed costs for the library sequences
// (fast paths of the CUDA 12.9 sm_100a FP64 routines, counted in SASS; the kernels' own routines in brackets):
//   division: 7 DFMA + 2 DMUL = 16      atan2: division + 19 DFMA polynomial + fix-ups = 60
//   [table logarithm, 64 entries: 8 DFMA + DMUL + DADD = 18]      [reciprocal: MUFU seed + one cubic step, 3 DFMA = 6]
// Integer work (lattice index arithmetic, table decoding) and comparisons count as zero.  The count is
// cross-checked against Nsight Compute's executed DFMA/DADD/DMUL thread-instruction counters (profiles/).
#include <algorithm>
#include <cstdlib>

#include "../../include/qmc_feynman.h"
#include "qmc_tables.h"

namespace {
const double F_LOG = 44.0, F_RCP = 10.0, F_ATAN2 = 60.0;
const double F_CMUL = 6.0, F_CADD = 2.0;                  // complex multiply (4 mul + 2 add), complex add
const double F_CINV = 3.0 + F_RCP + 2.0;                  // |a|^2, reciprocal, two scalings
const double F_CLOG = 3.0 + F_LOG + 1.0 + F_ATAN2;        // 0.5 log(|a|^2), atan2

int degree(const QmcMono &m, int n) {
  int d = 0;
  for (int j = 0; j < n; ++j) d += m.e[j];
  return d;
}
}  // namespace

extern "C" int qmc_flop_model(const qmc_tables *t, int32_t sector_begin, int32_t sector_end, double *flops_point,
                              double *flops_sectors, int64_t *corners) {
  if (!t) return QMC_EINVAL;
  const int n = t->n, nsec = (int)t->sectors.size();
  const int sb = sector_begin, se = sector_end > 0 ? sector_end : nsec;
  if (sb < 0 || se > nsec || sb >= se) return QMC_EINVAL;
  const bool cplx = t->lambda > 0.0;
  // Tables that only the generic kernel runs (propagator powers, sectors with alpha <= -2, integration by parts: t->generic_only)
  // are counted with the scheme of the table-driven kernels and every variable with alpha <= -1 as a singular one: a lower bound
  // of what their slow paths (power-series arithmetic) execute.  No reported number uses the model on such tables.
  // S1-S3, once per (point, shift): u = r/N (IEEE division), y = u + Delta (wrap), t = y^2 (3 - 2y), w *= 6 y (1 - y),
  // ln t (table logarithm)
  // (r / N as r * RN(1/N) with one FMA correction, 5 flops, on both paths)
  double per_point = n * (5.0 + 2.0 + 4.0 + 4.0 + 18.0);
  if (!cplx)  // the chunks' product slots, once per point and chunk touched
    for (const Qmc2Chunk &c : t->chunks)
      if (c.sec_end > sb && c.sec_begin < se) per_point += (double)(c.nslots - (2 * n + 2 + c.nconst));
  double per_sectors = 0.0;
  int64_t ncorners = 0;
  const int eU = std::abs(t->aU0), eF = std::abs(t->aF0);
  for (int si = sb; si < se; ++si) {
    const QmcSector &s = t->sectors[si];
    const int ns = s.nsing, K = t->kmax + ns + 1, nc = 1 << ns;
    double f = 0.0;
    // per-sector set-up: series (beta_j ln t_j)^p / p! of the singular variables, regular-variable factor and log
    for (int j = 0; j < n; ++j) {
      if (s.alpha[j] <= -1) {
        f += 1.0 + 2.0 * (K - 1);
      } else {
        if (s.alpha[j]) f += s.alpha[j];
        if (s.beta[j]) f += 2.0;
      }
    }
    if (!cplx) {
      // version-4 scheme (qmc_kernels4.cuh, qmc_image4.cpp).  A monomial record slot * slot accumulated onto its group is
      // one DFMA = 2; the first record of a group is one DMUL = 1.  The 0 * 0 stand-ins of empty groups and the sentinels
      // are not counted: they are the kernel's overhead, not the method's arithmetic.
      auto pow_muls = [](int e) {  // multiplications of x^e by repeated squaring (ipow_c), e >= 0
        int c = 0;
        for (int q = e; q > 1; q >>= 1) c += 1 + (q & 1);
        return (double)c;
      };
      const double F_RCP2 = 6.0;    // MUFU seed + 3 DFMA
      const double F_LOG2 = 18.0;   // table-driven: 9 DFMA
      int nL0 = 0;
      for (int j = 0; j < n; ++j)
        if (s.alpha[j] != -1 && s.beta[j]) ++nL0;
      const int nlocal = t->tab4.empty() ? 0 : (int)((t->tab4[(size_t)t->secoff4[si] * 4] >> 16) & 255u);
      f = 1.0 * nlocal;                        // sector-local product slots
      f += 3.0 + 2.0 * nL0;                    // G0 = c * slot * slot, times the weight; L0 = constant + sum beta_j ln t_j (FMAs)
      if (ns > 0) f += (ns - 1) + F_RCP2 + 1.0;  // 1 / prod t_k of the singular variables, times G0
      {
        int pos[QMC_MAXDIM], k = 0;
        for (int j = 0; j < n; ++j) pos[j] = s.alpha[j] <= -1 ? k++ : -1;
        for (int which = 0; which < 2; ++which) {
          unsigned seen = 0;
          for (const QmcMono &m : (which ? s.F : s.U)) {
            int g = 0;
            for (int j = 0; j < n; ++j)
              if (m.e[j] && pos[j] >= 0) g |= 1 << pos[j];
            f += (seen >> g & 1u) ? 2.0 : 1.0;   // first record of a group: DMUL; further records: DFMA
            seen |= 1u << g;
          }
        }
      }
      f += (double)ns * nc;                            // subset sums: ns * 2^(ns-1) additions per polynomial
      for (int j = 0; j < n; ++j)
        if (s.alpha[j] <= -1) f += 2.0 + 2.0 * std::max(0, K - 3);   // t_j / beta_j, beta_j ln t_j, then (.)^p / p! for p = 2 .. K-2
      // W = U^aU0 F^aF0 and the argument U^aU1 F^aF1 of the logarithm from U, 1/F (1/U), a = U/F (corner_powers)
      const int P = std::min(t->aU1, -t->aF1), Q = (t->aU0 > 0 && t->aF0 < 0) ? std::min(t->aU0, -t->aF0) : 0;
      auto factors_w = [&]() {
        double c = 0.0;
        int terms = 0;
        if (Q > 0) { c += pow_muls(Q); ++terms; }
        if (t->aU0 - Q > 0) { c += pow_muls(t->aU0 - Q); ++terms; }
        if (t->aU0 < 0) { c += pow_muls(-t->aU0); ++terms; }
        if (-t->aF0 - Q > 0) { c += pow_muls(-t->aF0 - Q); ++terms; }
        if (t->aF0 > 0) { c += pow_muls(t->aF0); ++terms; }
        return c + std::max(0, terms - 1);
      };
      auto factors_arg = [&]() {
        double c = pow_muls(P) - (Q > 0 ? pow_muls(std::min(P, Q)) : 0.0);  // powers of a shared with W
        int terms = 1;
        if (t->aU1 - P > 0) { c += pow_muls(t->aU1 - P); ++terms; }
        if (-t->aF1 - P > 0) { c += pow_muls(-t->aF1 - P); ++terms; }
        return c + (terms - 1);
      };
      for (int Z = 0; Z < nc; ++Z) {
        const int len = t->kmax + __builtin_popcount(Z) + 1;       // leaf window
        f += F_RCP2 + (t->aU0 < 0 ? F_RCP2 : 0.0);
        const bool need_a = Q > 0 || len > 1;
        f += (need_a ? 1.0 : 0.0) + factors_w();
        if (len > 1) f += factors_arg() + F_LOG2 + 1.0 + 2.0 * (len - 1) - 1.0;   // logarithm + L0; W Lambda^p / p!: two multiplications per term, one for p = 1
      }
      // fold: merge at level l with Z the choices of the levels below l: (len-1) differences, one product, len (len-1) / 2 FMAs
      for (int l = 0; l < ns; ++l)
        for (int Z = 0; Z < (1 << l); ++Z) {
          const int len = ns - l + t->kmax + __builtin_popcount(Z) + 1;
          f += (len - 1) + 1.0 + (double)len * (len - 1);
        }
      f += 2.0 * K;  // weight and accumulate
    } else {
      // version-5 scheme (qmc_kernels5.cuh)
      auto pow_muls = [](int e) {
        int c = 0;
        for (int q = e; q > 1; q >>= 1) c += 1 + (q & 1);
        return (double)c;
      };
      const double F_LOG2 = 18.0, F_CLOG3 = 3.0 + F_LOG2 + 1.0 + F_ATAN2;  // 64-entry table logarithm of |a|^2, atan2
      int pos_of[QMC_MAXDIM], kk = 0;
      for (int j = 0; j < n; ++j) pos_of[j] = (s.alpha[j] <= -1) ? kk++ : -1;
      int nprod_c = 0;  // complex product slots of the sector's chunk
      for (size_t ci = 0; ci < t->chunks3.size(); ++ci)
        if (si >= t->chunks3[ci].sec_begin && si < t->chunks3[ci].sec_end) nprod_c = t->chunk3_nslots_c[ci] - (n + 1);
      int nL0 = 0;
      for (int j = 0; j < n; ++j) {
        if (s.alpha[j] != -1 && s.beta[j]) ++nL0;
      }
      f = 3.0 * (1 + nL0);
      if (ns > 0) f += (ns - 1) + 6.0 + 1.0;   // 1 / prod t_k of the singular variables, onto G0
      for (int j = 0; j < n; ++j)
        if (s.alpha[j] <= -1) f += 2.0 + 2.0 * std::max(0, K - 3);   // t_k / beta_k, beta_k ln t_k, (.)^p / p!
      // record streams of all corners (derivative polynomials, U^(z), F^(z)): constants 0, real one-factor record 2 (an FMA),
      // real two-factor 3, complex one-factor 4, complex two-factor 10 -- counted by the table builder (qmc_image3.cpp)
      if ((size_t)si < t->rec_flops5.size()) f += t->rec_flops5[si];
      for (int Z = 0; Z < nc; ++Z) {
        auto in_Z = [&](int j) { return pos_of[j] >= 0 && (Z >> pos_of[j] & 1); };
        int nfree = 0;
        for (int j = 0; j < n; ++j)
          if (!in_Z(j)) ++nfree;
        f += n * 5.0 + (double)nfree * nfree * 3.0 + nfree * 3.0;  // rho, z, Jacobian entries
        for (int col = 0; col < n; ++col) {                         // elimination of the n x n complex matrix (no pivoting)
          f += F_CMUL;
          const int rem = n - col - 1;
          if (rem > 0) f += F_CINV + rem * (F_CMUL + rem * (F_CMUL + F_CADD));   // natural order, no pivot search
          // first elimination step: the off-diagonal entries of J = 1 + iB are purely imaginary, a product with one of
          // them is 2 multiplications, not 6 (ptxas folds the zeros; checked against ncu's executed FP64 counters)
          if (col == 0) f -= 4.0 * rem + 4.0 * rem * rem;
        }
        f += 6.0 * nprod_c;                                         // complex slot program
        f += 2.0;  // G0 det
        for (int j = 0; j < n; ++j)
          if (!in_Z(j)) f += std::abs(s.alpha[j]) * F_CMUL;
        f += (pow_muls(eU) + (eU ? 1 : 0) + pow_muls(eF) + (eF ? 1 : 0)) * F_CMUL + F_CINV + F_CMUL;
        if (t->kmax + __builtin_popcount(Z) > 0) {   // Lambda: only where the series window is longer than one term
          // ONE complex logarithm: Q = U^aU1 F^aF1 prod_j rho_j^beta_j by complex products (numerator over denominator), ln Q,
          // the winding number from single-precision phase estimates (no FP64) added by one FMA, + L0
          double qmuls = pow_muls(std::max(t->aU1, 0)) + pow_muls(std::max(-t->aF1, 0));
          for (int j = 0; j < n; ++j) qmuls += std::abs(s.beta[j]);
          f += qmuls * F_CMUL + F_CINV + F_CMUL + F_CLOG3 + 2.0;
        }
        f += (t->kmax + __builtin_popcount(Z)) * 8.0;               // series
      }
      for (int l = 0; l < ns; ++l)
        for (int Z = 0; Z < (1 << l); ++Z) {
          const int len = ns - l + t->kmax + __builtin_popcount(Z) + 1;
          f += 2.0 * (len - 1) + 2.0 + 2.0 * len * (len - 1);
        }
      f += 4.0 * K;
    }
    per_sectors += f;
    ncorners += nc;
  }
  if (flops_point) *flops_point = per_point;
  if (flops_sectors) *flops_sectors = per_sectors;
  if (corners) *corners = ncorners;
  return QMC_OK;
}
