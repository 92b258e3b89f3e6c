// Evaluation kernel of the real (Euclidean) path, "version 4", sm_100a.  Steps S1-S7 of DESIGN.md.
//
// One thread = one lattice point at a time.  Per point the thread fills its column of a shared-memory slot table
// (t_j, ln t_j, 1, 0, coefficient constants, then the chunk's product slots chosen by the byte-pair-encoding pass of
// qmc_image4.cpp); a monomial of U^ or F^ is then ONE 8-byte record: slot * slot, accumulated with one FMA (the
// coefficient lives in a slot).  Per sector with s singular variables:
//   1. partial sums of U^, F^ per group (= set of singular variables a monomial depends on), subset sums -> the values
//      at all 2^s corners t^Z of the subtraction (Eqs. 11-12) from one pass over the records;
//   2. per corner: W_Z = U^aU0 F^aF0 with one reciprocal, Lambda_Z = ln(U^aU1 F^aF1) + L0 with ONE table-driven
//      logarithm (exponents are compile-time: they depend only on the dimension and the loop number, Eq. 6);
//   3. the product form of the eps-expanded subtracted integrand, folded one singular variable at a time with series
//      windows of exactly the needed length (qmc_fold.cuh); the common factor G0' = c prod_reg t^alpha prod_sing 1/t
//      multiplies the weight once per sector.
// The chunk's slot program and the sector tables are part of the KERNEL PARAMETER BLOCK (constant bank 0, layout in
// qmc_launch.h): a record is one uniform load (LDCU.64; two records per LDCU.128 in the dense part), 2 LDS [R + UR] and one
// DFMA; the records of a sector sit at DENSE POSITIONS (a fixed number per group, qmc_tables.h) with compile-time
// destination registers: one basic block of independent load / multiply-add chains without a loop or a branch; what a
// group has beyond its positions was summed into a sector-local slot before (fused local entries).  The logarithm table
// is 64 entries x 8 interleaved copies (lane & 7 picks the copy): every lookup is a conflict-free LDS.128.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "qmc_fold.cuh"  // ipow_c, Expo, Ctx2, Fold2, finite_hi
#include "qmc_launch.h"

namespace qmc4 {

using qmc2::Ctx2;
using qmc2::Expo;
using qmc2::finite_hi;
using qmc2::Fold2;
using qmc2::ipow_c;

// ln x, absolute error ~1e-16: x = 2^e * z, z in [0.6875, 1.375), 64 sub-intervals with centre c_i;
// tab[i] = {1/c_i rounded, -ln(that) in extended precision}; r = z/c_i - 1 (one FMA, |r| < 2^-7), degree-7 log1p.
// `tabq` = this lane's copy of the table: entry i at tabq[i * QMC4_LOG_COPIES].
__constant__ double qmc4_logc[7] = {0.693147180559945309417, 1.0 / 7.0, -1.0 / 6.0, 0.2, -0.25, 1.0 / 3.0, -0.5};
__device__ __forceinline__ double fast_log(double x, const double2 *__restrict__ tabq) {
  const int hi = __double2hiint(x), lo = __double2loint(x);
  const bool ok = (unsigned)(hi - 0x00100000) < 0x7fe00000u;  // positive, normal
  const int tmp = hi - 0x3fe60000;
  const int e = tmp >> 20;
  const double2 T = *reinterpret_cast<const double2 *>(reinterpret_cast<const unsigned char *>(tabq) +
                                                      ((tmp >> (14 - 7)) & ((QMC4_LOG_ENTRIES - 1) << 7)));
  const double z = __hiloint2double(hi - (tmp & 0xfff00000), lo);
  const double r = fma(z, T.x, -1.0);
  const double y0 = fma((double)e, qmc4_logc[0], T.y);
  double q = fma(r, qmc4_logc[1], qmc4_logc[2]);
  q = fma(r, q, qmc4_logc[3]);
  q = fma(r, q, qmc4_logc[4]);
  q = fma(r, q, qmc4_logc[5]);
  q = fma(r, q, qmc4_logc[6]);
  const double v = fma(r * r, q, r) + y0;
  return ok ? v : __longlong_as_double(0x7ff8000000000000ll);
}
// the same without the argument test: `worst` collects max (hi - 0x00100000) as unsigned over a sector's corners, and the
// sector's result is dropped as a whole when worst >= 0x7fe00000 (some argument was not a positive normal number) --
// what the NaN of fast_log achieved through `finite_hi` of the results, at 2 instead of 4 integer instructions per corner
__device__ __forceinline__ double fast_log_unchecked(double x, const double2 *__restrict__ tabq, unsigned &worst) {
  const int hi = __double2hiint(x), lo = __double2loint(x);
  worst = max(worst, (unsigned)(hi - 0x00100000));
  const int tmp = hi - 0x3fe60000;
  const int e = tmp >> 20;
  const double2 T = *reinterpret_cast<const double2 *>(reinterpret_cast<const unsigned char *>(tabq) +
                                                      ((tmp >> (14 - 7)) & ((QMC4_LOG_ENTRIES - 1) << 7)));
  const double z = __hiloint2double(hi - (tmp & 0xfff00000), lo);
  const double r = fma(z, T.x, -1.0);
  const double y0 = fma((double)e, qmc4_logc[0], T.y);
  double q = fma(r, qmc4_logc[1], qmc4_logc[2]);
  q = fma(r, q, qmc4_logc[3]);
  q = fma(r, q, qmc4_logc[4]);
  q = fma(r, q, qmc4_logc[5]);
  q = fma(r, q, qmc4_logc[6]);
  // r + r^2 q + y0 as r (1 + r q) + y0: two FMAs instead of DMUL + DFMA + DADD (1 + r q carries 2^-53, times |r| < 2^-7)
  return fma(r, fma(r, q, 1.0), y0);
}
static_assert(QMC4_LOG_COPIES * 16 == 1 << 7, "fast_log index arithmetic assumes 128 bytes per table entry row");

// 1/x to ~1 ulp: MUFU.RCP64H seed (about 20 bits) + ONE cubic step r (1 + e + e^2), e = 1 - x r: 3 FP64 instructions
// (x normal, which U^, F^ and t_j are)
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  return fma(r, fma(e, e, e), r);
}

// sum of v over the block (valid in thread 0): warp shuffle tree, then pairwise over the warps; fixed order
template <int T>
__device__ __forceinline__ double block_sum_t(double v, double *scratch /*[T / 32]*/) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __syncthreads();
  if (lane == 0) scratch[wid] = v;
  __syncthreads();
  double r = 0.0;
  if (wid == 0) {
    r = (lane < T / 32) ? scratch[lane] : 0.0;
#pragma unroll
    for (int o = (T > 512 ? 16 : T / 64); o > 0; o >>= 1) r += __shfl_down_sync(0xffffffffu, r, o);
  }
  return r;
}

__device__ __forceinline__ double slot_at(const unsigned char *__restrict__ sl, uint32_t off) {
  return *reinterpret_cast<const double *>(sl + off);
}
__device__ __forceinline__ double u2d(uint32_t lo, uint32_t hi) { return __hiloint2double((int)hi, (int)lo); }
// 16-byte records {f64 c, u32 off0, u32 off1} of the complex path's real streams (qmc_kernels5.cuh): c * slot[off0] * slot[off1]
__device__ __forceinline__ double rec_val(const uint4 r, const unsigned char *__restrict__ sl) {
  return __hiloint2double((int)r.y, (int)r.x) * (slot_at(sl, r.z) * slot_at(sl, r.w));
}
__device__ __forceinline__ double rec_fma(const uint4 r, const unsigned char *__restrict__ sl, double acc) {
  return fma(__hiloint2double((int)r.y, (int)r.x), slot_at(sl, r.z) * slot_at(sl, r.w), acc);
}

// dense positions of group G (and, recursively, of the groups after it) of polynomial WHICH: P[G] = sum over the group's
// qmc4_cap positions of slot * slot; `fr` = first dense position of the sector (uniform), record index compile-time
template <int TPL, int NS, int WHICH, int G>
struct Dense4 {
  static __device__ __forceinline__ void eval(const unsigned char *__restrict__ fr, const unsigned char *__restrict__ sl,
                                              double (&P)[1 << NS]) {
    constexpr int CAP = qmc4_cap(TPL, NS, WHICH, qmc4_popc(G)), P0 = qmc4_pos(TPL, NS, WHICH, G);
    // a group with singular variable 0 starts from the sum of the group without it: the first level of the subset sums
    // (P[X] += P[X ^ 1]) rides on the first multiply-add instead of costing an addition of its own
    double acc = (G & 1) ? P[G ^ 1] : 0.0;
#pragma unroll
    for (int k = 0; k < CAP; ++k) {
      const uint4 q = *reinterpret_cast<const uint4 *>(fr + ((P0 + k) >> 1) * 16);
      const uint32_t oa = ((P0 + k) & 1) ? q.z : q.x, ob = ((P0 + k) & 1) ? q.w : q.y;
      acc = (k == 0 && !(G & 1)) ? slot_at(sl, oa) * slot_at(sl, ob) : fma(slot_at(sl, oa), slot_at(sl, ob), acc);
    }
    P[G] = acc;
    Dense4<TPL, NS, WHICH, G + 1>::eval(fr, sl, P);
  }
};
template <int TPL, int NS, int WHICH>
struct Dense4<TPL, NS, WHICH, 1 << NS> {
  static __device__ __forceinline__ void eval(const unsigned char *__restrict__, const unsigned char *__restrict__, double (&)[1 << NS]) {}
};

// W = U^aU0 F^aF0 and the argument U^aU1 F^aF1 of the logarithm (aU1 > 0 > aF1) from U, 1/F (and 1/U when aU0 < 0), with
// a = U / F shared between the two where both want it (double box: a, a^2, a^2 U, (1/F)^2, a (1/F)^2: five products)
template <class E>
__device__ __forceinline__ void corner_powers(double U, double F, double rF, double rU, double &W, double &arg) {
  constexpr int P = E::aU1 < -E::aF1 ? E::aU1 : -E::aF1;                              // arg = a^P U^(aU1-P) rF^(-aF1-P)
  constexpr int Q = (E::aU0 > 0 && E::aF0 < 0) ? (E::aU0 < -E::aF0 ? E::aU0 : -E::aF0) : 0;  // W = a^Q U^(aU0-Q) rF^(-aF0-Q)
  const double a = U * rF;
  double w = 1.0, g = 1.0;
  bool wset = false;
  if (Q > 0) { w = ipow_c<Q>(a); wset = true; }
  if (E::aU0 - Q > 0) { const double x = ipow_c<(E::aU0 - Q > 0 ? E::aU0 - Q : 0)>(U); w = wset ? w * x : x; wset = true; }
  if (E::aU0 < 0) { const double x = ipow_c<(E::aU0 < 0 ? -E::aU0 : 0)>(rU); w = wset ? w * x : x; wset = true; }
  if (-E::aF0 - Q > 0) { const double x = ipow_c<(-E::aF0 - Q > 0 ? -E::aF0 - Q : 0)>(rF); w = wset ? w * x : x; wset = true; }
  if (E::aF0 > 0) { const double x = ipow_c<(E::aF0 > 0 ? E::aF0 : 0)>(F); w = wset ? w * x : x; wset = true; }
  W = w;
  g = ipow_c<P>(a);
  if (E::aU1 - P > 0) g *= ipow_c<(E::aU1 - P > 0 ? E::aU1 - P : 0)>(U);
  if (-E::aF1 - P > 0) g *= ipow_c<(-E::aF1 - P > 0 ? -E::aF1 - P : 0)>(rF);
  arg = g;
}

// one sector at one point: out[i] = coefficient of eps^(i - NS) of the subtracted integrand without the weight w and
// without the sector's common factor G0' (returned in g0).  `o` = word offset of the sector block in p.tab (uniform).
template <int NDIM, int L, int NS, int KMAX, int T, int TPL>
__device__ __forceinline__ bool sector4(const Qmc4Launch &p, const uint32_t o, unsigned char *__restrict__ sl,
                                        const double2 *__restrict__ tabq, double (&out)[KMAX + NS + 1], double &g0) {
  unsigned worst = 0;  // fast_log_unchecked
  constexpr int K = KMAX + NS + 1, NC = 1 << NS, FULL = NC - 1;
  typedef Expo<NDIM, L> E;
  const unsigned char *tb = reinterpret_cast<const unsigned char *>(p.tab);
  const uint4 h0 = p.tab[o];
  constexpr uint32_t nL0 = NDIM - NS;  // one record per regular variable (beta_j = 0 where ln t_j does not enter)
  const uint32_t nlocal = (h0.x >> 16) & 255u, nfused = h0.x >> 24;
  {  // sector-local products: slot[local0 + i] = slot[a] * slot[b]
    const uint32_t lw = o + 9 + nL0;
#pragma unroll 1
    for (uint32_t i = 0; i < nlocal; i += 2) {
      const uint4 pw = p.tab[lw + (i >> 1)];
      *reinterpret_cast<double *>(sl + p.local0_off + i * (T * 8)) = slot_at(sl, pw.x) * slot_at(sl, pw.y);
      if (i + 1 < nlocal) *reinterpret_cast<double *>(sl + p.local0_off + (i + 1) * (T * 8)) = slot_at(sl, pw.z) * slot_at(sl, pw.w);
    }
    // fused entries: slot[dst] = slot[a] * slot[b] + slot[c] * slot[d] -- the monomials of a group beyond its dense positions
    const uint32_t fw = lw + ((nlocal + 1) >> 1);
#pragma unroll 1
    for (uint32_t i = 0; i < nfused; ++i) {
      const uint4 e = p.tab[fw + 2 * i];
      const uint32_t dst = p.tab[fw + 2 * i + 1].x;
      *reinterpret_cast<double *>(sl + dst) = fma(slot_at(sl, e.x), slot_at(sl, e.y), slot_at(sl, e.z) * slot_at(sl, e.w));
    }
  }
  {
    const uint4 g = p.tab[o + 7];
    g0 = u2d(g.x, g.y) * (slot_at(sl, g.z) * slot_at(sl, g.w));
    if (NS > 0) {  // the 1/t_k of the singular variables (Eq. 12), factored out of the fold: one reciprocal of their product
      const uint4 st = p.tab[o + 2];
      const uint32_t tw[4] = {st.x, st.y, st.z, st.w};
      double pt = slot_at(sl, tw[0]);
#pragma unroll
      for (int k = 1; k < NS; ++k) pt *= slot_at(sl, tw[k]);
      g0 *= fast_rcp(pt);
    }
  }
  double L0 = u2d(p.tab[o + 8].x, p.tab[o + 8].y);
#pragma unroll
  for (uint32_t i = 0; i < nL0; ++i) {
    const uint4 r = p.tab[o + 9 + i];
    L0 = fma(u2d(r.x, r.y), slot_at(sl, r.z), L0);
  }
  Ctx2<NS, K> c;
  {
    // dense positions (qmc_tables.h: qmc4_cap): every group of U^ and F^ owns a fixed number of records with compile-time
    // destination registers -- one basic block of independent load / multiply-add chains, no loop, no branch;
    // subset sums: P[X] = value with the singular variables outside X set to zero
    double PU[NC], PF[NC];
    const unsigned char *fr = tb + (o + h0.z) * 16u;
    Dense4<TPL, NS, 0, 0>::eval(fr, sl, PU);
    Dense4<TPL, NS, 1, 0>::eval(fr, sl, PF);
#pragma unroll
    for (int b = 1; b < NS; ++b)  // (level b = 0 is done by Dense4)
#pragma unroll
      for (int X = 0; X < NC; ++X)
        if (X >> b & 1) {
          PU[X] += PU[X ^ (1 << b)];
          PF[X] += PF[X ^ (1 << b)];
        }
    // corners: W = U^aU0 F^aF0 (one reciprocal), Lambda = ln(U^aU1 F^aF1) + L0 (one logarithm)
#pragma unroll
    for (int X = 0; X < NC; ++X) {
      const double U = PU[X], F = PF[X];
      const double rF = fast_rcp(F);
      const double rU = E::aU0 < 0 ? fast_rcp(U) : 0.0;
      double W, arg;
      corner_powers<E>(U, F, rF, rU, W, arg);
      c.W[X] = W;
      if (KMAX > 0 || X != FULL) c.Lam[X] = fast_log_unchecked(arg, tabq, worst) + L0;
    }
  }
  if (NS > 0) {
    const uint4 sln = p.tab[o + 1], st = p.tab[o + 2];
    const uint4 ib01 = p.tab[o + 3], ib23 = p.tab[o + 4], b01 = p.tab[o + 5], b23 = p.tab[o + 6];
    const uint32_t lnw[4] = {sln.x, sln.y, sln.z, sln.w}, tw[4] = {st.x, st.y, st.z, st.w};
    const double ibv[4] = {u2d(ib01.x, ib01.y), u2d(ib01.z, ib01.w), u2d(ib23.x, ib23.y), u2d(ib23.z, ib23.w)};
    const double bv[4] = {u2d(b01.x, b01.y), u2d(b01.z, b01.w), u2d(b23.x, b23.y), u2d(b23.z, b23.w)};
#pragma unroll
    for (int k = 0; k < NS; ++k) {
      c.bt[k] = ibv[k] * slot_at(sl, tw[k]);
      const double Lk = bv[k] * slot_at(sl, lnw[k]);
      c.cL[k][0] = 1.0;
#pragma unroll
      for (int q = 1; q < K - 1; ++q) c.cL[k][q] = c.cL[k][q - 1] * (Lk * (1.0 / q));
    }
  }
  Fold2<NS, KMAX, K, 0, 0>::eval(c, out);
  return worst < 0x7fe00000u;
}

}  // namespace qmc4

// partial layout: [row][shift][slice][NACC], row = run of sectors (fused mode) or sector (per-sector mode: one launch per
// sector, so that the accumulators stay in registers)        (NACC = QMC_MAXSING + KMAX + 1, index a <-> order a - QMC_MAXSING)
// T = threads per block (128 or 512; 512 registers-worth of threads per SM either way: 128 registers per thread)
template <int NDIM, int L, int KMAX, int T, int TPL>
__global__ void __launch_bounds__(T, T >= 256 ? 1 : 512 / T) qmc4_eval_kernel(const __grid_constant__ Qmc4Launch p) {
  using namespace qmc4;
  constexpr int NACC = QMC_MAXSING + KMAX + 1;
  constexpr int SMAX = NDIM < QMC_MAXSING ? NDIM : QMC_MAXSING;

  extern __shared__ __align__(16) unsigned char smem[];
  const int tid = threadIdx.x;

  // shared memory carve-up (all offsets multiples of 16)
  double2 *logtab = reinterpret_cast<double2 *>(smem);
  size_t o = (size_t)QMC4_LOG_ENTRIES * QMC4_LOG_COPIES * 16;
  double *shf = reinterpret_cast<double *>(smem + o);
  o += (((size_t)p.m * NDIM * 8) + 15) & ~(size_t)15;
  double *scratch = reinterpret_cast<double *>(smem + o);
  o += (T / 32) * 8;
  double *slots = reinterpret_cast<double *>(smem + o);
  unsigned char *sl = reinterpret_cast<unsigned char *>(slots + tid);
  const double2 *tabq = logtab + (tid & (QMC4_LOG_COPIES - 1));

  for (int i = tid; i < QMC4_LOG_ENTRIES * QMC4_LOG_COPIES; i += T)
    logtab[i] = reinterpret_cast<const double2 *>(p.logtab)[i / QMC4_LOG_COPIES];
  for (int i = tid; i < p.m * NDIM; i += T) shf[i] = p.shifts[i];
  slots[2 * NDIM * T + tid] = 1.0;        // the constant slots: 1, 0, the chunk's coefficient constants
  slots[(2 * NDIM + 1) * T + tid] = 0.0;
  for (uint32_t i = 0; i < p.nconst; ++i) slots[(2 * NDIM + 2 + i) * T + tid] = p.cval[i];
  __syncthreads();

  const uint32_t N = p.N;

  const uint32_t stride = (uint32_t)p.nslices * T;
  uint32_t dz[NDIM];
#pragma unroll
  for (int j = 0; j < NDIM; ++j) dz[j] = (uint32_t)(((uint64_t)stride * p.zeff[j]) % N);

  unsigned cntNonFinite = 0, cntBoundary = 0;

  // One block = one shift vector (blockIdx.y): with the shift loop inside the block, the block reduction (barriers,
  // shuffles under `if (warp == 0)`) sat on the back edge of a loop around the table walk, and ptxas then kept the whole
  // walk off the uniform datapath.
  const int kap = blockIdx.y;
  {
    double acc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) acc[a] = 0.0;

    // The point loop has a UNIFORM trip count (threads past the end of the index range, and boundary points, carry the
    // weight 0 at a harmless stand-in point): only then may ptxas keep the table walk on the uniform datapath.
    const uint32_t c0 = (uint32_t)blockIdx.x * T;
    uint32_t r[NDIM];
#pragma unroll
    for (int j = 0; j < NDIM; ++j) r[j] = (uint32_t)((p.off[j] + (uint64_t)(c0 + tid) * p.zeff[j]) % N);

    uint32_t since_sync = 0;
    for (uint32_t cb = c0; cb < p.count; cb += stride) {
      // S1-S3: lattice point (Eq. 17), shift + wrap (Eq. 18), periodising transform (Eq. 21), per-point slot table
      const bool valid = cb + tid < p.count;
      double w = 1.0;
      bool inside = true;
#pragma unroll
      for (int j = 0; j < NDIM; ++j) {
        // u = r / N correctly rounded (the oracle's IEEE division) without the division routine: q = r * RN(1/N),
        // remainder by FMA (exact), one correction -- Markstein's theorem (r, N integers below 2^31: no exception case)
        const double rd = (double)r[j], q0 = rd * p.invN;
        const double u = fma(fma(-q0, p.dN, rd), p.invN, q0);
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
        reinterpret_cast<double *>(sl)[j * T] = tj;
        reinterpret_cast<double *>(sl)[(NDIM + j) * T] = fast_log(tj, tabq);  // t >= 3.7e-32 for y >= 2^-53: a normal number
        uint32_t rn = r[j] + dz[j];
        r[j] = rn >= N ? rn - N : rn;
      }
      if (valid && !inside && p.count_boundary) ++cntBoundary;
      const bool live = valid && inside;
      if (!live) w = 0.0;
      for (uint32_t i = 0; i < p.nprog; i += 2) {  // chunk-wide product slots
        const uint4 pw = p.tab[p.prog_word + (i >> 1)];
        *reinterpret_cast<double *>(sl + p.first_prod_off + i * (T * 8)) = slot_at(sl, pw.x) * slot_at(sl, pw.y);
        if (i + 1 < p.nprog)
          *reinterpret_cast<double *>(sl + p.first_prod_off + (i + 1) * (T * 8)) = slot_at(sl, pw.z) * slot_at(sl, pw.w);
      }
      // S4-S6: all sectors of the run at this point.  A barrier every few points (p.sync_every, kernels)
      // re-aligns the block's warps so that they share fetched instruction lines, while between two barriers they drift
      // apart again, which keeps the table-walk phase of one warp over the arithmetic phase of another.
      if (T >= 256 && p.sync_every) {
        if (since_sync == 0) __syncthreads();
        since_sync = since_sync + 1 == p.sync_every ? 0 : since_sync + 1;
      }
      // (sectors are sorted by their number of singular variables: p.nsb[ns] .. p.nsb[ns + 1] run the code path of ns;
      //  offsets come from an array indexed by the induction variable: a loop-carried offset read from the table
      //  itself makes ptxas give up the uniform datapath for the whole table walk)
#define QMC4_CLASS(NS_)                                                                                      \
  if (NS_ <= SMAX) {                                                                                         \
    constexpr int NSC = NS_ <= SMAX ? NS_ : 0, KK = KMAX + NSC + 1;                                          \
    for (int si = p.nsb[NS_]; si < p.nsb[NS_ + 1]; ++si) {                                                   \
      const uint32_t so = p.secw[si];                                                                        \
      double res[KK], g0;                                                                                    \
      bool fin = sector4<NDIM, L, NSC, KMAX, T, TPL>(p, so, sl, tabq, res, g0);                                   \
      const double wg = w * g0;                                                                              \
      fin = fin && finite_hi(g0);                                                                            \
      _Pragma("unroll") for (int i = 0; i < KK; ++i) fin = fin && finite_hi(res[i]);                         \
      /* a non-finite evaluation is dropped (and counted); a dead thread has w = 0.  Predicated, not branched */ \
      cntNonFinite += (live && !fin) ? 1u : 0u;                                                              \
      _Pragma("unroll") for (int i = 0; i < KK; ++i)                                                         \
        if (fin) acc[QMC_MAXSING - NSC + i] = fma(wg, res[i], acc[QMC_MAXSING - NSC + i]);                   \
    }                                                                                                        \
  }
      QMC4_CLASS(0)
      QMC4_CLASS(1)
      QMC4_CLASS(2)
      QMC4_CLASS(3)
      QMC4_CLASS(4)
#undef QMC4_CLASS
    }

    // S7: block reduction -> one partial per (row, shift, block)
    double *dst = p.partial + (((size_t)p.out_row * p.m + kap) * p.max_slices + blockIdx.x) * NACC;
#pragma unroll
    for (int a = 0; a < NACC; ++a) {
      double sr = block_sum_t<T>(acc[a], scratch);
      if (tid == 0) dst[a] = sr;
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
