// Internal (not part of the C ABI): host-side sector tables and the device table image.
// Shared by qmc_prepare.cpp (host decomposer), qmc_api.cu (launcher) and the kernels.
#pragma once
#include <cstddef>
#include <cstdint>
#include <vector>

#include "../../include/qmc_feynman.h"

#define QMC_MAXDIM 8    // integration variables per sector (P - 1)
#define QMC_IBP_JET 16    // integration by parts: largest number of Taylor coefficients prod_b (1 - alpha_b) of a sector
#define QMC_MAXTAYLOR 3   // most negative exponent -alpha of a variable the generic kernel's Taylor corners handle
#define QMC_MAXSING 4   // singular variables (alpha = -1) per sector handled by the kernels
#define QMC_MAXK 8      // eps orders kept: k_max - k_min + 1
#define QMC_KMAX_MAX 2  // highest eps_order the kernels are instantiated for
#define QMC_NACC_MAX (QMC_MAXSING + QMC_KMAX_MAX + 1)  // accumulators per thread: order k <-> index k + QMC_MAXSING

// ---- device image -------------------------------------------------------------------------------
// One 64-byte header per sector, followed by coef[nU+nF] (f64) and exps[nU+nF] (u32, 4 bits per variable),
// padded to 16 bytes so that a run of sectors can be moved with one TMA bulk copy.
// Variables are PERMUTED per sector: the nsing singular ones (alpha = -1) first, in increasing original
// index, then the others.  perm[k] = original index of position k.  Monomials of U^ then F^, each sorted by
// "group" = set of singular positions on which the monomial depends; cntU/cntF[g] = monomials in group g.
struct QmcSectorHdr {
  uint8_t nsing, nU, nF, flags;
  uint8_t perm[QMC_MAXDIM];
  int8_t alpha[QMC_MAXDIM];  // permuted order
  int8_t beta[QMC_MAXDIM];
  uint8_t cntU[1 << QMC_MAXSING];
  uint8_t cntF[1 << QMC_MAXSING];
  uint8_t pad[4];
};
static_assert(sizeof(QmcSectorHdr) == 64, "sector header must be 64 bytes");

// ---- real path ("version 4" tables, built by qmc_image4.cpp; layout of the kernel-side tables: qmc_launch.h) ----------
// Sectors are grouped into CHUNKS.  Every chunk owns a "slot program": each thread keeps, per lattice point, a column
// of per-point values in shared memory (slot s of thread tid at slots[s * T + tid]):
//   [0,n) t_j | [n,2n) ln t_j | 2n: 1.0 | 2n+1: 0.0 | 2n+2 ..: coefficient constants | products slot[k] = slot[a] * slot[b]
// chosen per chunk by a byte-pair-encoding style pass over the chunk's monomials (most frequent pair of factors
// first) until every monomial is a product of at most two slots.  A monomial is then one 8-byte record.
#define QMC2_MAXSLOTS 56
#define QMC2_MAXLOCAL 8
#ifndef QMC4_TBIG
#define QMC4_TBIG 512  // threads per block of the real-path kernel for tables dominated by sectors with 3-4 singular variables
#endif
#define QMC4_MAXCONST 12   // distinct coefficient constants (other than 1) per chunk
// Real-path walk: DENSE POSITIONS per group of a sector's U^ and F^ (group = set of singular variables a monomial depends
// on), by (template, number of singular variables, polynomial, popcount of the group).  The kernel evaluates every position
// in straight-line code with a compile-time destination register; a group with fewer monomials fills up with 0 * 0 records,
// a group with more sums its overflow into a sector-local slot first (qmc_image4.cpp).  Two templates, chosen per tables
// object by modelled cost: 0 = lean (one-loop sized polynomials: one or two monomials per group), 1 = tuned on the group
// statistics of the two-loop planar double box.  Any shape is exact under either.
#if defined(__CUDACC__)
#define QMC_HD __host__ __device__
#else
#define QMC_HD
#endif
QMC_HD constexpr int qmc4_cap(int tpl, int nsing, int poly, int popc) {
  constexpr int capU1[5][5] = {{6, 0, 0, 0, 0}, {8, 10, 0, 0, 0}, {4, 4, 7, 0, 0}, {2, 2, 3, 5, 0}, {1, 1, 1, 2, 5}};
  constexpr int capF1[5][5] = {{6, 0, 0, 0, 0}, {8, 3, 0, 0, 0}, {6, 2, 2, 0, 0}, {4, 2, 2, 1, 0}, {3, 1, 1, 1, 1}};
  constexpr int capU0[5][5] = {{3, 0, 0, 0, 0}, {2, 2, 0, 0, 0}, {2, 1, 1, 0, 0}, {2, 1, 1, 1, 0}, {1, 1, 1, 1, 1}};
  constexpr int capF0[5][5] = {{3, 0, 0, 0, 0}, {2, 1, 0, 0, 0}, {2, 1, 1, 0, 0}, {2, 1, 1, 1, 0}, {2, 1, 1, 1, 1}};
  return tpl ? (poly ? capF1[nsing][popc] : capU1[nsing][popc]) : (poly ? capF0[nsing][popc] : capU0[nsing][popc]);
}
QMC_HD constexpr int qmc4_popc(int g) { return (g & 1) + ((g >> 1) & 1) + ((g >> 2) & 1) + ((g >> 3) & 1); }
// index of the first dense position of group g of polynomial poly (U^ positions first, then F^); g = 2^nsing: the total
QMC_HD constexpr int qmc4_pos(int tpl, int nsing, int poly, int g) {
  int p = 0;
  for (int q = 0; q <= poly; ++q)
    for (int h = 0; h < (q < poly ? (1 << nsing) : g); ++h) p += qmc4_cap(tpl, nsing, q, qmc4_popc(h));
  return p;
}
struct Qmc2Rec {        // complex-path record: value = c * slot[s0] * slot[s1]; s0, s1 are BYTE offsets into the thread's column
  double c;
  uint32_t s0, s1;
};
static_assert(sizeof(Qmc2Rec) == 16, "record must be 16 bytes");
struct Qmc2Chunk {      // host description of one chunk
  int sec_begin = 0, sec_end = 0;
  int nslots = 0;     // chunk-wide slots (base + constants + products)
  int nconst = 0;     // coefficient constants (real path)
  int max_local = 0;  // largest number of sector-local product slots in the chunk
  int nrec = 0, nsingle = 0, nlocal = 0, noverflow = 0;  // monomial records / sector-local products / monomials beyond the dense positions (describe)
  uint32_t tab_words = 0;                 // 16-byte words of sector blocks (real path)
  uint32_t prog_off = 0, prog_bytes = 0;  // complex path: chunk header + slot programs in image3
  double cost = 0.0;                      // modelled flops per point (load balancing)
};

// ---- planning image of the complex path ("version 3": host only; the kernels read the version-5 tables) ------
// Same idea as version 2, with TWO slot tables per thread: a REAL one at the lattice point (t_j, ln t_j, 1,
// products) that serves the gradient and Hessian polynomials of F^ -- emitted by qmc_prepare as record lists of their
// own -- and the regular-variable factors; and a COMPLEX one over the deformed variables z_j (z_j, 1, products),
// refilled at every corner, that serves U^(z) and F^(z).  Records are sorted per polynomial by group; a corner Z keeps
// the groups disjoint from Z.
#define QMC3_THREADS 128
// Complex path, stream A of a corner (one-factor records c * slot of the derivative polynomials): FIXED positions per polynomial,
// evaluated in straight-line code (a polynomial with fewer records fills up with c = 0, a surplus goes to stream B as
// c * slot * 1).  Gradient polynomials d_i F^ get QMC5_CAPG positions, Hessian polynomials d_i d_k F^ QMC5_CAPH: for L loops F^ has
// degree L + 1, so at one loop the Hessian is constant (no positions) and the gradient linear (up to n terms); at two loops the
// Hessian is linear (measured on cfg5: 3.5 one-factor records per Hessian polynomial, 4.4 per gradient polynomial).
#if defined(__CUDACC__)
#define QMC5_HD __host__ __device__
#else
#define QMC5_HD
#endif
#ifndef QMC5_CAPG2
#define QMC5_CAPG2 6  // two loops: positions per gradient polynomial
#define QMC5_CAPH2 3  // ... per Hessian polynomial.  Measured on B200 (cfg5 / paper I_C / I_D, ms per step): (4,3) 138.1 / 267.4 /
                      // 288.2; (5,4) 140.4 / 267.6 / 284.6; (6,3) 136.9 / 263.7 / 282.5; (6,4) 139.8 / 268.8 / 284.1; (8,5) 143.6 / 273.1 /
                      // 293.1; (10,6) 151.1 / 285.3 / 295.9; (12,8) 162.0 / 304.0 / 315.4 (larger tables: more launches)
#endif
QMC5_HD constexpr int qmc5_capA(int ndim, int loops, int q) { return q < ndim ? (loops == 1 ? ndim : QMC5_CAPG2) : (loops == 1 ? 0 : QMC5_CAPH2); }
QMC5_HD constexpr int qmc5_posA(int ndim, int loops, int q) {  // first position of polynomial q; q = number of derivative polynomials: the total
  int p = 0;
  for (int i = 0; i < q; ++i) p += qmc5_capA(ndim, loops, i);
  return p;
}
#define QMC3_MAXSLOTS_R 56
#define QMC3_MAXSLOTS_C 40
#define QMC3_MAXLOCAL 8
struct Qmc3ChunkHdr {  // 32 bytes; followed by program R then program C: {u16 a, u16 b} slot indices, each padded to 16 bytes
  uint32_t nslots_r, nprog_r, first_prod_r;
  uint32_t nslots_c, nprog_c, first_prod_c;
  uint32_t pad[2];
};
struct Qmc3SectorHdr {  // 96 bytes; followed by: group counts u8 [npoly][2^nsing] (npoly = n + n(n+1)/2 + 2: F_i, F_ik (i<=k),
                        // U, F), padded to 16 | local program R | local program C (each padded to 16) | real records
                        // [G0][L0 x nL0][F_1..F_n][F_11, F_12, .., F_nn] | complex records [U^][F^]
  uint8_t nsing, nL0, nlocal_r, nlocal_c;
  uint16_t nrec_r, nrec_c;
  uint8_t sing_var[QMC_MAXSING];   // variable index of singular position k
  uint8_t pad0[4];
  int8_t alpha[QMC_MAXDIM], beta[QMC_MAXDIM];  // original variable order
  double invbeta[QMC_MAXSING];     // 1/beta of singular position k
  double betas[QMC_MAXSING];       // beta of singular position k
};
static_assert(sizeof(Qmc3SectorHdr) == 96, "v3 sector header");

// ---- host tables --------------------------------------------------------------------------------
struct QmcMono {
  double c;
  uint8_t e[QMC_MAXDIM];  // original variable order
};

struct QmcSector {
  int primary;
  int alpha[QMC_MAXDIM], beta[QMC_MAXDIM];  // original variable order
  int nsing;  // variables with alpha <= -1 (each can give a pole)
  int ndeep = 0;  // ... of which alpha <= -2 (Taylor terms p >= 1 of Eq. 11; generic kernel, real path only)
  std::vector<QmcMono> U, F;  // evaluation order (group-sorted)
};

struct qmc_tables {
  int n = 0, P = 0, L = 0;
  int kmin = 0, kmax = 0;
  int aU0 = 0, aU1 = 0, aF0 = 0, aF1 = 0;
  double lambda = 0.0;
  int transform = 0;
  int lattice = 0;  // qmc_options::lattice
  std::vector<QmcSector> sectors;
  std::vector<int> row_of_sector;  // batch of kinematic points (qmc_prepare_batch): kinematic point of every sector; else empty
  int n_rows = 1;                  // kinematic points in the batch
  // device image
  std::vector<uint8_t> image;     // concatenated sector blocks (16-byte aligned each)
  std::vector<uint32_t> secoff;   // [n_sectors + 1] byte offsets
  std::vector<Qmc2Chunk> chunks;  // real path (empty when lambda > 0)
  std::vector<double> sec_cost;   // modelled cost per sector (load balancing of the launch)
  // version 4 tables (real path; laid out for the kernel-parameter constant bank: see qmc_launch.h)
  int tpl_real = 1;                 // dense-position template of the real-path tables (qmc4_cap)
  int threads_real = 512;           // threads per block of the real-path kernel: the slot offsets in tab4 / prog4 are
                                    // premultiplied by it (chosen by qmc_build_tables4, see there)
  std::vector<uint32_t> tab4;       // sector blocks, 32-bit words (4 per 16-byte table word)
  std::vector<uint32_t> secoff4;    // [n_sectors + 1] offsets into tab4 in 16-byte words
  std::vector<std::vector<uint32_t>> prog4;  // per chunk: slot program {a_off, b_off} byte offsets, padded to 16 bytes
  std::vector<std::vector<double>> const4;   // per chunk: values of the coefficient-constant slots
  double logtab4[128] = {0};        // 64 x {1/c_i, -ln(1/c_i)}
  // version 5 tables (complex path; same chunks and slot programs as version 3, laid out for the constant bank)
  std::vector<uint32_t> tab5, secoff5;             // sector blocks (32-bit words) and their offsets in 16-byte words
  std::vector<std::vector<uint32_t>> prog5r, prog5c;  // per chunk: real / complex slot programs {a_off, b_off}
  void *side_streams[8] = {nullptr};  // cudaStream_t: the launches of one integration are spread over these
  void *side_events[9] = {nullptr};   // cudaEvent_t: fork + one join per side stream
  // planning image of the complex path (host only)
  std::vector<uint8_t> image3;
  std::vector<uint32_t> secoff3, secend3;
  std::vector<Qmc2Chunk> chunks3;    // nslots = real slots; prog_off/prog_bytes cover the chunk header + both programs
  std::vector<int> chunk3_nslots_c, chunk3_max_local_c;
  std::vector<double> rec_flops5;    // per sector: FP64 operations of the record streams of all its corners (flop model)
  // launcher state (host-side caches; not thread-safe by design: one tables object per stream)
  const void *resident_ws = nullptr;  // workspace the image was last uploaded to
  int resident_kind = 0;              // 4: logarithm table (versions 4, 5), 1: version-1 image
  int resident_m = 0;                 // number of shift vectors resident in that workspace (0 = none)
  uint64_t resident_seed = 0;         // seed that produced them ...
  bool ibp = false;                   // qmc_options.pole_extraction = 1: Eq. 13 instead of Eqs. 11-12 (generic kernel, real path)
  bool has_taylor = false;            // some sector has a variable with alpha <= -2
  bool generic_only = false;          // propagator powers other than 1: only the generic kernel has run-time exponents
  bool resident_explicit = false;     // ... or: they were passed explicitly (qmc_run.shifts)
  uint64_t cached_N = 0;              // generating vector cache
  uint64_t cached_z[QMC_MAXDIM] = {0};
  std::vector<double> shifts_host;    // staging of the shift vectors (must outlive the async H2D copy)
  std::vector<double> stat_host;      // staging of the fetched statistics block
  std::vector<int> run_begin_host;    // batch mode: first run of every kinematic point (must outlive the async H2D copy)
  void *ev0 = nullptr, *ev1 = nullptr, *evm = nullptr;  // cudaEvent_t: before / after all kernels, after the evaluation kernel
  struct {
    bool valid = false;
    const void *ws = nullptr;
    int m = 0, mode = 0, nrows = 0;
    size_t h2d = 0;
    int launches = 3;
  } last;
};

// builds sectors (+ image) from a graph; returns a qmc_status
// builds tab4 / secoff4 / prog4 / const4 / chunks from `sectors` (real path); returns a qmc_status.
// slot_budget, chunk_bytes, threads: 0 = the measured defaults (qmc_tuning in qmc_feynman.h)
int qmc_build_tables4(qmc_tables *t, int slot_budget, int chunk_bytes, int threads, int dense_template);
// builds image3 / secoff3 / chunks3 (complex path); returns a qmc_status
int qmc_build_image3(qmc_tables *t, int slots_r, int slots_c, int chunk_bytes);  // 0 = the measured defaults
int qmc_build_tables(const qmc_graph *g, const qmc_kinematics *kin, int eps_order, const qmc_options *opt,
                     qmc_tables *out);
int qmc_build_tables_batch(const qmc_graph *g, const qmc_kinematics *kins, int n_points, int eps_order, const qmc_options *opt,
                           qmc_tables *out);
