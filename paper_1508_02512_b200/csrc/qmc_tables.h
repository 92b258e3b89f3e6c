// Internal (not part of the C ABI): host-side sector tables and the device table image.
// Shared by qmc_prepare.cpp (host decomposer), qmc_api.cu (launcher) and the kernels.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/qmc_feynman.h"

#define QMC_MAXDIM 8    // integration variables per sector (P - 1)
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

// ---- host tables --------------------------------------------------------------------------------
struct QmcMono {
  double c;
  uint8_t e[QMC_MAXDIM];  // original variable order
};

struct QmcSector {
  int primary;
  int alpha[QMC_MAXDIM], beta[QMC_MAXDIM];  // original variable order
  int nsing;
  std::vector<QmcMono> U, F;  // evaluation order (group-sorted)
};

struct qmc_tables {
  int n = 0, P = 0, L = 0;
  int kmin = 0, kmax = 0;
  int aU0 = 0, aU1 = 0, aF0 = 0, aF1 = 0;
  double lambda = 0.0;
  int transform = 0;
  std::vector<QmcSector> sectors;
  // device image
  std::vector<uint8_t> image;     // concatenated sector blocks (16-byte aligned each)
  std::vector<uint32_t> secoff;   // [n_sectors + 1] byte offsets
  // launcher state (host-side caches; not thread-safe by design: one tables object per stream)
  const void *resident_ws = nullptr;  // workspace the image was last uploaded to
  int resident_m = 0;                 // number of shift vectors resident in that workspace (0 = none)
  uint64_t cached_N = 0;              // generating vector cache
  uint64_t cached_z[QMC_MAXDIM] = {0};
  std::vector<double> shifts_host;    // staging of the shift vectors (must outlive the async H2D copy)
  std::vector<double> stat_host;      // staging of the fetched statistics block
  void *ev0 = nullptr, *ev1 = nullptr, *evm = nullptr;  // cudaEvent_t: before / after all kernels, after the evaluation kernel
  struct {
    bool valid = false;
    const void *ws = nullptr;
    int m = 0, mode = 0, nrows = 0;
    size_t h2d = 0;
  } last;
};

// builds sectors (+ image) from a graph; returns a qmc_status
int qmc_build_tables(const qmc_graph *g, const qmc_kinematics *kin, int eps_order, const qmc_options *opt,
                     qmc_tables *out);
