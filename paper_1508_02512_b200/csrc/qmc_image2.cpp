// Version-2 device image of the sector tables (real path): chunks, per-chunk slot programs, 16-byte monomial records.
// Host only.  See qmc_tables.h for the layout and DESIGN.md "Data layout" for the rationale.
//
// The slot program is found by a byte-pair-encoding style pass: a monomial is a multiset of factors (initially the
// variables t_j, repeated by exponent); the most frequent pair of factors over the chunk becomes a new slot (their
// product, computed once per lattice point) and replaces the pair everywhere; repeat until every monomial has at
// most two factors (mandatory) and, with the slots that are left, as many as possible have one.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "../../include/qmc_feynman.h"
#include "qmc_bpe.h"
#include "qmc_tables.h"

using namespace qmcbpe;

namespace {

void collect(const qmc_tables *t, int s0, int s1, ChunkPlan &pl) {
  pl.mono.clear();
  const int n = t->n;
  for (int si = s0; si < s1; ++si) {
    const QmcSector &s = t->sectors[si];
    uint8_t g[QMC_MAXDIM] = {0};
    for (int j = 0; j < n; ++j) g[j] = (uint8_t)(s.alpha[j] > 0 ? s.alpha[j] : 0);
    pl.mono.push_back(factors_of(g, n));  // G0 = prod over regular variables of t_j^alpha_j
    for (const QmcMono &m : s.U) pl.mono.push_back(factors_of(m.e, n));
    for (const QmcMono &m : s.F) pl.mono.push_back(factors_of(m.e, n));
  }
}

// relative cost of one sector at one point, fitted to measured per-chunk kernel times on B200 (cfg4, r01d):
// time ~ 7.8 per corner (reciprocal, logarithm, series, its share of the fold) + 1 per record
double sector_cost(const QmcSector &s, int kmax) {
  const int nc = 1 << s.nsing;
  return 7.8 * nc * (1.0 + 0.15 * kmax) + (double)(s.U.size() + s.F.size() + 2);
}

}  // namespace

// table of the kernels' logarithm: z in [0.6875, 1.375), 64 intervals by the top bits of the high word, c_i = interval centre;
// tab[i] = {1/c_i rounded, -ln(that) in extended precision}
static void build_logtab4(double *tab) {
  for (int i = 0; i < 64; ++i) {
    const uint64_t lo = ((uint64_t)(0x3fe60000u + ((uint32_t)i << 14))) << 32, hi = lo + ((uint64_t)0x4000 << 32);
    double zl, zh;
    std::memcpy(&zl, &lo, 8);
    std::memcpy(&zh, &hi, 8);
    const double invc = (double)(1.0L / (0.5L * ((long double)zl + (long double)zh)));
    tab[2 * i] = invc;
    tab[2 * i + 1] = (double)(-logl((long double)invc));
  }
}

namespace {
void put32(std::vector<uint32_t> &v, uint32_t x) { v.push_back(x); }
void putf64(std::vector<uint32_t> &v, double d) {
  uint64_t b;
  std::memcpy(&b, &d, 8);
  v.push_back((uint32_t)b);
  v.push_back((uint32_t)(b >> 32));
}
void pad4(std::vector<uint32_t> &v) {
  while (v.size() % 4) v.push_back(0);
}
// record of the planning image (offsets = slot * QMC2_THREADS * 8) -> record for T threads per block
void put_rec(std::vector<uint32_t> &v, const Qmc2Rec &r, uint32_t T) {
  putf64(v, r.c);
  v.push_back(r.s0 / (QMC2_THREADS * 8u) * T * 8u);
  v.push_back(r.s1 / (QMC2_THREADS * 8u) * T * 8u);
}
}  // namespace

int qmc_build_image2(qmc_tables *t) {
  build_logtab4(t->logtab4);
  t->tab4.clear();
  t->secoff4.clear();
  t->prog4.clear();
  {
    // Threads per block of the real-path kernel, measured on B200 (kernels): tables dominated by sectors
    // with three or four singular variables execute long straight-line code paths, and one 512-thread block per SM (all
    // 16 warps walking the same sectors) fetches instructions better than four independent 128-thread blocks
    // (cfg4: 247 / 261 / 304 ms at 512 / 256 / 128 threads); tables of short paths prefer the small blocks (cfg2: 23.4 /
    // 22.4 / 21.6 ms).
    int big = 0;
    for (const QmcSector &s : t->sectors) big += s.nsing >= 3;
    t->threads_real = 2 * big >= (int)t->sectors.size() ? 512 : 128;
    if (const char *e = std::getenv("QMC4_THREADS")) t->threads_real = std::atoi(e) == 128 ? 128 : 512;
  }
  const uint32_t T4 = (uint32_t)t->threads_real;
  t->image2.clear();
  t->secoff2.clear();
  t->chunks.clear();
  t->secend2.clear();
  t->sec_cost.clear();
  const int n = t->n, nsec = (int)t->sectors.size();
  if (t->lambda > 0.0 || nsec == 0) return QMC_OK;  // complex path keeps the version-1 image
  if (3 * n + 1 >= QMC2_MAXSLOTS) return QMC_EUNSUPPORTED;

  // ---- chunk boundaries: contiguous ranges of about equal modelled cost, about 20 KB of tables each ------------
  std::vector<double> cost(nsec);
  double total_cost = 0.0, total_bytes = 0.0;
  for (int i = 0; i < nsec; ++i) {
    const QmcSector &s = t->sectors[i];
    cost[i] = sector_cost(s, t->kmax);
    t->sec_cost.push_back(cost[i]);
    total_cost += cost[i];
    total_bytes += sizeof(Qmc2SectorHdr) + 16.0 * (s.U.size() + s.F.size() + 1 + n);
  }
  // defaults measured on B200 (profiles/r01b_sweep.md): 36 chunk-wide slots + up to 8 sector-local ones keep two
  // 256-thread blocks resident per SM (2 x (44 x 2 KB + 16 KB of tables) < 227 KB); more slots halve the occupancy
  int max_slots = std::min(QMC2_MAXSLOTS, std::max(36, 3 * n + 2));
  double chunk_bytes = 16000.0;
  if (const char *e = std::getenv("QMC2_SLOTS")) max_slots = std::min(QMC2_MAXSLOTS, std::max(3 * n + 2, std::atoi(e)));
  if (const char *e = std::getenv("QMC2_CHUNK_BYTES")) chunk_bytes = std::max(1000.0, std::atof(e));
  int nch = std::max(1, (int)(total_bytes / chunk_bytes + 0.999));
  std::vector<std::pair<int, int>> todo;  // ranges still to plan (processed in order)
  {
    int b = 0;
    double acc = 0.0;
    for (int c = 0; c < nch; ++c) {
      const double target = total_cost * (c + 1) / nch;
      int e = b;
      while (e < nsec && (acc + cost[e] <= target || e == b)) acc += cost[e++];
      if (c == nch - 1) e = nsec;
      if (e > b) todo.push_back({b, e});
      b = e;
    }
  }
  // ---- plan (split a range in two when the slot budget does not suffice) and emit -----------------------------
  t->secoff2.assign(nsec + 1, 0);
  t->secend2.assign(nsec, 0);
  for (size_t w = 0; w < todo.size(); ++w) {
    const int s0 = todo[w].first, s1 = todo[w].second;
    ChunkPlan pl;
    collect(t, s0, s1, pl);
    plan_chunk(pl, 3 * n + 1, max_slots);
    Qmc2Chunk ch;
    ch.sec_begin = s0;
    ch.sec_end = s1;
    ch.nslots = pl.nslots;
    ch.prog_off = (uint32_t)t->image2.size();
    Qmc2ChunkHdr chh = {(uint32_t)pl.nslots, (uint32_t)pl.prog.size(), (uint32_t)pl.first_prod, 0u};
    put(t->image2, chh);
    for (auto &pr : pl.prog) {
      put(t->image2, (uint16_t)(pr.first * QMC2_THREADS));
      put(t->image2, (uint16_t)(pr.second * QMC2_THREADS));
    }
    while (t->image2.size() % 16) t->image2.push_back(0);
    ch.prog_bytes = (uint32_t)t->image2.size() - ch.prog_off;
    std::vector<uint32_t> prog4;
    for (auto &pr : pl.prog) {
      put32(prog4, (uint32_t)pr.first * T4 * 8u);
      put32(prog4, (uint32_t)pr.second * T4 * 8u);
    }
    pad4(prog4);
    const size_t tab4_mark = t->tab4.size();
    const uint32_t ONE = (uint32_t)(3 * n) * QMC2_THREADS * 8u;
    size_t mi = 0;  // index into pl.mono, same order as collect()
    auto rec_of = [&](double c, const Factors &f) {
      Qmc2Rec r;
      r.c = c;
      r.s0 = f.size() > 0 ? (uint32_t)f[0] * QMC2_THREADS * 8u : ONE;
      r.s1 = f.size() > 1 ? (uint32_t)f[1] * QMC2_THREADS * 8u : ONE;
      return r;
    };
    bool too_many_locals = false;
    const size_t image_mark = t->image2.size();
    for (int si = s0; si < s1 && !too_many_locals; ++si) {
      const QmcSector &s = t->sectors[si];
      ch.cost += cost[si];
      // sector-local products for the monomials the chunk-wide slots leave with more than two factors
      std::vector<std::pair<uint8_t, uint8_t>> local;
      {
        size_t cnt_m = 1 + s.U.size() + s.F.size();
        for (size_t q = 0; q < cnt_m; ++q) {
          Factors &f = pl.mono[mi + q];
          while (f.size() > 2) {
            const std::pair<uint8_t, uint8_t> pr(f[0], f[1]);
            size_t id = 0;
            while (id < local.size() && local[id] != pr) ++id;
            if (id == local.size()) local.push_back(pr);
            f.erase(f.begin(), f.begin() + 2);
            f.insert(f.begin(), (uint8_t)(pl.nslots + id));  // may exceed the sorted order: only the first two are merged next
          }
        }
        if (local.size() > QMC2_MAXLOCAL || pl.nslots + (int)local.size() > 255) {
          too_many_locals = true;
          break;
        }
      }
      Qmc2SectorHdr h;
      std::memset(&h, 0, sizeof h);
      int pos_of[QMC_MAXDIM], k = 0;
      for (int j = 0; j < n; ++j) pos_of[j] = -1;
      for (int j = 0; j < n; ++j)
        if (s.alpha[j] == -1) {
          h.sing_ln[k] = (uint16_t)((n + j) * QMC2_THREADS);
          h.sing_inv[k] = (uint16_t)((2 * n + j) * QMC2_THREADS);
          h.beta[k] = (double)s.beta[j];
          h.invbeta[k] = 1.0 / (double)s.beta[j];
          pos_of[j] = k++;
        }
      h.nsing = (uint8_t)s.nsing;
      std::vector<Qmc2Rec> recs;
      recs.push_back(rec_of(1.0, pl.mono[mi++]));  // G0
      for (int j = 0; j < n; ++j)                  // L0 = sum over regular variables of beta_j ln t_j
        if (s.alpha[j] != -1 && s.beta[j] != 0) {
          Qmc2Rec r;
          r.c = (double)s.beta[j];
          r.s0 = (uint32_t)(n + j) * QMC2_THREADS * 8u;
          r.s1 = ONE;
          recs.push_back(r);
          ++h.nL0;
        }
      for (int which = 0; which < 2; ++which) {
        const std::vector<QmcMono> &M = which ? s.F : s.U;  // already group-sorted by qmc_build_tables
        int gprev = 0;
        for (const QmcMono &m : M) {
          int g = 0;
          for (int j = 0; j < n; ++j)
            if (m.e[j] && pos_of[j] >= 0) g |= 1 << pos_of[j];
          if (g < gprev) return QMC_EINVAL;  // monomials must arrive sorted by group
          gprev = g;
          uint8_t &c = (which ? h.cntF : h.cntU)[g];
          if (c == 255) return QMC_EUNSUPPORTED;
          ++c;
          recs.push_back(rec_of(m.c, pl.mono[mi++]));
        }
      }
      h.nrec = (uint16_t)recs.size();
      h.nlocal = (uint8_t)local.size();
      ch.max_local = std::max(ch.max_local, (int)local.size());
      t->secoff2[si] = (uint32_t)t->image2.size();
      put(t->image2, h);
      for (auto &pr : local) {
        put(t->image2, (uint16_t)(pr.first * QMC2_THREADS));
        put(t->image2, (uint16_t)(pr.second * QMC2_THREADS));
      }
      while (t->image2.size() % 16) t->image2.push_back(0);
      for (const Qmc2Rec &r : recs) put(t->image2, r);
      t->secend2[si] = (uint32_t)t->image2.size();
      {  // version-4 block of the same sector (layout: qmc_launch.h)
        std::vector<uint32_t> &v = t->tab4;
        if ((int)t->secoff4.size() <= si) t->secoff4.resize(si + 1, 0);
        t->secoff4[si] = (uint32_t)(v.size() / 4);
        const size_t b0 = v.size();
        const int nc = 1 << s.nsing;
        const uint32_t nlw = (uint32_t)((local.size() + 1) / 2);
        put32(v, (uint32_t)s.nsing | ((uint32_t)h.nL0 << 8) | ((uint32_t)local.size() << 16));
        put32(v, 0);         // size of the block in words (patched below)
        put32(v, 9 + nlw);   // first record
        put32(v, 0);
        for (int k = 0; k < QMC_MAXSING; ++k) put32(v, (uint32_t)(h.sing_ln[k] / QMC2_THREADS) * T4 * 8u);
        for (int k = 0; k < QMC_MAXSING; ++k) put32(v, (uint32_t)(h.sing_inv[k] / QMC2_THREADS) * T4 * 8u);
        for (int k = 0; k < QMC_MAXSING; ++k) putf64(v, h.invbeta[k]);
        for (int k = 0; k < QMC_MAXSING; ++k) putf64(v, h.beta[k]);
        uint8_t extraU[16] = {0}, extraF[16] = {0};
        for (int g = 0; g < nc; ++g) {
          extraU[g] = h.cntU[g] ? (uint8_t)(h.cntU[g] - 1) : 0;
          extraF[g] = h.cntF[g] ? (uint8_t)(h.cntF[g] - 1) : 0;
        }
        for (int q = 0; q < 4; ++q) put32(v, extraU[4 * q] | (extraU[4 * q + 1] << 8) | (extraU[4 * q + 2] << 16) | ((uint32_t)extraU[4 * q + 3] << 24));
        for (int q = 0; q < 4; ++q) put32(v, extraF[4 * q] | (extraF[4 * q + 1] << 8) | (extraF[4 * q + 2] << 16) | ((uint32_t)extraF[4 * q + 3] << 24));
        for (auto &pr : local) {
          put32(v, (uint32_t)pr.first * T4 * 8u);
          put32(v, (uint32_t)pr.second * T4 * 8u);
        }
        pad4(v);
        size_t ri = 0;
        put_rec(v, recs[ri++], T4);                                  // G0
        for (int q = 0; q < h.nL0; ++q) put_rec(v, recs[ri++], T4);  // L0
        const Qmc2Rec empty = {0.0, ONE, ONE};
        std::vector<Qmc2Rec> extra;
        for (int which = 0; which < 2; ++which)
          for (int g = 0; g < nc; ++g) {
            const int cnt = (which ? h.cntF : h.cntU)[g];
            put_rec(v, cnt ? recs[ri] : empty, T4);
            for (int q = 1; q < cnt; ++q) extra.push_back(recs[ri + q]);
            ri += cnt;
          }
        for (const Qmc2Rec &r : extra) put_rec(v, r, T4);
        put_rec(v, empty, T4);  // sentinels: the kernel requests operands one record and offsets two records past the last
        put_rec(v, empty, T4);
        v[b0 + 1] = (uint32_t)((v.size() - b0) / 4);
      }
    }
    if (too_many_locals) {  // split the range in two and plan again
      t->image2.resize(ch.prog_off);
      t->tab4.resize(tab4_mark);
      (void)image_mark;
      if (s1 - s0 == 1) return QMC_EUNSUPPORTED;
      const int mid = (s0 + s1) / 2;
      todo[w] = {s0, mid};
      todo.insert(todo.begin() + w + 1, {mid, s1});
      --w;
      continue;
    }
    t->chunks.push_back(ch);
    t->prog4.push_back(prog4);
  }
  t->secoff2[nsec] = (uint32_t)t->image2.size();
  t->secoff4.resize(nsec + 1, 0);
  t->secoff4[nsec] = (uint32_t)(t->tab4.size() / 4);
  return QMC_OK;
}
