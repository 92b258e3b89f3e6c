// Sector tables of the real (Euclidean) path, "version 4": chunks, per-chunk slot programs, 8-byte monomial records.
// Host only.  Layout: qmc_launch.h; rationale: DESIGN.md "Data layout".
//
// Every thread keeps, per lattice point, a column of per-point values ("slots") in shared memory:
//   [0,n) t_j | [n,2n) ln t_j | 2n: 1.0 | 2n+1: 0.0 | coefficient constants | chunk products | sector-local products
// A monomial c * prod t_j^e_j is a multiset of FACTORS: the variables repeated by exponent and -- when c != 1 -- one
// symbol for the constant c, which owns a slot of its own.  A byte-pair-encoding style pass over the chunk's monomials
// (most frequent pair of factors first) turns pairs of factors into product slots, computed once per lattice point,
// until every monomial is a product of at most two slots.  A monomial is then ONE 8-byte record {u32 off0, u32 off1}:
// value = slot[off0] * slot[off1], accumulated with a single FMA -- the coefficient travels inside a slot.
// The records of a sector sit at DENSE POSITIONS: group g of polynomial q owns qmc4_cap(nsing, q, popcount g) positions
// (qmc_tables.h), which the kernel evaluates in straight-line code.  A group with more monomials than positions sums the
// overflow into a sector-local slot first ("fused" local entries slot = a*b + c*d; further monomials chain slot = slot*1 +
// c*d), and its last position reads that slot.
// To keep the constants few, every sector's U^ and F^ are divided by their most frequent |coefficient| c_U, c_F
// (U^ = c_U U', F^ = c_F F'): W picks up the factor c_U^aU0 c_F^aF0 (folded into the coefficient of G0) and Lambda the
// constant aU1 ln c_U + aF1 ln c_F (folded into L0).  On the double box every coefficient of U' is 1 and F' has one
// monomial with coefficient 1/3.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "../../include/qmc_feynman.h"
#include "qmc_bpe.h"
#include "qmc_tables.h"

using namespace qmcbpe;

namespace {

// relative cost of one sector at one point, fitted to measured per-chunk kernel times on B200:
// time ~ 7.8 per corner (reciprocal, logarithm, series, its share of the fold) + 1 per record
double sector_cost(const QmcSector &s, int kmax) {
  const int nc = 1 << s.nsing;
  return 7.8 * nc * (1.0 + 0.15 * kmax) + (double)(s.U.size() + s.F.size() + 2);
}

// most frequent |coefficient| of a polynomial (ties: the one met first)
double common_coefficient(const std::vector<QmcMono> &M) {
  double best = 1.0;
  int best_cnt = 0;
  for (size_t i = 0; i < M.size(); ++i) {
    const double a = std::fabs(M[i].c);
    int cnt = 0;
    for (const QmcMono &m : M) cnt += std::fabs(m.c) == a;
    if (cnt > best_cnt) {
      best_cnt = cnt;
      best = a;
    }
  }
  return best;
}

double ipow(double x, int e) {
  double r = 1.0;
  for (int i = 0; i < std::abs(e); ++i) r *= x;
  return e < 0 ? 1.0 / r : r;
}

struct ChunkConsts {
  std::vector<double> val;  // constants other than 1.0, slot 3n + 2 + index
  int id(double c) {
    for (size_t i = 0; i < val.size(); ++i)
      if (val[i] == c) return (int)i;
    val.push_back(c);
    return (int)val.size() - 1;
  }
};

// factors of all monomials of sectors [s0, s1), in the order [G0, U^ ..., F^ ...] per sector.
// G0 = prod_{regular j} t_j^alpha_j  (the kernel multiplies the 1/t_j of the singular variables, Eq. 12, factored out of the
// fold, qmc_fold.cuh, onto it)
bool collect(const qmc_tables *t, int s0, int s1, ChunkPlan &pl, ChunkConsts &cc, std::vector<double> &cU, std::vector<double> &cF) {
  pl.mono.clear();
  cc.val.clear();
  cU.clear();
  cF.clear();
  const int n = t->n;
  for (int si = s0; si < s1; ++si) {
    const QmcSector &s = t->sectors[si];
    Factors g;
    for (int j = 0; j < n; ++j)
      for (int q = 0; q < s.alpha[j]; ++q) g.push_back((uint8_t)j);
    std::sort(g.begin(), g.end());
    pl.mono.push_back(g);
    const double cu = common_coefficient(s.U), cf = common_coefficient(s.F);
    cU.push_back(cu);
    cF.push_back(cf);
    for (int which = 0; which < 2; ++which)
      for (const QmcMono &m : (which ? s.F : s.U)) {
        Factors f = factors_of(m.e, n);
        const double c = m.c / (which ? cf : cu);
        if (c != 1.0) {
          const int id = cc.id(c);
          if (id >= QMC4_MAXCONST) return false;
          f.push_back((uint8_t)(2 * n + 2 + id));
        }
        std::sort(f.begin(), f.end());
        pl.mono.push_back(f);
      }
  }
  return true;
}

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

int qmc_build_tables4(qmc_tables *t, int slot_budget, int chunk_bytes_opt, int threads_opt, int tpl_opt) {
  build_logtab4(t->logtab4);
  t->tab4.clear();
  t->secoff4.clear();
  t->prog4.clear();
  t->const4.clear();
  t->chunks.clear();
  t->sec_cost.clear();
  {
    // Threads per block of the real-path kernel, measured on B200 (kernels): tables dominated by sectors
    // with three or four singular variables execute long straight-line code paths, and one 512-thread block per SM (all
    // 16 warps walking the same sectors) fetches instructions better than four independent 128-thread blocks; tables of
    // short paths prefer the small blocks.
    int big = 0;
    for (const QmcSector &s : t->sectors) big += s.nsing >= 3;
    t->threads_real = 2 * big >= (int)t->sectors.size() ? QMC4_TBIG : 128;
    if (threads_opt == 128) t->threads_real = 128;
    if (threads_opt == 512) t->threads_real = QMC4_TBIG;
  }
  const uint32_t T4 = (uint32_t)t->threads_real;
  const int n = t->n, nsec = (int)t->sectors.size();
  if (t->lambda > 0.0 || nsec == 0) return QMC_OK;
  {
    // dense-position template (qmc_tables.h): the one with the lower modelled instruction count over all sectors --
    // 3.5 per position (its share of the table load, two slot loads, one multiply-add), 13 per monomial beyond a group's
    // positions (a fused sector-local entry)
    double cost_tpl[2] = {0.0, 0.0};
    for (const QmcSector &s : t->sectors) {
      int pos_of[QMC_MAXDIM], k = 0;
      for (int j = 0; j < n; ++j) pos_of[j] = s.alpha[j] == -1 ? k++ : -1;
      for (int which = 0; which < 2; ++which) {
        int cnt[1 << QMC_MAXSING] = {0};
        for (const QmcMono &m : (which ? s.F : s.U)) {
          int g = 0;
          for (int j = 0; j < n; ++j)
            if (m.e[j] && pos_of[j] >= 0) g |= 1 << pos_of[j];
          ++cnt[g];
        }
        for (int tpl = 0; tpl < 2; ++tpl)
          for (int g = 0; g < (1 << s.nsing); ++g) {
            const int cap = qmc4_cap(tpl, s.nsing, which, qmc4_popc(g));
            cost_tpl[tpl] += 3.5 * cap + 13.0 * std::max(0, cnt[g] - cap);
          }
      }
    }
    t->tpl_real = cost_tpl[1] < cost_tpl[0] ? 1 : 0;
    if (tpl_opt == 1 || tpl_opt == 2) t->tpl_real = tpl_opt - 1;
  }
  if (2 * n + 2 >= QMC2_MAXSLOTS) return QMC_EUNSUPPORTED;

  // ---- chunk boundaries: contiguous ranges of about equal modelled cost, about chunk_bytes of tables each ------
  std::vector<double> cost(nsec);
  double total_cost = 0.0, total_bytes = 0.0;
  for (int i = 0; i < nsec; ++i) {
    const QmcSector &s = t->sectors[i];
    cost[i] = sector_cost(s, t->kmax);
    t->sec_cost.push_back(cost[i]);
    total_cost += cost[i];
    total_bytes += 16.0 * (11 + n) + 8.0 * qmc4_pos(t->tpl_real, s.nsing, 1, 1 << s.nsing);
  }
  // 44 chunk-wide slots (+ the coefficient constants) + up to 8 sector-local ones: 53 columns of 8 T bytes = 212 KB at
  // T = 512 (one block per SM); the more slots, the fewer sector-local products and chunks (measured on B200, cfg4:
  // 32 / 36 / 40 / 44 slots -> 232 / 211 / 187 / 183 ms per step)
  const int max_slots_base = slot_budget > 0 ? slot_budget : 44;
  const double chunk_bytes = chunk_bytes_opt > 0 ? std::max(1000.0, (double)chunk_bytes_opt) : 24000.0;
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
  t->secoff4.assign(nsec + 1, 0);
  for (size_t w = 0; w < todo.size(); ++w) {
    const int s0 = todo[w].first, s1 = todo[w].second;
    ChunkPlan pl;
    ChunkConsts cc;
    std::vector<double> cU, cF;
    if (!collect(t, s0, s1, pl, cc, cU, cF)) return QMC_EUNSUPPORTED;
    const int nconst = (int)cc.val.size();
    const int first_prod = 2 * n + 2 + nconst;
    const int max_slots = std::min(QMC2_MAXSLOTS - QMC2_MAXLOCAL, std::max(max_slots_base + std::min(nconst, 6), first_prod + 1));
    plan_chunk(pl, first_prod, max_slots, true);  // a record costs the same with one factor or two: stop at two
    Qmc2Chunk ch;
    ch.sec_begin = s0;
    ch.sec_end = s1;
    ch.nslots = pl.nslots;
    ch.nconst = nconst;
    std::vector<uint32_t> prog4;
    for (auto &pr : pl.prog) {
      put32(prog4, (uint32_t)pr.first * T4 * 8u);
      put32(prog4, (uint32_t)pr.second * T4 * 8u);
    }
    pad4(prog4);
    const size_t tab4_mark = t->tab4.size();
    const uint32_t ONE = (uint32_t)(2 * n) * T4 * 8u, ZERO = (uint32_t)(2 * n + 1) * T4 * 8u;
    size_t mi = 0;  // index into pl.mono, same order as collect()
    auto put_rec = [&](std::vector<uint32_t> &v, const Factors &f) {
      v.push_back(f.size() > 0 ? (uint32_t)f[0] * T4 * 8u : ONE);
      v.push_back(f.size() > 1 ? (uint32_t)f[1] * T4 * 8u : ONE);
    };
    bool too_many_locals = false;
    for (int si = s0; si < s1 && !too_many_locals; ++si) {
      const QmcSector &s = t->sectors[si];
      ch.cost += cost[si];
      // sector-local products for the monomials the chunk-wide slots leave with more than two factors
      std::vector<std::pair<uint8_t, uint8_t>> local;
      {
        const size_t cnt_m = 1 + s.U.size() + s.F.size();
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
        if (local.size() > QMC2_MAXLOCAL || pl.nslots + (int)local.size() > QMC2_MAXSLOTS) {
          too_many_locals = true;
          break;
        }
      }
      int pos_of[QMC_MAXDIM], k = 0;
      uint32_t sing_ln[QMC_MAXSING] = {0}, sing_t[QMC_MAXSING] = {0};
      double invbeta[QMC_MAXSING] = {0}, beta[QMC_MAXSING] = {0};
      for (int j = 0; j < n; ++j) pos_of[j] = -1;
      for (int j = 0; j < n; ++j)
        if (s.alpha[j] == -1) {
          sing_ln[k] = (uint32_t)(n + j) * T4 * 8u;
          sing_t[k] = (uint32_t)j * T4 * 8u;
          beta[k] = (double)s.beta[j];
          invbeta[k] = 1.0 / (double)s.beta[j];
          pos_of[j] = k++;
        }
      for (; k < QMC_MAXSING; ++k) sing_ln[k] = sing_t[k] = ONE;
      const int ns = s.nsing, nc = 1 << ns;
      // monomials per group (qmc_build_tables sorted them by group)
      std::vector<const Factors *> grp[2][1 << QMC_MAXSING];
      const Factors &g0f = pl.mono[mi++];
      for (int which = 0; which < 2; ++which) {
        int gprev = 0;
        for (const QmcMono &m : (which ? s.F : s.U)) {
          int g = 0;
          for (int j = 0; j < n; ++j)
            if (m.e[j] && pos_of[j] >= 0) g |= 1 << pos_of[j];
          if (g < gprev) return QMC_EINVAL;  // monomials must arrive sorted by group
          gprev = g;
          grp[which][g].push_back(&pl.mono[mi++]);
        }
      }
      // dense positions; overflowing groups sum their surplus into a sector-local slot (fused entries)
      struct Fused { uint32_t a, b, c, d, dst; };
      std::vector<Fused> fused;
      std::vector<uint32_t> posrec;  // {off0, off1} per position
      auto off_of = [&](const Factors &f, int i) { return (int)f.size() > i ? (uint32_t)f[i] * T4 * 8u : ONE; };
      int nlocal_slots = (int)local.size();
      for (int which = 0; which < 2 && !too_many_locals; ++which)
        for (int g = 0; g < nc; ++g) {
          const int cap = qmc4_cap(t->tpl_real, ns, which, qmc4_popc(g));
          const std::vector<const Factors *> &R = grp[which][g];
          const int cnt = (int)R.size();
          ch.nrec += cnt;
          for (const Factors *f : R) ch.nsingle += f->size() < 2;
          if (cap < 1) return QMC_EUNSUPPORTED;
          if (cnt <= cap) {
            for (int q = 0; q < cap; ++q) {
              posrec.push_back(q < cnt ? off_of(*R[q], 0) : ZERO);
              posrec.push_back(q < cnt ? off_of(*R[q], 1) : ZERO);
            }
          } else {
            for (int q = 0; q < cap - 1; ++q) {
              posrec.push_back(off_of(*R[q], 0));
              posrec.push_back(off_of(*R[q], 1));
            }
            if (nlocal_slots >= QMC2_MAXLOCAL || pl.nslots + nlocal_slots >= QMC2_MAXSLOTS) {
              too_many_locals = true;
              break;
            }
            const uint32_t dst = (uint32_t)(pl.nslots + nlocal_slots) * T4 * 8u;
            ++nlocal_slots;
            int q = cap - 1;
            fused.push_back({off_of(*R[q], 0), off_of(*R[q], 1), off_of(*R[q + 1], 0), off_of(*R[q + 1], 1), dst});
            for (q += 2; q < cnt; ++q) fused.push_back({dst, ONE, off_of(*R[q], 0), off_of(*R[q], 1), dst});
            posrec.push_back(dst);
            posrec.push_back(ONE);
            ch.noverflow += cnt - cap;
          }
        }
      if (too_many_locals) break;
      if (posrec.size() % 4) {  // pad to a whole 16-byte word
        posrec.push_back(ONE);
        posrec.push_back(ONE);
      }
      ch.nlocal += (int)local.size();
      ch.max_local = std::max(ch.max_local, nlocal_slots);
      // ---- the sector block (layout: qmc_launch.h) ----
      std::vector<uint32_t> &v = t->tab4;
      t->secoff4[si] = (uint32_t)(v.size() / 4);
      const size_t b0 = v.size();
      const int nL0 = n - ns;  // one record per regular variable
      const uint32_t nlw = (uint32_t)((local.size() + 1) / 2);
      put32(v, (uint32_t)ns | ((uint32_t)nL0 << 8) | ((uint32_t)local.size() << 16) | ((uint32_t)fused.size() << 24));
      put32(v, 0);                                                    // size of the block in words (patched below)
      put32(v, 9 + (uint32_t)nL0 + nlw + 2u * (uint32_t)fused.size());  // first dense position
      put32(v, 0);
      for (int q = 0; q < QMC_MAXSING; ++q) put32(v, sing_ln[q]);
      for (int q = 0; q < QMC_MAXSING; ++q) put32(v, sing_t[q]);
      for (int q = 0; q < QMC_MAXSING; ++q) putf64(v, invbeta[q]);
      for (int q = 0; q < QMC_MAXSING; ++q) putf64(v, beta[q]);
      const double cu = cU[si - s0], cf = cF[si - s0];
      putf64(v, ipow(cu, t->aU0) * ipow(cf, t->aF0));  // w7: coefficient of G0, then its two slots
      v.push_back(off_of(g0f, 0));
      v.push_back(off_of(g0f, 1));
      putf64(v, t->aU1 * std::log(cu) + t->aF1 * std::log(cf));  // w8: constant of L0
      put32(v, 0);
      put32(v, 0);
      for (int j = 0; j < n; ++j)  // w9..: L0 = constant + sum over regular variables of beta_j ln t_j
        if (s.alpha[j] != -1) {
          putf64(v, (double)s.beta[j]);
          put32(v, (uint32_t)(n + j) * T4 * 8u);
          put32(v, 0);
        }
      for (auto &pr : local) {
        put32(v, (uint32_t)pr.first * T4 * 8u);
        put32(v, (uint32_t)pr.second * T4 * 8u);
      }
      pad4(v);
      for (const Fused &fu : fused) {
        put32(v, fu.a); put32(v, fu.b); put32(v, fu.c); put32(v, fu.d);
        put32(v, fu.dst); put32(v, 0); put32(v, 0); put32(v, 0);
      }
      for (uint32_t x : posrec) v.push_back(x);
      v[b0 + 1] = (uint32_t)((v.size() - b0) / 4);
    }
    if (too_many_locals) {  // split the range in two and plan again
      t->tab4.resize(tab4_mark);
      if (s1 - s0 == 1) return QMC_EUNSUPPORTED;
      const int mid = (s0 + s1) / 2;
      todo[w] = {s0, mid};
      todo.insert(todo.begin() + w + 1, {mid, s1});
      --w;
      continue;
    }
    ch.tab_words = (uint32_t)((t->tab4.size() - tab4_mark) / 4);
    t->chunks.push_back(ch);
    t->prog4.push_back(prog4);
    t->const4.push_back(cc.val);
  }
  t->secoff4[nsec] = (uint32_t)(t->tab4.size() / 4);
  return QMC_OK;
}
