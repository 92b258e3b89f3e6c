// Version-3 device image of the sector tables (complex path, contour deformation Eq. 14).  Host only.
// Layout in qmc_tables.h.  The gradient and the Hessian of F^ (needed for rho_j, z_j and the Jacobian, R:C12) are
// emitted as polynomials of their own: d/dt_i (c prod t^e) = c e_i t^(e - 1_i), and likewise for second derivatives.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "../../include/qmc_feynman.h"
#include "qmc_bpe.h"
#include "qmc_tables.h"

using namespace qmcbpe;

namespace {

struct Mono3 {
  double c;
  uint8_t e[QMC_MAXDIM];
  int group;
};
typedef std::vector<Mono3> Poly3;

// polynomials of one sector in emission order: F_1..F_n, F_11, F_12, .., F_nn, U, F
void sector_polys(const QmcSector &s, int n, const int *pos_of, std::vector<Poly3> &out) {
  auto group_of = [&](const uint8_t *e) {
    int g = 0;
    for (int j = 0; j < n; ++j)
      if (e[j] && pos_of[j] >= 0) g |= 1 << pos_of[j];
    return g;
  };
  auto push = [&](Poly3 &P, double c, const uint8_t *e) {
    Mono3 m;
    m.c = c;
    std::memset(m.e, 0, sizeof m.e);
    for (int j = 0; j < n; ++j) m.e[j] = e[j];
    m.group = group_of(m.e);
    P.push_back(m);
  };
  out.clear();
  for (int i = 0; i < n; ++i) {
    Poly3 P;
    for (const QmcMono &m : s.F)
      if (m.e[i] >= 1) {
        uint8_t e[QMC_MAXDIM];
        std::memcpy(e, m.e, sizeof e);
        e[i] -= 1;
        push(P, m.c * m.e[i], e);
      }
    out.push_back(P);
  }
  for (int i = 0; i < n; ++i)
    for (int k = i; k < n; ++k) {
      Poly3 P;
      for (const QmcMono &m : s.F) {
        uint8_t e[QMC_MAXDIM];
        std::memcpy(e, m.e, sizeof e);
        double c;
        if (i == k) {
          if (m.e[i] < 2) continue;
          c = m.c * m.e[i] * (m.e[i] - 1);
          e[i] -= 2;
        } else {
          if (m.e[i] < 1 || m.e[k] < 1) continue;
          c = m.c * m.e[i] * m.e[k];
          e[i] -= 1;
          e[k] -= 1;
        }
        push(P, c, e);
      }
      out.push_back(P);
    }
  for (int which = 0; which < 2; ++which) {
    Poly3 P;
    for (const QmcMono &m : (which ? s.F : s.U)) push(P, m.c, m.e);
    out.push_back(P);
  }
  for (Poly3 &P : out)
    std::stable_sort(P.begin(), P.end(), [](const Mono3 &a, const Mono3 &b) { return a.group < b.group; });
}

void positions(const QmcSector &s, int n, int *pos_of) {
  int k = 0;
  for (int j = 0; j < n; ++j) pos_of[j] = (s.alpha[j] == -1) ? k++ : -1;
}

// make every monomial a product of at most two slots, adding sector-local products; false if too many are needed
bool localise(std::vector<Factors> &mono, size_t first, size_t count, int nslots, std::vector<std::pair<uint8_t, uint8_t>> &local) {
  for (size_t q = 0; q < count; ++q) {
    Factors &f = mono[first + q];
    while (f.size() > 2) {
      const std::pair<uint8_t, uint8_t> pr(f[0], f[1]);
      size_t id = 0;
      while (id < local.size() && local[id] != pr) ++id;
      if (id == local.size()) local.push_back(pr);
      f.erase(f.begin(), f.begin() + 2);
      f.insert(f.begin(), (uint8_t)(nslots + id));
    }
  }
  return local.size() <= QMC3_MAXLOCAL && nslots + (int)local.size() <= 255;
}

}  // namespace

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
void put_rec(std::vector<uint32_t> &v, const Qmc2Rec &r) {
  putf64(v, r.c);
  v.push_back(r.s0);
  v.push_back(r.s1);
}
}  // namespace

int qmc_build_image3(qmc_tables *t, int slots_r_opt, int slots_c_opt, int chunk_bytes_opt) {
  t->tab5.clear();
  t->secoff5.clear();
  t->prog5r.clear();
  t->prog5c.clear();
  t->image3.clear();
  t->secoff3.clear();
  t->secend3.clear();
  t->chunks3.clear();
  t->chunk3_nslots_c.clear();
  t->chunk3_max_local_c.clear();
  t->rec_flops5.assign(t->sectors.size(), 0.0);
  const int n = t->n, nsec = (int)t->sectors.size();
  if (!(t->lambda > 0.0) || nsec == 0) return QMC_OK;
  const int T = QMC3_THREADS;
  const int npoly = n + n * (n + 1) / 2 + 2, nderiv = npoly - 2;
  int max_r = std::min(QMC3_MAXSLOTS_R, 2 * n + 1 + 20), max_c = std::min(QMC3_MAXSLOTS_C, n + 1 + 12);
  if (n == 5) {
    // n = 5 runs three 128-thread blocks per SM (168 registers, qmc_kernels5.cuh), which needs <= 75 KB of shared memory per
    // block: 8 KB logarithm table + 1 KB per real slot + 2 KB per complex slot.  Measured on B200 (cfg5, ms per step):
    // budgets 31/18 (two blocks) 202; 24/14 151; 21/14 152; 19/13 153; 21/15 (76 KB: two blocks again) 203
    max_r = 2 * n + 1 + 13;
    max_c = n + 1 + 8;
  }
  double chunk_bytes = 16000.0;
  if (slots_r_opt > 0) max_r = std::min(QMC3_MAXSLOTS_R, std::max(2 * n + 2, slots_r_opt));
  if (slots_c_opt > 0) max_c = std::min(QMC3_MAXSLOTS_C, std::max(n + 2, slots_c_opt));
  if (chunk_bytes_opt > 0) chunk_bytes = std::max(1000.0, (double)chunk_bytes_opt);

  // ---- per-sector polynomials, chunk ranges by table bytes ------------------------------------------------------
  std::vector<std::vector<Poly3>> polys(nsec);
  std::vector<double> bytes(nsec);
  if (t->sec_cost.size() != (size_t)nsec) t->sec_cost.assign(nsec, 0.0);
  for (int si = 0; si < nsec; ++si) {
    int pos_of[QMC_MAXDIM];
    positions(t->sectors[si], n, pos_of);
    sector_polys(t->sectors[si], n, pos_of, polys[si]);
    size_t nrec = 1 + n;
    for (const Poly3 &P : polys[si]) nrec += P.size();
    bytes[si] = sizeof(Qmc3SectorHdr) + npoly * (1 << t->sectors[si].nsing) + 64 + 16.0 * (nrec + nderiv / 2);
    t->sec_cost[si] = (double)(1 << t->sectors[si].nsing) * (nrec + 400.0);
  }
  std::vector<std::pair<int, int>> todo;
  for (int b = 0; b < nsec;) {
    int e = b;
    double acc = 0.0;
    while (e < nsec && (acc + bytes[e] <= chunk_bytes || e == b)) acc += bytes[e++];
    todo.push_back({b, e});
    b = e;
  }
  t->secoff3.assign(nsec + 1, 0);
  t->secend3.assign(nsec, 0);
  for (size_t w = 0; w < todo.size(); ++w) {
    const int s0 = todo[w].first, s1 = todo[w].second;
    // ---- plan the two slot programs of the chunk ------------------------------------------------------------
    ChunkPlan pr, pc;  // monomial order: per sector [G0][derivative polynomials...] resp. [U][F]
    for (int si = s0; si < s1; ++si) {
      const QmcSector &s = t->sectors[si];
      uint8_t g[QMC_MAXDIM] = {0};
      for (int j = 0; j < n; ++j) g[j] = (uint8_t)(s.alpha[j] > 0 ? s.alpha[j] : 0);
      pr.mono.push_back(factors_of(g, n));
      for (int p = 0; p < nderiv; ++p)
        for (const Mono3 &m : polys[si][p]) pr.mono.push_back(factors_of(m.e, n));
      for (int p = nderiv; p < npoly; ++p)
        for (const Mono3 &m : polys[si][p]) pc.mono.push_back(factors_of(m.e, n));
    }
    plan_chunk(pr, 2 * n + 1, max_r);
    plan_chunk(pc, n + 1, max_c);
    // ---- emit --------------------------------------------------------------------------------------------------
    Qmc2Chunk ch;
    ch.sec_begin = s0;
    ch.sec_end = s1;
    ch.nslots = pr.nslots;
    ch.prog_off = (uint32_t)t->image3.size();
    Qmc3ChunkHdr chh;
    std::memset(&chh, 0, sizeof chh);
    chh.nslots_r = pr.nslots; chh.nprog_r = (uint32_t)pr.prog.size(); chh.first_prod_r = pr.first_prod;
    chh.nslots_c = pc.nslots; chh.nprog_c = (uint32_t)pc.prog.size(); chh.first_prod_c = pc.first_prod;
    put(t->image3, chh);
    for (auto &q : pr.prog) { put(t->image3, (uint16_t)q.first); put(t->image3, (uint16_t)q.second); }
    while (t->image3.size() % 16) t->image3.push_back(0);
    for (auto &q : pc.prog) { put(t->image3, (uint16_t)q.first); put(t->image3, (uint16_t)q.second); }
    while (t->image3.size() % 16) t->image3.push_back(0);
    ch.prog_bytes = (uint32_t)t->image3.size() - ch.prog_off;
    std::vector<uint32_t> p5r, p5c;
    for (auto &q : pr.prog) { put32(p5r, (uint32_t)q.first * T * 8u); put32(p5r, (uint32_t)q.second * T * 8u); }
    pad4(p5r);
    for (auto &q : pc.prog) { put32(p5c, (uint32_t)q.first * T * 16u); put32(p5c, (uint32_t)q.second * T * 16u); }
    pad4(p5c);
    const size_t tab5_mark = t->tab5.size();
    const uint32_t ONE_R = (uint32_t)(2 * n) * T * 8u, ONE_C = (uint32_t)n * T * 16u;
    auto rec_r = [&](double c, const Factors &f) {
      Qmc2Rec r;
      r.c = c;
      r.s0 = f.size() > 0 ? (uint32_t)f[0] * T * 8u : ONE_R;
      r.s1 = f.size() > 1 ? (uint32_t)f[1] * T * 8u : ONE_R;
      return r;
    };
    auto rec_c = [&](double c, const Factors &f) {
      Qmc2Rec r;
      r.c = c;
      r.s0 = f.size() > 0 ? (uint32_t)f[0] * T * 16u : ONE_C;
      r.s1 = f.size() > 1 ? (uint32_t)f[1] * T * 16u : ONE_C;
      return r;
    };
    size_t mr = 0, mc = 0;
    bool split = false;
    int max_local_c = 0;
    for (int si = s0; si < s1 && !split; ++si) {
      const QmcSector &s = t->sectors[si];
      const int ng = 1 << s.nsing;
      size_t cnt_r = 1, cnt_c = 0;
      for (int p = 0; p < nderiv; ++p) cnt_r += polys[si][p].size();
      for (int p = nderiv; p < npoly; ++p) cnt_c += polys[si][p].size();
      std::vector<std::pair<uint8_t, uint8_t>> loc_r, loc_c;
      if (!localise(pr.mono, mr, cnt_r, pr.nslots, loc_r) || !localise(pc.mono, mc, cnt_c, pc.nslots, loc_c)) {
        split = true;
        break;
      }
      Qmc3SectorHdr h;
      std::memset(&h, 0, sizeof h);
      h.nsing = (uint8_t)s.nsing;
      int k = 0;
      for (int j = 0; j < n; ++j) {
        h.alpha[j] = (int8_t)s.alpha[j];
        h.beta[j] = (int8_t)s.beta[j];
        if (s.alpha[j] == -1) {
          h.sing_var[k] = (uint8_t)j;
          h.betas[k] = (double)s.beta[j];
          h.invbeta[k] = 1.0 / (double)s.beta[j];
          ++k;
        }
      }
      std::vector<uint8_t> counts((size_t)npoly * ng, 0);
      std::vector<Qmc2Rec> rr, rc;
      rr.push_back(rec_r(1.0, pr.mono[mr++]));  // G0
      for (int j = 0; j < n; ++j)
        if (s.alpha[j] != -1 && s.beta[j] != 0) {  // L0 = sum over regular variables of beta_j ln t_j
          Qmc2Rec r;
          r.c = (double)s.beta[j];
          r.s0 = (uint32_t)(n + j) * T * 8u;
          r.s1 = ONE_R;
          rr.push_back(r);
          ++h.nL0;
        }
      for (int p = 0; p < npoly; ++p)
        for (const Mono3 &m : polys[si][p]) {
          uint8_t &c = counts[(size_t)p * ng + m.group];
          if (c == 255) return QMC_EUNSUPPORTED;
          ++c;
          if (p < nderiv) rr.push_back(rec_r(m.c, pr.mono[mr++]));
          else rc.push_back(rec_c(m.c, pc.mono[mc++]));
        }
      if (rr.size() > 65535 || rc.size() > 65535) return QMC_EUNSUPPORTED;
      h.nrec_r = (uint16_t)rr.size();
      h.nrec_c = (uint16_t)rc.size();
      h.nlocal_r = (uint8_t)loc_r.size();
      h.nlocal_c = (uint8_t)loc_c.size();
      ch.max_local = std::max(ch.max_local, (int)loc_r.size());
      max_local_c = std::max(max_local_c, (int)loc_c.size());
      ch.cost += t->sec_cost[si];
      t->secoff3[si] = (uint32_t)t->image3.size();
      put(t->image3, h);
      t->image3.insert(t->image3.end(), counts.begin(), counts.end());
      while (t->image3.size() % 16) t->image3.push_back(0);
      for (auto &q : loc_r) { put(t->image3, (uint16_t)q.first); put(t->image3, (uint16_t)q.second); }
      while (t->image3.size() % 16) t->image3.push_back(0);
      for (auto &q : loc_c) { put(t->image3, (uint16_t)q.first); put(t->image3, (uint16_t)q.second); }
      while (t->image3.size() % 16) t->image3.push_back(0);
      for (const Qmc2Rec &r : rr) put(t->image3, r);
      for (const Qmc2Rec &r : rc) put(t->image3, r);
      t->secend3[si] = (uint32_t)t->image3.size();
      {  // version-5 block of the same sector (layout: qmc_launch.h)
        std::vector<uint32_t> &v = t->tab5;
        if ((int)t->secoff5.size() <= si) t->secoff5.resize(si + 1, 0);
        t->secoff5[si] = (uint32_t)(v.size() / 4);
        const size_t b0 = v.size();
        const uint32_t nlr = (uint32_t)((loc_r.size() + 1) / 2), nlc = (uint32_t)((loc_c.size() + 1) / 2);
        put32(v, (uint32_t)s.nsing | ((uint32_t)h.nL0 << 8) | ((uint32_t)loc_r.size() << 16) | ((uint32_t)loc_c.size() << 24));
        put32(v, 0);                // size of the block in words (patched below)
        put32(v, 8 + nlr + nlc);    // first real record (G0)
        put32(v, 0);
        auto pack4 = [](const int8_t *a) {
          return (uint32_t)(uint8_t)a[0] | ((uint32_t)(uint8_t)a[1] << 8) | ((uint32_t)(uint8_t)a[2] << 16) | ((uint32_t)(uint8_t)a[3] << 24);
        };
        put32(v, (uint32_t)h.sing_var[0] | ((uint32_t)h.sing_var[1] << 8) | ((uint32_t)h.sing_var[2] << 16) | ((uint32_t)h.sing_var[3] << 24));
        put32(v, 0);
        put32(v, pack4(h.alpha));
        put32(v, pack4(h.alpha + 4));
        put32(v, pack4(h.beta));
        put32(v, pack4(h.beta + 4));
        put32(v, 0);
        put32(v, 0);
        for (int q = 0; q < QMC_MAXSING; ++q) putf64(v, h.invbeta[q]);
        for (int q = 0; q < QMC_MAXSING; ++q) putf64(v, h.betas[q]);
        const size_t dir = v.size();
        for (int q = 0; q < 4; ++q) put32(v, 0);  // corner directory (patched below)
        for (auto &q : loc_r) { put32(v, (uint32_t)q.first * T * 8u); put32(v, (uint32_t)q.second * T * 8u); }
        pad4(v);
        for (auto &q : loc_c) { put32(v, (uint32_t)q.first * T * 16u); put32(v, (uint32_t)q.second * T * 16u); }
        pad4(v);
        for (int q = 0; q < 1 + h.nL0; ++q) put_rec(v, rr[q]);  // G0, L0
        const Qmc2Rec empty_r = {0.0, ONE_R, ONE_R}, empty_c = {0.0, ONE_C, ONE_C};
        for (int Z = 0; Z < ng; ++Z) {
          v[dir + Z] = (uint32_t)((v.size() - b0) / 4);
          // the surviving records per polynomial (a monomial survives iff its group is disjoint from Z), by number of slot
          // factors: constants are summed on the spot (c0), one-factor records c * slot form stream A, two-factor records
          // c * slot * slot stream B.  Measured on cfg5: 12 % constants, 55 % one-factor, 29 % two-factor.
          std::vector<uint8_t> cA(npoly, 0), cB(npoly, 0);
          std::vector<double> c0(npoly, 0.0);
          std::vector<Qmc2Rec> rA, rB, kA, kB;  // real streams A, B; complex streams A, B
          size_t ir = 1 + h.nL0, ic = 0;
          for (int p = 0; p < npoly; ++p) {
            const bool real = p < nderiv;
            const uint32_t ONE = real ? ONE_R : ONE_C;
            for (const Mono3 &m : polys[si][p]) {
              const Qmc2Rec &r = real ? rr[ir++] : rc[ic++];
              if ((m.group & Z) != 0) continue;
              if (r.s0 == ONE && r.s1 == ONE) {
                c0[p] += r.c;
              } else if ((r.s1 == ONE || r.s0 == ONE) && (!real || cA[p] < qmc5_capA(n, t->L, p))) {
                Qmc2Rec q = {r.c, r.s1 == ONE ? r.s0 : r.s1, 0u};
                (real ? rA : kA).push_back(q);
                if (++cA[p] == 255) return QMC_EUNSUPPORTED;
              } else {  // (a one-factor record beyond the fixed positions of its polynomial travels as c * slot * 1)
                (real ? rB : kB).push_back(r);
                if (++cB[p] == 255) return QMC_EUNSUPPORTED;
              }
            }
          }
          if (Z == 0) t->rec_flops5[si] = 0.0;  // (a chunk that is split and planned again visits the sector twice)
          t->rec_flops5[si] += 2.0 * rA.size() + 3.0 * rB.size() + 4.0 * kA.size() + 10.0 * kB.size();  // (unused positions: not counted)
          for (int pass = 0; pass < 2; ++pass) {
            const std::vector<uint8_t> &cz = pass ? cB : cA;
            for (int p = 0; p < npoly; p += 4) {
              uint32_t w = 0;
              for (int q = 0; q < 4 && p + q < npoly; ++q) w |= (uint32_t)cz[p + q] << (8 * q);
              put32(v, w);
            }
            pad4(v);
          }
          for (int p = 0; p < npoly; ++p) putf64(v, c0[p]);
          pad4(v);
          // every stream ends with two sentinels: the kernel requests operands one record and table words two records ahead
          const Qmc2Rec sentA_r = {0.0, ONE_R, 0u}, sentA_c = {0.0, ONE_C, 0u};
          {  // real stream A: qmc5_capA fixed positions per derivative polynomial (rA is in polynomial order)
            size_t ia = 0;
            for (int p = 0; p < nderiv; ++p) {
              for (int k = 0; k < qmc5_capA(n, t->L, p); ++k) put_rec(v, k < cA[p] ? rA[ia + k] : sentA_r);
              ia += cA[p];
            }
          }
          for (const Qmc2Rec &r : rB) put_rec(v, r);
          put_rec(v, empty_r); put_rec(v, empty_r);
          for (const Qmc2Rec &r : kA) put_rec(v, r);
          put_rec(v, sentA_c); put_rec(v, sentA_c);
          for (const Qmc2Rec &r : kB) put_rec(v, r);
          put_rec(v, empty_c); put_rec(v, empty_c);
        }
        v[b0 + 1] = (uint32_t)((v.size() - b0) / 4);
      }
    }
    if (split) {
      t->image3.resize(ch.prog_off);
      t->tab5.resize(tab5_mark);
      if (s1 - s0 == 1) return QMC_EUNSUPPORTED;
      const int mid = (s0 + s1) / 2;
      todo[w] = {s0, mid};
      todo.insert(todo.begin() + w + 1, {mid, s1});
      --w;
      continue;
    }
    t->chunks3.push_back(ch);
    t->prog5r.push_back(p5r);
    t->prog5c.push_back(p5c);
    t->chunk3_nslots_c.push_back(pc.nslots);
    t->chunk3_max_local_c.push_back(max_local_c);
  }
  t->secoff3[nsec] = (uint32_t)t->image3.size();
  t->secoff5.resize(nsec + 1, 0);
  t->secoff5[nsec] = (uint32_t)(t->tab5.size() / 4);
  return QMC_OK;
}
