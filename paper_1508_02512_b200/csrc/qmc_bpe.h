// Byte-pair-encoding style planning of product slots (host only; shared by the table image builders).
// A monomial is a multiset of factors (slot ids; initially the variables, repeated by exponent); the most frequent pair
// of factors over a chunk becomes a new slot (their product, computed once per lattice point) and replaces the pair
// everywhere; repeat while slots are left and a new slot would serve at least two monomials.
#pragma once
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <vector>

#include "qmc_tables.h"

namespace qmcbpe {

typedef std::vector<uint8_t> Factors;  // sorted slot ids

struct ChunkPlan {
  int nslots = 0, first_prod = 0;
  std::vector<std::pair<uint8_t, uint8_t>> prog;  // slot[first_prod + i] = slot[a] * slot[b]
  std::vector<Factors> mono;                      // per monomial (order of collection)
};

inline Factors factors_of(const uint8_t *e, int n) {
  Factors f;
  for (int j = 0; j < n; ++j)
    for (int q = 0; q < e[j]; ++q) f.push_back((uint8_t)j);
  return f;
}

// replace every occurrence of the pair (a, b) in m by `nw`
inline void merge_pair(Factors &m, int a, int b, int nw) {
  for (;;) {
    auto ia = std::find(m.begin(), m.end(), (uint8_t)a);
    if (ia == m.end()) return;
    auto ib = (a == b) ? std::find(ia + 1, m.end(), (uint8_t)b) : std::find(m.begin(), m.end(), (uint8_t)b);
    if (ib == m.end()) return;
    if (ib < ia) std::swap(ia, ib);
    m.erase(ib);
    m.erase(ia);
    m.push_back((uint8_t)nw);
  }
}

// returns false if some monomial still has more than two factors when the slots run out
inline bool plan_chunk(ChunkPlan &pl, int first_prod, int max_slots, bool stop_at_two = false) {
  pl.first_prod = first_prod;
  pl.nslots = pl.first_prod;
  pl.prog.clear();
  for (;;) {
    static thread_local int cnt[QMC2_MAXSLOTS][QMC2_MAXSLOTS];
    std::memset(cnt, 0, sizeof cnt);
    bool any_big = false;
    for (const Factors &m : pl.mono) {
      if (m.size() < 2) continue;
      const int wgt = m.size() > 2 ? 64 : 1;
      if (m.size() > 2) any_big = true;
      std::pair<uint8_t, uint8_t> seen[128];  // each distinct pair counts once per monomial (m is sorted)
      int nseen = 0;
      for (size_t i = 0; i < m.size(); ++i)
        for (size_t k = i + 1; k < m.size(); ++k) {
          const std::pair<uint8_t, uint8_t> pr(m[i], m[k]);
          bool dup = false;
          for (int q = 0; q < nseen; ++q) dup = dup || seen[q] == pr;
          if (dup || nseen >= 128) continue;
          seen[nseen++] = pr;
          cnt[pr.first][pr.second] += wgt;
        }
    }
    int best = 0, ba = -1, bb = -1;
    for (int a = 0; a < pl.nslots; ++a)
      for (int b = a; b < pl.nslots; ++b)
        if (cnt[a][b] > best) {
          best = cnt[a][b];
          ba = a;
          bb = b;
        }
    if (stop_at_two && !any_big) break;   // every monomial is a product of at most two slots: enough for a record
    if (ba < 0) break;                    // every monomial has at most one factor
    if (best < 2) break;                  // a chunk-wide slot must serve at least two monomials
    if (pl.nslots >= max_slots) break;    // leftovers with more than two factors get sector-local products
    const int nw = pl.nslots++;
    pl.prog.push_back({(uint8_t)ba, (uint8_t)bb});
    for (Factors &m : pl.mono) {
      merge_pair(m, ba, bb, nw);
      std::sort(m.begin(), m.end());
    }
  }
  return true;
}

template <class T>
inline void put(std::vector<uint8_t> &img, const T &v) {
  const uint8_t *b = reinterpret_cast<const uint8_t *>(&v);
  img.insert(img.end(), b, b + sizeof(T));
}


}  // namespace qmcbpe
