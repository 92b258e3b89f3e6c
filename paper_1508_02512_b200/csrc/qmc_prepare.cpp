// qmc_prepare: Feynman graph -> Symanzik polynomials -> primary sectors -> iterated sub-sectors -> sector tables.
// Host only.  arXiv:1508.02512 Sec. 2.  "P:<n>" = PAPER.md line, "R:Cxx" = DESIGN.md reading.
//
// Written independently of oracle/ (no shared code): polynomials are flat sorted vectors with exponents packed
// 4 bits per variable; U comes from a deletion-contraction recursion, F from U of the graphs with two leg
// vertices identified; the decomposition runs on an explicit stack.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstring>

#include "../../include/qmc_feynman.h"
#include "qmc_tables.h"

namespace {

typedef uint64_t Key;  // exponent of variable j in bits [4j, 4j+4)
struct Term {
  Key k;
  double c;
};
typedef std::vector<Term> Poly;

inline int expo(Key k, int j) { return (int)((k >> (4 * j)) & 15u); }
inline Key unit(int j) { return (Key)1 << (4 * j); }

void canonical(Poly &p) {
  std::sort(p.begin(), p.end(), [](const Term &a, const Term &b) { return a.k < b.k; });
  size_t w = 0;
  for (size_t r = 0; r < p.size();) {
    Key k = p[r].k;
    double c = 0.0;
    while (r < p.size() && p[r].k == k) c += p[r++].c;
    if (c != 0.0) p[w++] = Term{k, c};
  }
  p.resize(w);
}

struct Edge {
  int u, v, idx;
};

// sum over spanning trees T of prod_{e not in T} x_e, by deletion / contraction of the last edge
void dual_kirchhoff(int nv, std::vector<Edge> edges, Key carry, Poly &out) {
  if (edges.empty()) {
    if (nv == 1) out.push_back(Term{carry, 1.0});
    return;
  }
  Edge e = edges.back();
  edges.pop_back();
  // e not in the tree: factor x_e, graph without e
  dual_kirchhoff(nv, edges, carry + unit(e.idx), out);
  if (e.u == e.v) return;  // a self-loop is never in a tree
  // e in the tree: contract (merge the larger label into the smaller, close the gap)
  int keep = std::min(e.u, e.v), drop = std::max(e.u, e.v);
  for (Edge &f : edges) {
    if (f.u == drop) f.u = keep;
    if (f.v == drop) f.v = keep;
    if (f.u > drop) --f.u;
    if (f.v > drop) --f.v;
  }
  dual_kirchhoff(nv - 1, edges, carry, out);
}

Poly spanning_poly(int nv, const std::vector<Edge> &edges) {
  Poly p;
  dual_kirchhoff(nv, edges, 0, p);
  canonical(p);
  return p;
}

struct Node {  // one (sub-)sector under construction
  int primary;
  Poly U, F;
  int alpha[QMC_MAXDIM], beta[QMC_MAXDIM];
  int depth;
  long long weight = 1;  // geometric strategy: |det V| of the cone's substitution (must be 1)
  bool final = false;    // geometric strategy: the substitution is complete, nothing left to split
};

bool constant_term(const Poly &p) { return !p.empty() && p.front().k == 0; }  // sorted: key 0 first

// rule R:C7 step 1: divide the common monomial out of Q and book its exponents
void pull_common(Poly &Q, int n, int a0, int a1, int *alpha, int *beta) {
  for (int j = 0; j < n; ++j) {
    int lo = 15;
    for (const Term &t : Q) lo = std::min(lo, expo(t.k, j));
    if (lo == 0 || Q.empty()) continue;
    for (Term &t : Q) t.k -= (Key)lo << (4 * j);
    alpha[j] += lo * a0;
    beta[j] += lo * a1;
  }
  canonical(Q);
}

// rule R:C7 step 3: smallest set of variables hitting every monomial; ties -> lexicographically smallest tuple.
// Sets are bit masks; tuple order: at the lowest differing bit, the set owning that bit is smaller.
unsigned smallest_hitting_set(const Poly &target, int n) {
  std::vector<unsigned> supp;
  for (const Term &t : target) {
    unsigned s = 0;
    for (int j = 0; j < n; ++j)
      if (expo(t.k, j)) s |= 1u << j;
    supp.push_back(s);
  }
  unsigned best = 0;
  int best_size = n + 1;
  for (unsigned S = 1; S < (1u << n); ++S) {
    int size = __builtin_popcount(S);
    if (size > best_size) continue;
    bool hits = true;
    for (unsigned s : supp)
      if (!(s & S)) {
        hits = false;
        break;
      }
    if (!hits) continue;
    bool better = size < best_size;
    if (!better) {
      unsigned diff = S ^ best;
      better = (S & (diff & (~diff + 1u))) != 0;
    }
    if (better) {
      best = S;
      best_size = size;
    }
  }
  return best;
}

// ---- geometric decomposition strategy (the strategy the paper says it uses, refs [25, 26]) ------
// Kaneko-Ueda: for a primary sector with polynomials U_l, F_l in t_1..t_n, the Newton polyhedron of P = U_l F_l,
//   Delta = conv{exponent vectors of P} + R^n_{>=0},
// has facets with inward primitive integer normals v >= 0.  The normal cones of its vertices tile the orthant x = -ln t >= 0.
// Every cone is cut into simplicial cones with generators v_1..v_n (rows of V); on such a cone the monomial substitution
//   t_j = prod_k y_k^(v_kj),  y in (0,1]^n,   d^n t prod_j t_j^(a_j) = |det V| prod_k y_k^(<v_k, a+1> - 1) d^n y
// turns every monomial t^e into y^(V e), and both polynomials into a monomial times a polynomial with a constant term
// (the minimum of <v_k, e> over a polynomial's monomials is attained at ONE monomial for all k: the vertex).  One step, no
// iteration, termination guaranteed.  A cone with |det V| > 1 would put a constant factor on its sector, which the tables
// do not carry: QMC_EUNSUPPORTED (none was met: on every graph tried all cones are unimodular, reading C31).
// Facets are found by testing the primitive vectors with entries 0..B: v is a facet normal iff the points where <v, e> is
// minimal, together with the free directions e_j (v_j = 0), span an affine set of dimension n-1.  Completeness is CHECKED, not
// assumed: the simplicial cones must tile the orthant, sum |det V| / prod_k <v_k, 1> = 1 (the integral of the Jacobian alone);
// if they do not, B is raised, and beyond B = 5 the call fails (QMC_EDEPTH) rather than return a partial decomposition.
typedef std::array<int, QMC_MAXDIM> IVec;
#ifndef QMC_GEO_ORDERS
#define QMC_GEO_ORDERS 24  // generator orders tried per non-simplicial cone
#endif
#define QMC_GEO_MAX_SIMPLICES 200u  // per vertex cone; beyond: QMC_EUNSUPPORTED (the double box needs at most a few per cone)

// work done by one geometric_cones call (exact determinants and ranks): beyond QMC_GEO_MAX_WORK the call gives up (QMC_EUNSUPPORTED)
// instead of running for minutes on polytopes with hundreds of vertices (a six-loop banana); the double box needs about 4e5
thread_local long long geo_work = 0;
#define QMC_GEO_MAX_WORK 20000000ll

long long det_exact(int n, std::vector<std::array<long long, QMC_MAXDIM>> M) {  // fraction-free (Bareiss) elimination
  geo_work += n * n;
  long long prev = 1, sign = 1;
  for (int k = 0; k < n; ++k) {
    int piv = -1;
    for (int i = k; i < n; ++i)
      if (M[i][k] != 0) {
        piv = i;
        break;
      }
    if (piv < 0) return 0;
    if (piv != k) {
      std::swap(M[piv], M[k]);
      sign = -sign;
    }
    for (int i = k + 1; i < n; ++i)
      for (int j = k + 1; j < n; ++j) M[i][j] = (M[i][j] * M[k][k] - M[i][k] * M[k][j]) / prev;
    prev = M[k][k];
  }
  return sign * M[n - 1][n - 1];
}

int rank_exact(int n, std::vector<std::array<long long, QMC_MAXDIM>> M) {  // integer row reduction, rows kept primitive
  geo_work += (long long)n * (long long)M.size();
  int rank = 0;
  for (int col = 0; col < n && rank < (int)M.size(); ++col) {
    int piv = -1;
    for (size_t i = rank; i < M.size(); ++i)
      if (M[i][col] != 0) {
        piv = (int)i;
        break;
      }
    if (piv < 0) continue;
    std::swap(M[piv], M[rank]);
    for (size_t i = rank + 1; i < M.size(); ++i) {
      if (M[i][col] == 0) continue;
      const long long a = M[rank][col], b = M[i][col];
      long long g = 0;
      for (int j = 0; j < n; ++j) {
        M[i][j] = M[i][j] * a - M[rank][j] * b;
        g = std::__gcd(g, M[i][j] < 0 ? -M[i][j] : M[i][j]);
      }
      if (g > 1)
        for (int j = 0; j < n; ++j) M[i][j] /= g;
    }
    ++rank;
  }
  return rank;
}

struct GeoCone {
  IVec v[QMC_MAXDIM];  // generators (rows)
  long long weight;    // |det V|
};

// simplicial cones of the normal fan of the Newton polyhedron of U * F (n variables); QMC_EDEPTH if they do not tile the orthant
int geometric_cones(const Poly &U, const Poly &F, int n, std::vector<GeoCone> &out) {
  std::vector<IVec> supp;  // exponent vectors of the product (Minkowski sum of the supports)
  {
    std::vector<Key> keys;
    for (const Term &a : U)
      for (const Term &b : F) keys.push_back(a.k + b.k);  // (4-bit fields: exponents of a product of two graph polynomials stay below 16)
    std::sort(keys.begin(), keys.end());
    keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
    for (Key k : keys) {
      IVec e{};
      for (int j = 0; j < n; ++j) e[j] = expo(k, j);
      supp.push_back(e);
    }
  }
  if (supp.empty()) return QMC_EINVAL;
  geo_work = 0;
  for (int B = 2; B <= 5; ++B) {
    // facets
    std::vector<IVec> normal;
    std::vector<int> level;
    IVec v{};
    long long ncand = 1;
    for (int j = 0; j < n; ++j) ncand *= B + 1;
    for (long long code = 1; code < ncand; ++code) {
      if (geo_work > QMC_GEO_MAX_WORK) return QMC_EUNSUPPORTED;
      long long c = code;
      int g = 0;
      for (int j = 0; j < n; ++j) {
        v[j] = (int)(c % (B + 1));
        c /= B + 1;
        g = std::__gcd(g, v[j]);
      }
      if (g != 1) continue;
      int m = 1 << 30;
      for (const IVec &e : supp) {
        int d = 0;
        for (int j = 0; j < n; ++j) d += v[j] * e[j];
        m = std::min(m, d);
      }
      std::vector<std::array<long long, QMC_MAXDIM>> rows;
      const IVec *first = nullptr;
      for (const IVec &e : supp) {
        int d = 0;
        for (int j = 0; j < n; ++j) d += v[j] * e[j];
        if (d != m) continue;
        if (!first) {
          first = &e;
          continue;
        }
        std::array<long long, QMC_MAXDIM> r{};
        for (int j = 0; j < n; ++j) r[j] = e[j] - (*first)[j];
        rows.push_back(r);
      }
      for (int j = 0; j < n; ++j)
        if (v[j] == 0) {
          std::array<long long, QMC_MAXDIM> r{};
          r[j] = 1;
          rows.push_back(r);
        }
      if ((int)rows.size() < n - 1 || rank_exact(n, rows) != n - 1) continue;
      normal.push_back(v);
      level.push_back(m);
    }
    // vertices and their normal cones
    std::vector<GeoCone> cones;
    bool ok = true;
    for (const IVec &e : supp) {
      if (geo_work > QMC_GEO_MAX_WORK) return QMC_EUNSUPPORTED;
      std::vector<int> gens;
      for (size_t f = 0; f < normal.size(); ++f) {
        int d = 0;
        for (int j = 0; j < n; ++j) d += normal[f][j] * e[j];
        if (d == level[f]) gens.push_back((int)f);
      }
      if ((int)gens.size() < n) continue;
      std::vector<std::array<long long, QMC_MAXDIM>> rows;
      for (int f : gens) {
        std::array<long long, QMC_MAXDIM> r{};
        for (int j = 0; j < n; ++j) r[j] = normal[f][j];
        rows.push_back(r);
      }
      if (rank_exact(n, rows) != n) continue;  // not a vertex
      // placing triangulation of cone{normal[g] : g in gens}: start from n independent generators, then add the others; a
      // new generator is joined to every boundary facet of the cone built so far that it sees from outside
      auto detof = [&](const std::vector<int> &idx) {
        std::vector<std::array<long long, QMC_MAXDIM>> M;
        for (int f : idx) {
          std::array<long long, QMC_MAXDIM> r{};
          for (int j = 0; j < n; ++j) r[j] = normal[f][j];
          M.push_back(r);
        }
        return det_exact(n, M);
      };
      // Placing triangulation for one order of the generators: start from the first n independent ones, then join every further
      // generator to the boundary facets of the cone built so far that it sees from outside.  Empty result: too many simplices.
      auto triangulate = [&](const std::vector<int> &order) {
        std::vector<int> start, rest;
        std::vector<std::array<long long, QMC_MAXDIM>> acc;
        for (int f : order) {
          std::array<long long, QMC_MAXDIM> r{};
          for (int j = 0; j < n; ++j) r[j] = normal[f][j];
          acc.push_back(r);
          if ((int)start.size() < n && rank_exact(n, acc) == (int)acc.size()) {
            start.push_back(f);
          } else {
            acc.pop_back();
            rest.push_back(f);
          }
        }
        std::vector<std::vector<int>> simp{start};
        for (int g : rest) {
          if (geo_work > QMC_GEO_MAX_WORK) return std::vector<std::vector<int>>();
          std::vector<std::vector<int>> add;
          for (size_t si = 0; si < simp.size(); ++si)
            for (int k = 0; k < n; ++k) {
              std::vector<int> face;
              for (int q = 0; q < n; ++q)
                if (q != k) face.push_back(simp[si][q]);
              std::vector<int> key = face;
              std::sort(key.begin(), key.end());
              geo_work += (long long)simp.size() * n;
              int shared = 0;  // a boundary facet belongs to exactly one simplex
              for (size_t sj = 0; sj < simp.size(); ++sj) {
                std::vector<int> o = simp[sj];
                std::sort(o.begin(), o.end());
                if (std::includes(o.begin(), o.end(), key.begin(), key.end())) ++shared;
              }
              if (shared != 1) continue;
              std::vector<int> with_u = face, with_g = face;
              with_u.push_back(simp[si][k]);
              with_g.push_back(g);
              const long long du = detof(with_u), dg = detof(with_g);
              if ((du > 0 && dg < 0) || (du < 0 && dg > 0)) add.push_back(with_g);
            }
          for (auto &sx : add) simp.push_back(sx);
          if (simp.size() > QMC_GEO_MAX_SIMPLICES) return std::vector<std::vector<int>>();  // (the boundary test is cubic in their number)
        }
        return simp;
      };
      // The triangulation depends on the order of the generators: a few deterministic orders are tried (as found, reversed,
      // rotations, fixed shuffles) and the one with the fewest simplices is kept -- fewer sectors, same integral.  If the first
      // order already needs too many simplices the others are not tried.
      std::vector<std::vector<int>> best;
      const int m = (int)gens.size(), ntry = m > n ? QMC_GEO_ORDERS : 1;
      for (int attempt = 0; attempt < ntry; ++attempt) {
        std::vector<int> order = gens;
        if (attempt == 1) std::reverse(order.begin(), order.end());
        if (attempt >= 2 && attempt < 2 + m) std::rotate(order.begin(), order.begin() + (attempt - 2) % m, order.end());
        if (attempt >= 2 + m) {
          unsigned long long st = 0x9E3779B97F4A7C15ull * (unsigned long long)(attempt + 1);
          for (int i = m - 1; i > 0; --i) {
            st = st * 6364136223846793005ull + 1442695040888963407ull;
            std::swap(order[i], order[(int)((st >> 33) % (unsigned long long)(i + 1))]);
          }
        }
        const std::vector<std::vector<int>> simp = triangulate(order);
        if (simp.empty()) {
          if (attempt == 0) break;
          continue;
        }
        if (best.empty() || simp.size() < best.size()) best = simp;
      }
      if (best.empty()) return QMC_EUNSUPPORTED;  // a cone that needs more than QMC_GEO_MAX_SIMPLICES simplices
      for (auto &s : best) {
        GeoCone c;
        for (int k = 0; k < n; ++k) c.v[k] = normal[s[k]];
        const long long d = detof(s);
        c.weight = d < 0 ? -d : d;
        if (c.weight == 0) ok = false;
        cones.push_back(c);
      }
    }
    // the cones must tile the orthant: sum |det V| / prod_k <v_k, 1> = 1
    double tile = 0.0;
    for (const GeoCone &c : cones) {
      double den = 1.0;
      for (int k = 0; k < n; ++k) {
        int sum = 0;
        for (int j = 0; j < n; ++j) sum += c.v[k][j];
        den *= sum;
      }
      tile += (double)c.weight / den;
    }
    if (ok && std::fabs(tile - 1.0) < 1e-9) {
      out = cones;
      return QMC_OK;
    }
  }
  return QMC_EDEPTH;
}

}  // namespace

// graph + kinematics -> T->sectors (appended), exponents, kmin (the most negative so far); no table images yet
static int qmc_build_sectors(const qmc_graph *g, const qmc_kinematics *kin, int eps_order, const qmc_options *opt,
                             qmc_tables *T) {
  if (!g || !kin || !kin->gram || !T) return QMC_EINVAL;
  const int V = g->n_vertices, P = g->n_edges, NL = g->n_legs;
  if (V < 1 || P < 2 || NL < 0 || P - 1 > QMC_MAXDIM) return QMC_EINVAL;
  if (eps_order < 0) return QMC_EINVAL;
  if (eps_order > QMC_KMAX_MAX) return QMC_EUNSUPPORTED;
  for (int e = 0; e < P; ++e) {
    if (g->edge_u[e] < 0 || g->edge_u[e] >= V || g->edge_v[e] < 0 || g->edge_v[e] >= V) return QMC_EINVAL;
    if (g->edge_nu && (g->edge_nu[e] < 1 || g->edge_nu[e] > 8)) return QMC_EINVAL;  // propagator powers: positive integers
  }
  for (int a = 0; a < NL; ++a)
    if (g->leg_vertex[a] < 0 || g->leg_vertex[a] >= V) return QMC_EINVAL;
  const int L = P - V + 1;
  if (L < 1) return QMC_EINVAL;

  // ---- Symanzik polynomials --------------------------------------------------------------
  std::vector<Edge> edges;
  for (int e = 0; e < P; ++e) edges.push_back(Edge{g->edge_u[e], g->edge_v[e], e});
  Poly U = spanning_poly(V, edges);
  if (U.empty()) return QMC_EINVAL;  // disconnected graph
  // F0 = - sum_{2-forests} (p_T1)^2 prod x = sum_{a<b} (p_a.p_b) * [2-forests separating v_a, v_b]  (momentum
  // conservation), and the bracket is the spanning polynomial of the graph with v_a and v_b identified.
  Poly F;
  double scale = 0.0;
  for (int i = 0; i < NL * NL; ++i) scale = std::max(scale, std::fabs(kin->gram[i]));
  for (int a = 0; a < NL; ++a)
    for (int b = a + 1; b < NL; ++b) {
      int va = g->leg_vertex[a], vb = g->leg_vertex[b];
      double dot = kin->gram[a * NL + b];
      if (va == vb || dot == 0.0) continue;
      int keep = std::min(va, vb), drop = std::max(va, vb);
      std::vector<Edge> merged = edges;
      for (Edge &f : merged) {
        if (f.u == drop) f.u = keep;
        if (f.v == drop) f.v = keep;
        if (f.u > drop) --f.u;
        if (f.v > drop) --f.v;
      }
      Poly phi = spanning_poly(V - 1, merged);
      for (const Term &t : phi) F.push_back(Term{t.k, dot * t.c});
    }
  canonical(F);
  {  // kinematic zeros must be exact (R:C24): drop rounding residues of the Gram matrix
    Poly kept;
    for (const Term &t : F)
      if (std::fabs(t.c) > 1e-12 * scale) kept.push_back(t);
    F.swap(kept);
  }
  for (int e = 0; e < P; ++e) {  // + U * sum_e m_e^2 x_e
    double m2 = g->edge_m2 ? g->edge_m2[e] : 0.0;
    if (m2 == 0.0) continue;
    for (const Term &t : U) F.push_back(Term{t.k + unit(e), m2 * t.c});
  }
  canonical(F);
  if (F.empty()) return QMC_EINVAL;  // scaleless integral

  // ---- exponents (Eq. 6, D = 4 - 2 eps): a_U = N_nu - (L+1) D/2, a_F = -(N_nu - L D/2), N_nu = sum_j nu_j; the integrand
  //      carries prod_j x_j^(nu_j - 1) (restored Eq. 2, R:C1).  nu_j = 1 everywhere: N_nu = P, the case the table-driven kernels
  //      are compiled for (their exponents are functions of n and L); any other powers run on the generic kernel --------------
  int Nnu = 0;
  for (int e = 0; e < P; ++e) Nnu += g->edge_nu ? g->edge_nu[e] : 1;
  if (Nnu != P) T->generic_only = true;  // (the points of a batch share the graph and its powers)
  T->n = P - 1;
  T->P = P;
  T->L = L;
  T->aU0 = Nnu - 2 * (L + 1);
  T->aU1 = L + 1;
  T->aF0 = -(Nnu - 2 * L);
  T->aF1 = -L;
  T->lambda = opt ? opt->lambda : 0.0;
  T->transform = opt ? opt->transform : 0;
  T->lattice = opt ? opt->lattice : 0;
  if (T->lambda < 0.0 || (T->transform < 0 || T->transform > 2) || (T->lattice != 0 && T->lattice != 1)) return QMC_EINVAL;
  const int pole = opt ? opt->pole_extraction : 0;
  if (pole != 0 && pole != 1) return QMC_EINVAL;
  if (pole == 1) {  // integration by parts (Eq. 13; R:C30): real path, generic kernel (its Taylor flavour)
    if (T->lambda > 0.0) return QMC_EUNSUPPORTED;
    T->ibp = T->has_taylor = T->generic_only = true;
  }
  const int max_depth = (opt && opt->max_depth > 0) ? opt->max_depth : 64;
  const int strategy = opt ? opt->strategy : 0;  // 0: iterated (rule R:C7), 1: geometric (Kaneko-Ueda)
  if (strategy != 0 && strategy != 1) return QMC_EINVAL;
  const int n = T->n;
  T->kmax = eps_order;

  // ---- primary sectors (Eqs. 3-6) and iterated decomposition (Eqs. 7-9), depth first ------------
  std::vector<Node> stack;
  for (int l = P - 1; l >= 0; --l) {  // pushed in reverse so that primary sector 0 is processed first
    Node nd;
    nd.primary = l;
    nd.depth = 0;
    std::memset(nd.alpha, 0, sizeof nd.alpha);
    std::memset(nd.beta, 0, sizeof nd.beta);
    if (g->edge_nu)  // x_j^(nu_j - 1) of the variables that stay (x_l = 1)
      for (int e = 0, j = 0; e < P; ++e)
        if (e != l) nd.alpha[j++] = g->edge_nu[e] - 1;
    for (int which = 0; which < 2; ++which) {
      const Poly &Q = which ? F : U;
      Poly &R = which ? nd.F : nd.U;
      for (const Term &t : Q) {  // x_l = 1, the others renamed t_1..t_{P-1} in increasing order (Eq. 4)
        Key lowmask = ((Key)1 << (4 * l)) - 1;
        Key k = (t.k & lowmask) | ((t.k >> (4 * (l + 1))) << (4 * l));
        R.push_back(Term{k, t.c});
      }
      canonical(R);
    }
    if (strategy == 0) {
      stack.push_back(nd);
      continue;
    }
    // geometric strategy: one monomial substitution per simplicial cone of the normal fan, pushed in reverse so that the
    // cones of a primary sector come out in the order geometric_cones found them
    std::vector<GeoCone> cones;
    const int rcg = geometric_cones(nd.U, nd.F, n, cones);
    if (rcg != QMC_OK) return rcg;
    for (size_t ci = cones.size(); ci-- > 0;) {
      const GeoCone &cn = cones[ci];
      Node ch;
      ch.primary = l;
      ch.depth = 1;
      ch.final = true;
      ch.weight = cn.weight;
      std::memset(ch.alpha, 0, sizeof ch.alpha);
      std::memset(ch.beta, 0, sizeof ch.beta);
      for (int k = 0; k < n; ++k) {  // y_k^(<v_k, alpha + 1> - 1 + eps <v_k, beta>)
        int a = -1, b = 0;
        for (int j = 0; j < n; ++j) {
          a += cn.v[k][j] * (nd.alpha[j] + 1);
          b += cn.v[k][j] * nd.beta[j];
        }
        ch.alpha[k] = a;
        ch.beta[k] = b;
      }
      for (int which = 0; which < 2; ++which) {
        const Poly &Q = which ? nd.F : nd.U;
        Poly &R = which ? ch.F : ch.U;
        std::vector<IVec> ex(Q.size());
        IVec lo;
        lo.fill(1 << 30);
        for (size_t q = 0; q < Q.size(); ++q)
          for (int k = 0; k < n; ++k) {
            int d = 0;
            for (int j = 0; j < n; ++j) d += cn.v[k][j] * expo(Q[q].k, j);
            ex[q][k] = d;
            lo[k] = std::min(lo[k], d);
          }
        const int a0 = which ? T->aF0 : T->aU0, a1 = which ? T->aF1 : T->aU1;
        for (int k = 0; k < n; ++k) {  // the common monomial y^lo goes to the exponents at once (the keys hold 4 bits per variable)
          ch.alpha[k] += lo[k] * a0;
          ch.beta[k] += lo[k] * a1;
        }
        for (size_t q = 0; q < Q.size(); ++q) {
          Key key = 0;
          for (int k = 0; k < n; ++k) {
            if (ex[q][k] - lo[k] > 15) return QMC_EUNSUPPORTED;
            key += (Key)(ex[q][k] - lo[k]) << (4 * k);
          }
          R.push_back(Term{key, Q[q].c});
        }
        canonical(R);
      }
      stack.push_back(ch);
    }
  }
  int smax = -T->kmin;  // (a batch appends the sectors of several kinematic points: kmin = the most negative of all)
  while (!stack.empty()) {
    Node nd = stack.back();
    stack.pop_back();
    pull_common(nd.U, n, T->aU0, T->aU1, nd.alpha, nd.beta);
    pull_common(nd.F, n, T->aF0, T->aF1, nd.alpha, nd.beta);
    const Poly *target = !constant_term(nd.U) ? &nd.U : (!constant_term(nd.F) ? &nd.F : nullptr);
    if (target && nd.final) return QMC_EDEPTH;  // (cannot happen when the cones tile the orthant: checked in geometric_cones)
    if (!target) {  // emit
      QmcSector s;
      s.primary = nd.primary;
      if (nd.weight != 1) return QMC_EUNSUPPORTED;  // a non-unimodular cone (|det V| > 1) would need a constant factor per sector: R:C31
      s.nsing = 0;
      s.ndeep = 0;
      std::memset(s.alpha, 0, sizeof s.alpha);
      std::memset(s.beta, 0, sizeof s.beta);
      for (int j = 0; j < n; ++j) {
        s.alpha[j] = nd.alpha[j];
        s.beta[j] = nd.beta[j];
        if (nd.alpha[j] <= -2) {  // needs the p >= 1 Taylor terms of Eq. 11 (R:C9, R:C28): real path, alpha >= -3, two per sector
          if (T->lambda > 0.0 || nd.alpha[j] < -QMC_MAXTAYLOR || nd.beta[j] == 0 || ++s.ndeep > 2) return QMC_EUNSUPPORTED;
          ++s.nsing;  // (a variable that can give a pole: counted with the singular ones)
        }
        if (nd.alpha[j] == -1) {
          if (nd.beta[j] == 0) return QMC_EUNSUPPORTED;
          ++s.nsing;
        }
        if (nd.alpha[j] > 127 || nd.beta[j] > 127 || nd.beta[j] < -127) return QMC_EUNSUPPORTED;
      }
      if (s.nsing > QMC_MAXSING) return QMC_EUNSUPPORTED;
      if (T->ibp) {  // Taylor coefficients around the point: orders 0 .. -alpha_b in every variable with alpha_b <= -1
        int njet = 1;
        for (int j = 0; j < n; ++j)
          if (nd.alpha[j] <= -1) njet *= 1 - nd.alpha[j];
        if (njet > QMC_IBP_JET) return QMC_EUNSUPPORTED;
      }
      if (s.ndeep) T->has_taylor = T->generic_only = true;  // only the generic kernel has Taylor-coefficient corners
      smax = std::max(smax, s.nsing);
      for (int which = 0; which < 2; ++which)
        for (const Term &t : (which ? nd.F : nd.U)) {
          QmcMono m;
          m.c = t.c;
          for (int j = 0; j < QMC_MAXDIM; ++j) m.e[j] = (uint8_t)(j < n ? expo(t.k, j) : 0);
          (which ? s.F : s.U).push_back(m);
        }
      if (s.U.size() > 255 || s.F.size() > 255) return QMC_EUNSUPPORTED;
      T->sectors.push_back(s);
      continue;
    }
    if (nd.depth >= max_depth) return QMC_EDEPTH;
    unsigned S = smallest_hitting_set(*target, n);
    if (!S) return QMC_EDEPTH;
    int size = __builtin_popcount(S);
    for (int k = n - 1; k >= 0; --k) {  // children in increasing k => push in decreasing k
      if (!(S >> k & 1u)) continue;
      Node ch;
      ch.primary = nd.primary;
      ch.depth = nd.depth + 1;
      std::memcpy(ch.alpha, nd.alpha, sizeof ch.alpha);
      std::memcpy(ch.beta, nd.beta, sizeof ch.beta);
      for (int j = 0; j < n; ++j)
        if ((S >> j & 1u) && j != k) {  // t_j -> t_k t_j
          ch.alpha[k] += nd.alpha[j];
          ch.beta[k] += nd.beta[j];
        }
      ch.alpha[k] += size - 1;  // Jacobian t_k^{|S|-1} (a monomial)
      for (int which = 0; which < 2; ++which) {
        const Poly &Q = which ? nd.F : nd.U;
        Poly &R = which ? ch.F : ch.U;
        R.reserve(Q.size());
        for (const Term &t : Q) {
          int add = 0;
          for (int j = 0; j < n; ++j)
            if ((S >> j & 1u) && j != k) add += expo(t.k, j);
          if (expo(t.k, k) + add > 15) return QMC_EUNSUPPORTED;
          R.push_back(Term{t.k + ((Key)add << (4 * k)), t.c});
        }
        canonical(R);
      }
      stack.push_back(ch);
    }
  }
  T->kmin = -smax;
  if (T->kmax - T->kmin + 1 > QMC_MAXK) return QMC_EUNSUPPORTED;
  return QMC_OK;
}

// T->sectors -> the generic table image and the tables of the table-driven kernels
static int qmc_finish_tables(qmc_tables *T, const qmc_options *opt) {
  const int n = T->n;
  // ---- device image -----------------------------------------------------------------------------
  T->image.clear();
  T->secoff.clear();
  for (QmcSector &s : T->sectors) {
    QmcSectorHdr h;
    std::memset(&h, 0, sizeof h);
    int pos = 0, inv[QMC_MAXDIM];
    for (int pass = 0; pass < 2; ++pass)
      for (int j = 0; j < n; ++j)
        if ((s.alpha[j] <= -1) == (pass == 0)) {  // the variables that can give a pole first
          h.perm[pos] = (uint8_t)j;
          inv[j] = pos;
          h.alpha[pos] = (int8_t)s.alpha[j];
          h.beta[pos] = (int8_t)s.beta[j];
          ++pos;
        }
    h.nsing = (uint8_t)s.nsing;
    if (s.ndeep) h.flags |= 2;  // a Taylor sector (sector_eval_taylor)
    auto group_of = [&](const QmcMono &m) {
      int gmask = 0;
      for (int b = 0; b < s.nsing; ++b)
        if (m.e[h.perm[b]]) gmask |= 1 << b;
      return gmask;
    };
    for (int which = 0; which < 2; ++which) {
      std::vector<QmcMono> &M = which ? s.F : s.U;
      std::stable_sort(M.begin(), M.end(), [&](const QmcMono &a, const QmcMono &b) { return group_of(a) < group_of(b); });
      for (const QmcMono &m : M) {
        uint8_t &cnt = (which ? h.cntF : h.cntU)[group_of(m)];
        ++cnt;
        for (int j = 0; j < n; ++j)
          if (m.e[j] >= 2) h.flags |= 1;
      }
    }
    h.nU = (uint8_t)s.U.size();
    h.nF = (uint8_t)s.F.size();
    T->secoff.push_back((uint32_t)T->image.size());
    const uint8_t *hb = reinterpret_cast<const uint8_t *>(&h);
    T->image.insert(T->image.end(), hb, hb + sizeof h);
    for (int which = 0; which < 2; ++which)
      for (const QmcMono &m : (which ? s.F : s.U)) {
        const uint8_t *cb = reinterpret_cast<const uint8_t *>(&m.c);
        T->image.insert(T->image.end(), cb, cb + 8);
      }
    for (int which = 0; which < 2; ++which)
      for (const QmcMono &m : (which ? s.F : s.U)) {
        uint32_t w = 0;
        for (int j = 0; j < n; ++j) w |= (uint32_t)m.e[j] << (4 * inv[j]);
        const uint8_t *wb = reinterpret_cast<const uint8_t *>(&w);
        T->image.insert(T->image.end(), wb, wb + 4);
      }
    while (T->image.size() % 16) T->image.push_back(0);
  }
  T->secoff.push_back((uint32_t)T->image.size());
  // table-driven kernels: real path (version 4) and complex path (version 5).  What a builder cannot represent falls back
  // to the generic kernel: on failure EVERYTHING the builder left behind is dropped, so that qmc_integrate sees no
  // half-built tables
  if (T->generic_only) {  // propagator powers other than 1: exponents the table-driven kernels are not compiled for
    T->sec_cost.assign(T->sectors.size(), 1.0);
    return QMC_OK;
  }
  if (qmc_build_tables4(T, opt ? opt->slot_budget : 0, opt ? opt->chunk_bytes : 0, opt ? opt->threads : 0, opt ? opt->dense_template : 0) != QMC_OK) {
    T->tab4.clear();
    T->secoff4.clear();
    T->prog4.clear();
    T->const4.clear();
    T->chunks.clear();
  }
  // complex path: the default slot budgets first; a graph whose sectors need more sector-local products than a launch has
  // room for (the paper's non-planar I_D at six variables) gets larger budgets before the generic kernel is the answer
  int rc3 = qmc_build_image3(T, opt ? opt->slot_budget_cplx_real : 0, opt ? opt->slot_budget_cplx : 0, opt ? opt->chunk_bytes : 0);
  if (rc3 != QMC_OK && !(opt && (opt->slot_budget_cplx_real > 0 || opt->slot_budget_cplx > 0))) {
    const int retry[3][2] = {{40, 0}, {48, 26}, {56, 32}};
    for (int q = 0; q < 3 && rc3 != QMC_OK; ++q) rc3 = qmc_build_image3(T, retry[q][0], retry[q][1], opt ? opt->chunk_bytes : 0);
  }
  if (rc3 != QMC_OK) {
    T->image3.clear();
    T->chunks3.clear();
    T->tab5.clear();
    T->secoff5.clear();
    T->prog5r.clear();
    T->prog5c.clear();
    T->chunk3_nslots_c.clear();
    T->chunk3_max_local_c.clear();
  }
  if (T->sec_cost.size() != T->sectors.size()) T->sec_cost.assign(T->sectors.size(), 1.0);
  return QMC_OK;
}

int qmc_build_tables(const qmc_graph *g, const qmc_kinematics *kin, int eps_order, const qmc_options *opt,
                     qmc_tables *T) {
  if (!T) return QMC_EINVAL;
  T->sectors.clear();
  T->kmin = 0;
  T->row_of_sector.clear();
  T->n_rows = 1;
  const int rc = qmc_build_sectors(g, kin, eps_order, opt, T);
  if (rc != QMC_OK) return rc;
  return qmc_finish_tables(T, opt);
}

// Kinematic points as a batch: ONE graph at n_points kinematic points.  The sectors of all points are
// concatenated (row_of_sector = point); the exponent structure of a point's tables does not depend on the kinematics unless a
// coefficient vanishes, so every point must decompose into the same number of sectors (else QMC_EINVAL).
int qmc_build_tables_batch(const qmc_graph *g, const qmc_kinematics *kins, int n_points, int eps_order, const qmc_options *opt,
                           qmc_tables *T) {
  if (!T || !kins || n_points < 1) return QMC_EINVAL;
  T->sectors.clear();
  T->kmin = 0;
  T->row_of_sector.clear();
  size_t per_point = 0;
  for (int p = 0; p < n_points; ++p) {
    const size_t before = T->sectors.size();
    const int rc = qmc_build_sectors(g, &kins[p], eps_order, opt, T);
    if (rc != QMC_OK) return rc;
    const size_t cnt = T->sectors.size() - before;
    if (p == 0) per_point = cnt;
    if (cnt != per_point || cnt == 0) return QMC_EINVAL;
    for (size_t i = 0; i < cnt; ++i) T->row_of_sector.push_back(p);
  }
  T->n_rows = n_points;
  return qmc_finish_tables(T, opt);
}
