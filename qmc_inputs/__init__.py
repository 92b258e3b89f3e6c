"""Seeded, synthetic INPUT generators shared by the oracle tests and the CUDA product tests.

This module holds none of the method's arithmetic: it only describes *what is integrated*
(graphs, masses, Gram matrices of external momenta: the five BASELINE.json configs plus a few
extra pins) and *which numbers are fed in* (lattice sizes, explicit generating vectors of Korobov
form, shift vectors from a SplitMix64 stream).  Neither oracle/ nor paper_1508_02512_b200/ is
imported here.

The workloads stand in for the paper's four analytically defined integrals (arXiv:1508.02512
Eqs. 22-27); the paper measures on no dataset.  Edge lists follow SURVEY.md 8(d).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

__all__ = [
    "Workload", "CONFIGS", "bubble", "massless_box", "massive_box", "gghh_box_scan", "paper_IC", "paper_ID", "double_box", "nonplanar_vertex",
    "triangle", "four_point_gram", "splitmix64_shifts", "korobov_vector", "good_vector", "GOOD_KOROBOV", "PRIMES",
    "primes_below_pow2",
]


@dataclass
class Workload:
    name: str
    n_vertices: int
    edges: List[Tuple[int, int, float]]          # (u, v, m^2); Feynman parameter x_k <-> edges[k-1]
    leg_vertex: List[int]                        # vertex of each (incoming) external leg
    gram: np.ndarray                             # [n_legs, n_legs] p_i . p_j
    lam: float = 0.0                             # contour deformation lambda (0 = Euclidean / real path)
    eps_order: int = 0                           # highest order of J(eps) wanted
    N_list: Sequence[int] = ()                   # lattice sizes (primes)
    m: int = 16                                  # number of random shifts
    seed: int = 0
    meta: dict = field(default_factory=dict)
    nu: Optional[Sequence[int]] = None           # propagator powers nu_k; None = all 1, as in every config

    @property
    def n_edges(self) -> int:
        return len(self.edges)

    @property
    def dim(self) -> int:
        return len(self.edges) - 1

    def arrays(self):
        eu = np.array([e[0] for e in self.edges], dtype=np.int32)
        ev = np.array([e[1] for e in self.edges], dtype=np.int32)
        m2 = np.array([e[2] for e in self.edges], dtype=np.float64)
        lv = np.array(self.leg_vertex, dtype=np.int32)
        return eu, ev, m2, lv, np.ascontiguousarray(self.gram, dtype=np.float64)


def four_point_gram(p2: Sequence[float], s: float, t: float) -> np.ndarray:
    """Gram matrix of four incoming momenta with p_i^2 = p2[i], s=(p1+p2)^2, t=(p2+p3)^2."""
    m1, m2, m3, m4 = p2
    u = m1 + m2 + m3 + m4 - s - t
    g = np.zeros((4, 4))
    for i, v in enumerate(p2):
        g[i, i] = v
    def put(i, j, inv):
        g[i, j] = g[j, i] = 0.5 * (inv - p2[i] - p2[j])
    put(0, 1, s); put(2, 3, s)
    put(1, 2, t); put(0, 3, t)
    put(0, 2, u); put(1, 3, u)
    return g


def bubble(p2: float = -1.0, m2a: float = 1.0, m2b: float = 1.0) -> Workload:
    """Config 1: one-loop bubble.  Gamma(eps) prefactor => J is needed through eps^1."""
    g = np.array([[p2, -p2], [-p2, p2]])
    return Workload("cfg1_bubble", 2, [(0, 1, m2a), (0, 1, m2b)], [0, 1], g, 0.0, 1, (10007,), 10, 1)


def triangle(s: float = -2.0) -> Workload:
    """Extra pin: one-loop massless triangle p1^2=p2^2=0, p3^2=s (Dirichlet closed form)."""
    g = np.array([[0.0, s / 2, -s / 2], [s / 2, 0.0, -s / 2], [-s / 2, -s / 2, s]])
    return Workload("triangle", 3, [(0, 1, 0.0), (1, 2, 0.0), (2, 0, 0.0)], [0, 1, 2], g, 0.0, 1, (99991,), 8, 3)


def massless_box(s: float = -3.0, t: float = -2.0) -> Workload:
    """Config 2: one-loop massless box; leg p_{i+1} at vertex i."""
    return Workload("cfg2_massless_box", 4, [(0, 1, 0.0), (1, 2, 0.0), (2, 3, 0.0), (3, 0, 0.0)], [0, 1, 2, 3],
                    four_point_gram([0, 0, 0, 0], s, t), 0.0, 0, (99991, 999983, 9999991), 16, 7)


def massive_box(s: float = 5.0, t: float = -1.5, m2: float = 1.0, mh2: float = 0.52, lam: float = 0.5) -> Workload:
    """Config 3: one-loop box, four equal internal masses, p3^2=p4^2=mh2, physical region for s > 4 m2."""
    return Workload("cfg3_massive_box", 4, [(0, 1, m2), (1, 2, m2), (2, 3, m2), (3, 0, m2)], [0, 1, 2, 3],
                    four_point_gram([0, 0, mh2, mh2], s, t), lam, 0, (99991, 999983, 9999991), 16, 11)


def gghh_box_scan(n_points: int = 1000, s_min: float = 70000.0, s_max: float = 500000.0, t: float = -6000.0,
                  mt: float = 172.0, mh: float = 125.0, lam: float = 0.5):
    """The paper's kinematic scan of the one-loop box I_A of gg -> HH (Eq. 22: 1000 values of s in
    [70000, 500000] at t = -6000, M_t = 172, M_H = 125; threshold at s = 4 M_t^2 = 118336), in units of M_t^2: the graph of
    config 3 at other kinematics.  Yields (s, Workload)."""
    mt2 = mt * mt
    for i in range(n_points):
        s = s_min + (s_max - s_min) * i / max(n_points - 1, 1)
        wl = massive_box(s=s / mt2, t=t / mt2, m2=1.0, mh2=mh * mh / mt2, lam=lam)
        wl.name = "gghh_box_scan"
        yield s, wl


def _gghh_two_loop(name: str, edges, lam: float, s: float, t: float, mt: float, mh: float) -> Workload:
    mt2 = mt * mt
    g = four_point_gram([0.0, 0.0, mh * mh / mt2, mh * mh / mt2], s / mt2, t / mt2)
    wl = Workload(name, 6, edges, [0, 1, 4, 5], g, lam, 0, primes_below_pow2(14, 27), 20, 5)
    wl.meta["s_over_mt2"] = s / mt2
    return wl


def paper_IC(lam: float = 0.3, s: float = 160000.0, t: float = -6000.0, mt: float = 172.0, mh: float = 125.0) -> Workload:
    """The paper's planar two-loop master integral I_C of gg -> HH (Eq. 25; Table 2), in
    units of M_t^2.  Propagators of Eq. 25 in order: k1, k1-p1, k1+p2 (massless), k1-k2-p1, k2, k1+p2-k2-p3, k1-k2+p2
    (mass M_t).  With k2' = k1 - k2 the rung is line 5; vertices: 0 (p1; lines 1, 2), 1 (p2; lines 1, 3),
    2 (lines 2, 4, 5), 3 (lines 3, 5, 7), 4 (p3 leaves; lines 6, 7), 5 (p4 leaves; lines 4, 6)."""
    edges = [(0, 1, 0.0), (0, 2, 0.0), (1, 3, 0.0), (2, 5, 1.0), (2, 3, 1.0), (4, 5, 1.0), (3, 4, 1.0)]
    return _gghh_two_loop("paper_IC_planar_double_box", edges, lam, s, t, mt, mh)


def paper_ID(lam: float = 0.3, s: float = 160000.0, t: float = -6000.0, mt: float = 172.0, mh: float = 125.0) -> Workload:
    """The paper's non-planar two-loop master integral I_D (Eq. 27; Table 3), in units of
    M_t^2.  Propagators of Eq. 27 in order: k1, k1+p1, k1-p2 (massless), k1+p1-k2, k2, k2-p4, k1+p1-k2-p3 (mass M_t).
    Vertices: 0 (p1; lines 1, 2), 1 (p2; lines 1, 3), 2 (lines 2, 4, 5), 3 (lines 3, 6, 7), 4 (p3 leaves; lines 4, 7),
    5 (p4 leaves; lines 5, 6): lines 5 and 6 carry both loop momenta -- non-planar."""
    edges = [(0, 1, 0.0), (0, 2, 0.0), (1, 3, 0.0), (2, 4, 1.0), (2, 5, 1.0), (5, 3, 1.0), (4, 3, 1.0)]
    return _gghh_two_loop("paper_ID_nonplanar_double_box", edges, lam, s, t, mt, mh)


def double_box(s: float = -3.0, t: float = -1.0, p2: Sequence[float] = (0, 0, 0, 0), eps_order: int = 0) -> Workload:
    """Config 4: two-loop planar double box (topology and leg placement of the paper's Eq. 23).

    Vertices a1,a2,a3,b1,b2,b3 = 0..5; rails e1=(0,1) e2=(1,2) e3=(3,4) e4=(4,5); rungs e5=(0,3) e6=(1,4)
    e7=(2,5); legs p1@0, p2@3, p3@5, p4@2."""
    edges = [(0, 1, 0.0), (1, 2, 0.0), (3, 4, 0.0), (4, 5, 0.0), (0, 3, 0.0), (1, 4, 0.0), (2, 5, 0.0)]
    return Workload("cfg4_double_box", 6, edges, [0, 3, 5, 2], four_point_gram(list(p2), s, t), 0.0, eps_order,
                    (999983, 9999991, 99999989), 20, 13)


def nonplanar_vertex(s: float = 5.0, m2: float = 1.0, lam: float = 0.3) -> Workload:
    """Config 5 (reading C22): two-loop non-planar vertex, vertices A,B,C,D,E = 0..4."""
    A, B, C, D, E = range(5)
    edges = [(C, D, m2), (C, E, m2), (D, A, m2), (D, B, 0.0), (E, A, 0.0), (E, B, 0.0)]
    g = np.array([[0.0, s / 2, -s / 2], [s / 2, 0.0, -s / 2], [-s / 2, -s / 2, s]])
    return Workload("cfg5_nonplanar_vertex", 5, edges, [A, B, C], g, lam, 0,
                    primes_below_pow2(14, 27), 20, 17)


# largest primes <= the nominal lattice sizes of the configs (checked in tests with sympy)
PRIMES = {10**4 + 7: 10007, 10**5: 99991, 10**6: 999983, 10**7: 9999991, 10**8: 99999989}

_POW2_PRIMES = {14: 16381, 15: 32749, 16: 65521, 17: 131071, 18: 262139, 19: 524287, 20: 1048573, 21: 2097143,
                22: 4194301, 23: 8388593, 24: 16777213, 25: 33554393, 26: 67108859, 27: 134217689}


def primes_below_pow2(k0: int = 14, k1: int = 27) -> Tuple[int, ...]:
    """Largest prime below 2^k for k0 <= k <= k1 (config 5's increasing lattice sizes)."""
    return tuple(_POW2_PRIMES[k] for k in range(k0, k1 + 1))


def CONFIGS() -> List[Workload]:
    """The five BASELINE.json configs, in order."""
    return [bubble(), massless_box(), massive_box(), double_box(), nonplanar_vertex()]


_MASK = (1 << 64) - 1


def splitmix64_shifts(seed: int, m: int, dim: int) -> np.ndarray:
    """m shift vectors in [0,1)^dim: SplitMix64 stream keyed by `seed`, shift-major / component-minor,
    Delta = (u64 >> 11) * 2^-53.  Pure input generation (PAPER.md:155 only asks for
    'uniform distribution in [0,1]^s')."""
    state = seed & _MASK
    out = np.empty((m, dim), dtype=np.float64)
    for k in range(m):
        for j in range(dim):
            state = (state + 0x9E3779B97F4A7C15) & _MASK
            x = state
            x = ((x ^ (x >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
            x = ((x ^ (x >> 27)) * 0x94D049BB133111EB) & _MASK
            x = x ^ (x >> 31)
            out[k, j] = (x >> 11) * (1.0 / 9007199254740992.0)
    return out


# Korobov multipliers with a small P_2 figure of merit, found offline by a random search (inputs only:
# any z with components coprime to N is a valid rule).  Key: (N, dim).
GOOD_KOROBOV = {
    (10007, 2): 6978, (10007, 3): 1227, (10007, 5): 1504, (10007, 6): 5373,
    (16381, 2): 2602, (16381, 3): 11560, (16381, 5): 5639, (16381, 6): 8801,
    (32749, 2): 20943, (32749, 3): 14857, (32749, 5): 25497, (32749, 6): 32330,
    (65521, 2): 9088, (65521, 3): 7548, (65521, 5): 46289, (65521, 6): 39389,
    (99991, 2): 21632, (99991, 3): 68700, (99991, 5): 73146, (99991, 6): 2057,
    (131071, 2): 100375, (131071, 3): 97565, (131071, 5): 61727, (131071, 6): 60941,
    (262139, 2): 103199, (262139, 3): 144590, (262139, 5): 217322, (262139, 6): 113603,
    (999983, 3): 848431, (999983, 5): 88126, (999983, 6): 803810,
}


def good_vector(N: int, dim: int) -> np.ndarray:
    """Explicit generating vector for tests: tabulated Korobov multiplier (1 for dim 1)."""
    return korobov_vector(N, dim, 1 if dim == 1 else GOOD_KOROBOV[(N, dim)])


def korobov_vector(N: int, dim: int, a: int) -> np.ndarray:
    """z = (1, a, a^2, ...) mod N -- an explicit generating vector to feed to both sides."""
    z = np.empty(dim, dtype=np.uint64)
    v = 1
    for j in range(dim):
        z[j] = v
        v = (v * a) % N
    return z
