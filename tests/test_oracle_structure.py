"""Pins for the oracle's host-side stages O1-O4, O9 -- nothing here needs a GPU.

Each test checks the oracle against something OTHER than itself: polynomials quoted in BASELINE.json /
SURVEY App. B.5, the Kirchhoff matrix-tree theorem, homogeneity, the tiling identity of a sector
decomposition, character sums of a rank-1 lattice, textbook integrals and numpy statistics.
"""
import itertools

import numpy as np
import pytest
import sympy

import qmc_inputs as qi
from oracle import Oracle, lattice, statistics


def poly_dict(coeff, expo):
    return {tuple(int(x) for x in e): float(c) for c, e in zip(coeff, expo)}


# ---------------------------------------------------------------- O1: graph polynomials
def test_bubble_polynomials_match_baseline_json():
    # BASELINE.json config 1: U = x1+x2, F = -p^2 x1 x2 + m^2 (x1+x2)^2 with p^2=-1, m^2=1
    o = Oracle.from_workload(qi.bubble())
    assert poly_dict(*o.graph_poly("U")) == {(1, 0): 1.0, (0, 1): 1.0}
    assert poly_dict(*o.graph_poly("F")) == {(2, 0): 1.0, (1, 1): 3.0, (0, 2): 1.0}
    assert (o.aU0, o.aU1, o.aF0, o.aF1) == (-2, 2, 0, -1)  # U^{-2+2eps} F^{-eps}, Eq. 6, D=4-2eps


def test_massive_box_F_matches_survey():
    # F = -5 x2x4 + 1.5 x1x3 - 0.52 x2x3 - 0.52 x3x4 + (sum x)^2
    o = Oracle.from_workload(qi.massive_box())
    x = sympy.symbols("x1:5")
    F = -5 * x[1] * x[3] + sympy.Rational(3, 2) * x[0] * x[2] - sympy.Rational(52, 100) * x[1] * x[2] \
        - sympy.Rational(52, 100) * x[2] * x[3] + sum(x) ** 2
    want = {tuple(int(e) for e in m): float(c) for m, c in sympy.Poly(sympy.expand(F), *x).terms()}
    got = poly_dict(*o.graph_poly("F"))
    assert set(got) == set(want)
    for k in want:
        assert got[k] == pytest.approx(want[k], abs=1e-14)
    assert o.n_terms_F == 10


def test_double_box_polynomials_match_survey_B5():
    wl = qi.double_box(s=-3.0, t=-1.0)
    o = Oracle.from_workload(wl)
    U = poly_dict(*o.graph_poly("U"))
    F = poly_dict(*o.graph_poly("F"))

    def mono(*idx):
        e = [0] * 7
        for i in idx:
            e[i - 1] += 1
        return tuple(e)
    wantU = [(1, 2), (1, 4), (1, 6), (1, 7), (2, 3), (2, 5), (2, 6), (3, 4), (3, 6), (3, 7), (4, 5), (4, 6), (5, 6),
             (5, 7), (6, 7)]
    assert U == {mono(*p): 1.0 for p in wantU}
    s_terms = [(1, 2, 3), (1, 2, 4), (1, 3, 4), (2, 3, 4), (1, 3, 6), (1, 3, 7), (1, 4, 6), (2, 3, 6), (2, 4, 5),
               (2, 4, 6)]
    wantF = {mono(*p): 3.0 for p in s_terms}
    wantF[mono(5, 6, 7)] = 1.0
    assert F == wantF


@pytest.mark.parametrize("wl", qi.CONFIGS() + [qi.triangle()], ids=lambda w: w.name)
def test_U_counts_spanning_trees_and_homogeneity(wl):
    o = Oracle.from_workload(wl)
    cU, eU = o.graph_poly("U")
    cF, eF = o.graph_poly("F")
    # Kirchhoff: number of spanning trees = any cofactor of the graph Laplacian
    lap = np.zeros((wl.n_vertices, wl.n_vertices))
    for u, v, _ in wl.edges:
        lap[u, u] += 1; lap[v, v] += 1; lap[u, v] -= 1; lap[v, u] -= 1
    ntrees = round(np.linalg.det(lap[1:, 1:]))
    assert cU.sum() == ntrees and np.all(cU == 1.0)
    L = wl.n_edges - wl.n_vertices + 1
    assert o.L == L
    assert np.all(eU.sum(axis=1) == L)        # U homogeneous of degree L
    assert np.all(eF.sum(axis=1) == L + 1)    # F homogeneous of degree L+1
    assert np.all(eU <= 1)                    # U is multilinear
    # exponents: a_U*L + a_F*(L+1) + P = 0 (needed for the delta-function integration, Eqs. 5-6)
    P = wl.n_edges
    assert o.aU0 * L + o.aF0 * (L + 1) + P == 0 and o.aU1 * L + o.aF1 * (L + 1) == 0


def test_euclidean_F_positive():
    for wl in (qi.bubble(), qi.massless_box(), qi.double_box(), qi.triangle()):
        o = Oracle.from_workload(wl)
        cF, _ = o.graph_poly("F")
        assert np.all(cF > 0)


def test_invalid_graph_rejected():
    wl = qi.massless_box()
    wl.edges = [(0, 1, 0.0), (0, 1, 0.0), (2, 3, 0.0), (2, 3, 0.0)]  # two disconnected bubbles: no spanning tree
    with pytest.raises(ValueError):
        Oracle.from_workload(wl)


# ---------------------------------------------------------------- O2/O3: decomposition
EXPECT = {  # SURVEY App. B.1 (rule A.3): sectors, per-primary counts, n_sing histogram
    "cfg1_bubble": (2, [1, 1], {0: 2}),
    "cfg2_massless_box": (12, [3, 3, 3, 3], {1: 4, 2: 8}),
    "cfg3_massive_box": (4, [1, 1, 1, 1], {0: 4}),
    "cfg4_double_box": (293, [28, 28, 28, 32, 75, 34, 68], {1: 26, 2: 72, 3: 102, 4: 93}),
    "cfg5_nonplanar_vertex": (36, [4, 4, 4, 6, 12, 6], {0: 24, 1: 12}),
    "triangle": (3, [1, 1, 1], {1: 2, 2: 1}),
}


@pytest.mark.parametrize("wl", qi.CONFIGS() + [qi.triangle()], ids=lambda w: w.name)
def test_decomposition_invariants(wl):
    o = Oracle.from_workload(wl)
    assert o.status == 0
    secs = [o.sector(s) for s in range(o.n_sectors)]
    nsec, per_primary, hist = EXPECT[wl.name]
    assert o.n_sectors == nsec
    assert [sum(1 for s in secs if s["primary"] == p) for p in range(wl.n_edges)] == per_primary
    ns = [s["n_sing"] for s in secs]
    assert {k: ns.count(k) for k in set(ns)} == hist
    assert o.k_min == -max(ns)
    for s in secs:
        # Eqs. 7-8: both polynomials are const + H with H(0) = 0, constants non-zero
        for name in ("U", "F"):
            c, e = s[name]
            zero = [i for i in range(len(c)) if not e[i].any()]
            assert len(zero) == 1 and c[zero[0]] != 0.0
        assert np.all(s["alpha"] >= -1)
        assert np.all(s["beta"][s["alpha"] == -1] != 0)
    # tiling identity: the sub-sectors of one primary sector tile the unit cube, so the integrals of
    # their Jacobian monomials add up to 1: sum_sub prod_j 1/(c_j + 1) = 1
    for p in range(wl.n_edges):
        tot = sum(np.prod(1.0 / (s["jac"] + 1.0)) for s in secs if s["primary"] == p)
        assert tot == pytest.approx(1.0, abs=1e-12)


# ---------------------------------------------------------------- O4: lattice, shift, transform
def test_lattice_is_exact_for_characters():
    # an unshifted rank-1 rule integrates exp(2 pi i h.x) to exactly 0 unless h.z = 0 mod N (textbook)
    N, dim = 10007, 3
    z = qi.korobov_vector(N, dim, 1227)
    y, _, _, _ = lattice(N, z, 0, N, np.zeros(dim))
    assert y.min() >= 0.0 and y.max() < 1.0
    rng = np.random.default_rng(5)
    hs = [rng.integers(-6, 7, size=dim) for _ in range(12)]
    dual = np.array([int(z[1]), -1, 0])      # h.z = z1*a^0... = a - a = 0 mod N
    hs += [dual, 2 * dual, np.array([N, 0, 0])]
    for h in hs:
        val = np.exp(2j * np.pi * (y @ h)).mean()
        if int(np.dot(h.astype(object), z.astype(object))) % N == 0:
            assert abs(val - 1) < 1e-9
        else:
            assert abs(val) < 1e-9


def test_lattice_points_are_i_z_over_N_exactly():
    N, dim = 99991, 5
    z = qi.good_vector(N, dim)
    sh = qi.splitmix64_shifts(3, 1, dim)[0]
    i0 = 77777
    y, t, w, inside = lattice(N, z, i0, 50, sh)
    for c in range(50):
        for j in range(dim):
            r = ((i0 + c) * int(z[j])) % N
            v = r / N + sh[j]
            v = v - 1.0 if v >= 1.0 else v
            assert y[c, j] == v
    assert inside.all()


@pytest.mark.parametrize("dim", [1, 2, 3])
def test_periodising_transform_integrates_monomials(dim):
    # Eq. 21: int prod x_j d^s x = 2^-s ; int prod x_j^2 = 3^-s
    N = 32749
    z = qi.good_vector(N, dim)
    sh = qi.splitmix64_shifts(11, 1, dim)[0]
    y, t, w, _ = lattice(N, z, 0, N, sh)
    assert np.mean(w * np.prod(t, axis=1)) == pytest.approx(2.0 ** -dim, rel=2e-6)
    assert np.mean(w * np.prod(t * t, axis=1)) == pytest.approx(3.0 ** -dim, rel=2e-6)
    assert np.mean(w) == pytest.approx(1.0, rel=2e-6)
    # g vanishes on the boundary: weight -> 0 as y -> 0
    y0, t0, w0, ins = lattice(N, z, 0, 1, np.zeros(dim))
    assert w0[0] == 0.0 and ins[0] == 0


def test_tent_transform():
    N = 10007
    z = qi.good_vector(N, 2)
    y, t, w, _ = lattice(N, z, 0, N, np.array([0.3, 0.7]), transform=1)
    assert np.all(w == 1.0)
    assert np.mean(np.prod(t, axis=1)) == pytest.approx(0.25, rel=1e-5)


@pytest.mark.parametrize("dim", [1, 2, 3])
def test_second_order_periodising_transform(dim):
    # transform = 2 (R:C20; the r = 2 member of Eq. 21's family): x = 10y^3 - 15y^4 + 6y^5, weight 30 y^2 (1-y)^2.
    # Pins: x(0) = 0, x(1/2) = 1/2, x -> 1; dx/dy = weight (central differences on y itself); the same monomial
    # integrals as Eq. 21; symmetry x(1-y) = 1 - x(y)
    N = 32749
    z = qi.good_vector(N, dim)
    sh = qi.splitmix64_shifts(11, 1, dim)[0]
    y, t, w, _ = lattice(N, z, 0, N, sh, transform=2)
    assert np.mean(w * np.prod(t, axis=1)) == pytest.approx(2.0 ** -dim, rel=1e-8)
    assert np.mean(w * np.prod(t * t, axis=1)) == pytest.approx(3.0 ** -dim, rel=1e-8)
    assert np.mean(w) == pytest.approx(1.0, rel=1e-8)
    if dim == 1:
        order = np.argsort(y[:, 0])
        ys, ts, ws = y[order, 0], t[order, 0], w[order]
        assert np.all(np.diff(ts) > 0) and ts[0] > 0 and ts[-1] < 1
        k = np.arange(1, N - 1)
        slope = (ts[k + 1] - ts[k - 1]) / (ys[k + 1] - ys[k - 1])
        assert np.allclose(slope, ws[k], rtol=0, atol=5e-8)
        x = lambda v: 10 * v ** 3 - 15 * v ** 4 + 6 * v ** 5          # the polynomial in its expanded form
        assert np.allclose(ts, x(ys), rtol=1e-13, atol=1e-300)
        assert np.allclose(x(1.0 - ys), 1.0 - ts, rtol=0, atol=3e-14)   # expanded form: terms of size 10 cancel
        one = lattice(3, [1], 0, 3, np.array([0.5]), transform=2)       # y = 1/2, 5/6, 1/6
        assert one[1][0, 0] == 0.5 and one[2][0] == pytest.approx(30.0 / 16.0, rel=1e-15)
    y0, t0, w0, ins = lattice(N, z, 0, 1, np.zeros(dim), transform=2)
    assert w0[0] == 0.0 and ins[0] == 0


def test_primes_and_vectors_are_valid():
    for nominal, p in qi.PRIMES.items():
        assert sympy.isprime(p) and sympy.prevprime(nominal + 1) == p
    for k, p in zip(range(14, 28), qi.primes_below_pow2()):
        assert sympy.prevprime(2 ** k) == p
    for (N, dim), a in qi.GOOD_KOROBOV.items():
        z = qi.korobov_vector(N, dim, a)
        assert all(np.gcd(int(v), N) == 1 for v in z)


def test_splitmix64_reference_values():
    # first outputs of SplitMix64 with seed 1234567 (published test vector of the generator)
    sh = qi.splitmix64_shifts(1234567, 1, 2)[0]
    assert sh[0] == (6457827717110365317 >> 11) / 2.0 ** 53
    assert sh[1] == (3203168211198807973 >> 11) / 2.0 ** 53


# ---------------------------------------------------------------- O9: statistics
def test_statistics_match_numpy():
    rng = np.random.default_rng(1)
    T = rng.normal(size=(5, 16)) + 1j * rng.normal(size=(5, 16))
    mean, err = statistics(T)
    assert np.allclose(mean, T.mean(axis=1), rtol=0, atol=1e-15)
    assert np.allclose(err.real, T.real.std(axis=1, ddof=1) / 4.0, rtol=1e-13)
    assert np.allclose(err.imag, T.imag.std(axis=1, ddof=1) / 4.0, rtol=1e-13)


def test_embedded_lattice_identity_on_the_oracle():
    """SURVEY 8(f) f4 / reading C26: with odd generating-vector components the even indices of the N = 2^(k+1) lattice are the
    points of the N = 2^k lattice ({2i z / 2N} = {i z / N}, Eq. 17), so per shift
    Q(2N) = Q(N) / 2 + (1/2N) sum over odd i -- checked on the oracle's own sums for a sector-decomposed integrand."""
    from oracle import Oracle
    wl = qi.massless_box()
    o = Oracle.from_workload(wl)
    z = np.array([1, 1237, 1237 * 1237 % 4096], dtype=np.uint64)          # odd components
    sh = qi.splitmix64_shifts(5, 3, 3)
    N = 2048
    S1, A1, _ = o.integrate(N, z % N, sh)
    S2, A2, _ = o.integrate(2 * N, z % (2 * N), sh)
    Sodd, Aodd, _ = o.integrate(2 * N, z % (2 * N), sh, index_range=(1, 2, N))
    assert np.all(np.abs(0.5 * S1 + Sodd - S2) <= 1e-13 * np.maximum(np.abs(S2), A2))
    # and the points themselves: lattice index 2i at 2N = lattice index i at N
    import oracle as orc
    y_even = orc.lattice(2 * N, z % (2 * N), 0, 2 * N, sh[0])[0]
    y_half = orc.lattice(N, z % N, 0, N, sh[0])[0]
    assert np.array_equal(np.asarray(y_even)[::2], np.asarray(y_half))
