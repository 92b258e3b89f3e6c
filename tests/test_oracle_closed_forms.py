"""Pins for the oracle's evaluator (O5-O8) and the whole chain: closed forms, brute-force quadrature,
invariants.  CPU only.  Closed forms are evaluated here with mpmath, never by the oracle.

Level-2 acceptance: |QMC - exact| <= 3 sigma (+ a rounding floor) per order.
"""
import mpmath as mp
import numpy as np
import pytest

import qmc_inputs as qi
from oracle import Oracle

mp.mp.dps = 40


def laurent(f, kmin, kmax):
    """Laurent coefficients eps^kmin..eps^kmax of f(eps) having a pole of order -kmin at 0."""
    c = mp.taylor(lambda e: e ** (-kmin) * f(e), 0, kmax - kmin, singular=True)
    return [complex(x) if abs(mp.im(x)) > 0 else float(mp.re(x)) for x in c]


def run(wl, N, m=None, **kw):
    o = Oracle.from_workload(wl, **kw)
    z = qi.good_vector(N, o.dim)
    sh = qi.splitmix64_shifts(wl.seed, m or wl.m, o.dim)
    S, A, cnt = o.integrate(N, z, sh)
    coeff, err = o.totals(S)
    return o, S, coeff, err, cnt


def assert_within(coeff, err, exact, nsig=3.0, floor=1e-13):
    for k, ex in enumerate(exact):
        tol = nsig * err[k].real + floor * max(1.0, abs(ex))
        assert abs(coeff[k].real - ex) <= tol, (k, coeff[k], err[k], ex)
        assert abs(coeff[k].imag) <= nsig * err[k].imag + floor


# ------------------------------------------------------------------------- config 1: bubble
def bubble_exact(kmax=2):
    # on the simplex U = 1:  J(eps) = int_0^1 dx [x(1-x) + 1]^(-eps)   (p^2 = -1, m^2 = 1; F from BASELINE.json)
    return [float(mp.quad(lambda x: (-mp.log(x * (1 - x) + 1)) ** k / mp.factorial(k), [0, 1])) for k in range(kmax + 1)]


def test_bubble_closed_form_config1():
    ex = bubble_exact(2)
    # BASELINE.json: finite part 2 - sqrt(1+4 m^2/|p^2|) ln((sqrt5+1)/(sqrt5-1)) = J_1 (Gamma(eps) J)
    r5 = mp.sqrt(5)
    assert ex[1] == pytest.approx(float(2 - r5 * mp.log((r5 + 1) / (r5 - 1))), abs=1e-15)
    assert ex[1] == pytest.approx(-0.152044704820020194, abs=1e-15)
    wl = qi.bubble()
    o, S, coeff, err, cnt = run(wl, 10007, eps_order=2)
    assert o.K == 3 and not cnt.any()
    assert_within(coeff, err, ex)
    assert np.all(err.real < 1e-8)
    # equal masses: each primary sector gives exactly half (sector-sum symmetry under swapping equal lines)
    sec = S.mean(axis=2)
    assert np.allclose(sec[0], sec[1], rtol=0, atol=1e-15)


def test_bubble_sector_integrand_and_quadrature():
    # sector integrand of primary sector 1: (1+t)^-2 [2 ln(1+t) - ln((1+t)^2 + t)]^k / k!
    o = Oracle.from_workload(qi.bubble(), eps_order=2)
    for t in (0.013, 0.5, 0.97):
        got = o.sector_integrand(0, [t])
        L = 2 * mp.log(1 + t) - mp.log((1 + t) ** 2 + t)
        for k in range(3):
            assert got[k].real == pytest.approx(float((1 + t) ** -2 * L ** k / mp.factorial(k)), rel=1e-13)
    for k in range(3):
        q = mp.quad(lambda t: (1 + t) ** -2 * (2 * mp.log(1 + t) - mp.log((1 + t) ** 2 + t)) ** k / mp.factorial(k), [0, 1])
        assert float(q) == pytest.approx(bubble_exact(2)[k] / 2, abs=1e-14)


def test_bubble_unequal_masses_changes_sectors_but_total_matches_quadrature():
    wl = qi.bubble(p2=-1.0, m2a=1.0, m2b=2.5)
    ex = [float(mp.quad(lambda x: (-mp.log(x * (1 - x) + x * 1.0 + (1 - x) * 2.5)) ** k / mp.factorial(k), [0, 1]))
          for k in range(2)]
    o, S, coeff, err, _ = run(wl, 10007)
    assert_within(coeff, err, ex)
    sec = S.mean(axis=2)
    assert abs(sec[0, 1] - sec[1, 1]) > 1e-3


# ------------------------------------------------------------------------- triangle (2-dim, double pole)
def test_triangle_dirichlet_closed_form():
    s = -2.0
    J = lambda e: mp.mpf(-s) ** (-1 - e) * mp.gamma(-e) ** 2 / mp.gamma(1 - 2 * e)
    ex = laurent(J, -2, 1)
    assert ex == pytest.approx([0.5, -0.346573590279973, -0.702353779944563, -0.659718252170579], abs=1e-14)
    o, S, coeff, err, cnt = run(qi.triangle(s), 32749)
    assert (o.k_min, o.k_max) == (-2, 1) and not cnt.any()
    assert_within(coeff, err, ex)
    assert np.all(err.real < 5e-6)


# ------------------------------------------------------------------------- config 2: massless box
def box_exact(s, t, kmax):
    """Gamma(2+eps) J = r_G/(st) (2/eps^2) [(-t)^-eps 2F1(1,-eps;1-eps;1+t/s) + (-s)^-eps 2F1(1,-eps;1-eps;1+s/t)].
    For s,t < 0 both 2F1 sit on their cut (argument > 1); the Euclidean integral is real and equals the
    real part (e^{-+ i pi eps} -> cos(pi eps) in the connection formula).  Orders eps^-2..eps^0 are
    cross-checked below against the textbook expansion r_G/(st){(2/eps^2)[(-s)^-eps+(-t)^-eps] - ln^2(s/t) - pi^2}."""
    def GJ(e):
        rG = mp.gamma(1 + e) * mp.gamma(1 - e) ** 2 / mp.gamma(1 - 2 * e)
        a = mp.mpf(-t) ** (-e) * mp.re(mp.hyp2f1(1, -e, 1 - e, 1 + mp.mpf(t) / s))
        b = mp.mpf(-s) ** (-e) * mp.re(mp.hyp2f1(1, -e, 1 - e, 1 + mp.mpf(s) / t))
        return rG / (mp.mpf(s) * t) * 2 / e ** 2 * (a + b)
    return laurent(lambda e: GJ(e) / mp.gamma(2 + e), -2, kmax)


def box_textbook(s, t):
    def GJ(e):
        rG = mp.gamma(1 + e) * mp.gamma(1 - e) ** 2 / mp.gamma(1 - 2 * e)
        return rG / (mp.mpf(s) * t) * (2 / e ** 2 * (mp.mpf(-s) ** (-e) + mp.mpf(-t) ** (-e))
                                       - mp.log(mp.mpf(s) / t) ** 2 - mp.pi ** 2)
    return laurent(lambda e: GJ(e) / mp.gamma(2 + e), -2, 0)


def test_massless_box_closed_form_config2():
    ex = box_exact(-3, -2, 1)
    assert ex[:3] == pytest.approx(box_textbook(-3, -2), abs=1e-14)
    assert ex == pytest.approx([0.666666666666667, -1.2639198230760183, -1.2238036181980894, 0.13431230702503515],
                               abs=1e-13)
    o, S, coeff, err, cnt = run(qi.massless_box(), 32749, m=8, eps_order=1)
    assert not cnt.any()
    assert_within(coeff, err, ex)
    assert np.all(err.real < 2e-5)
    # symmetry: primary sectors 1<->3 and 2<->4 (F = -s x2x4 - t x1x3) have equal sums
    prim = np.array([o.sector(i)["primary"] for i in range(o.n_sectors)])
    psum = np.array([S[prim == p].sum(axis=0) for p in range(4)])       # [4, K, m]
    for a, b in ((0, 2), (1, 3)):
        d = (psum[a] - psum[b]).mean(axis=1).real
        sd = (psum[a] - psum[b]).real.std(axis=1, ddof=1) / np.sqrt(S.shape[2])
        assert np.all(np.abs(d) <= 4 * sd + 1e-13)


def test_massless_box_closed_form_with_the_second_order_transform():
    # transform = 2 (R:C20, the r = 2 member of Eq. 21's family) changes the points, not the integral: same closed form,
    # and at equal N the error bars are not worse than with Eq. 21
    ex = box_exact(-3, -2, 0)
    wl = qi.massless_box()
    o = Oracle.from_workload(wl)
    N = 32749
    z = qi.good_vector(N, o.dim)
    sh = qi.splitmix64_shifts(wl.seed, 8, o.dim)
    S2, _, cnt = o.integrate(N, z, sh, transform=2)
    c2, e2 = o.totals(S2)
    assert not cnt.any()
    assert_within(c2, e2, ex, nsig=4.0)
    S0, _, _ = o.integrate(N, z, sh)
    _, e0 = o.totals(S0)
    assert np.all(e2.real < 2e-5) and e2.real[-1] < 3 * e0.real[-1]


def test_massless_box_crossing_symmetry():
    assert box_exact(-3, -2, 0) == pytest.approx(box_exact(-2, -3, 0), abs=1e-14)
    _, _, c1, e1, _ = run(qi.massless_box(-3.0, -2.0), 16381, m=6)
    _, _, c2, e2, _ = run(qi.massless_box(-2.0, -3.0), 16381, m=6)
    assert np.all(np.abs(c1 - c2).real <= 3 * np.hypot(e1.real, e2.real))


# ------------------------------------------------------------------------- config 4: double box
def test_double_box_leading_poles_and_symmetry_config4():
    """f(eps) = -e^{2 eps gammaE} (-s)^{2+2eps} (-t) Gamma(3+2eps) J = -4/eps^4 + 5 ln x/eps^3
    - (2 ln^2 x - 5 pi^2/2)/eps^2 + ...,  x = t/s  (three leading poles only)."""
    s, t = -3.0, -1.0
    x = mp.mpf(t) / s
    f = [-4, 5 * mp.log(x), -(2 * mp.log(x) ** 2 - 5 * mp.pi ** 2 / 2)]
    pref = lambda e: -mp.exp(2 * e * mp.euler) * mp.mpf(-s) ** (2 + 2 * e) * mp.mpf(-t) * mp.gamma(3 + 2 * e)
    inv = mp.taylor(lambda e: 1 / pref(e), 0, 2)
    ex = [float(sum(f[i] * inv[k - i] for i in range(k + 1))) for k in range(3)]
    assert ex[0] == pytest.approx(2.0 / 9.0, abs=1e-15)
    o, S, coeff, err, cnt = run(qi.double_box(s, t), 16381, m=8)
    assert o.n_sectors == 293 and (o.k_min, o.k_max) == (-4, 0) and not cnt.any()
    assert_within(coeff[:3], err[:3], ex, nsig=4.0)  # 8 shifts: Student-t tails
    assert np.all(err.real[:3] < 2e-3)
    # graph symmetry: the four rails e1..e4 have equal primary-sector sums, so have the outer rungs e5, e7,
    # although their sub-sector counts differ (28,28,28,32 and 75,68)
    prim = np.array([o.sector(i)["primary"] for i in range(o.n_sectors)])
    psum = np.array([S[prim == p].sum(axis=0).real for p in range(7)])   # [7, K, m]
    m = S.shape[2]
    for a, b in ((0, 1), (0, 2), (0, 3), (4, 6)):
        d = psum[a] - psum[b]
        assert np.all(np.abs(d.mean(axis=1)) <= 4.5 * d.std(axis=1, ddof=1) / np.sqrt(m) + 1e-12)
    # middle rung e6 has no eps^-4, eps^-3 poles
    assert np.all(np.abs(psum[5][:2].mean(axis=1)) <= 4.5 * psum[5][:2].std(axis=1, ddof=1) / np.sqrt(m) + 1e-12)
