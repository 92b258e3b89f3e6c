"""Pins of the oracle's p >= 1 Taylor terms (Eq. 11, reading C28) and of propagator
powers nu_j (Eq. 1), against what does not come from the oracle:

* the Taylor-term formula must reduce to the explicit double sum (A.4a) wherever every alpha_j >= -1;
* integrals of monomials, int_0^1 t^(k-a+b eps) dt = 1/(k+1-a+b eps), summed over a binomial expansion;
* int_0^1 t^eps/(1+t) dt = sum_k (-eps)^k eta(k+1) (Dirichlet eta) after partial fractions;
* Euler's integral int_0^1 t^(s-1) (1+t)^e dt = 2F1(-e, s; s+1; -1)/s continued to s = -1 + e;
* the massless one-loop propagator with powers (nu1, nu2): J = (-p^2)^(D/2-nu1-nu2) B(D/2-nu1, D/2-nu2);
* the one-loop triangle with two light-like legs and powers nu: a Dirichlet integral of Gamma functions;
* a massive bubble with a squared propagator: one-dimensional quadrature over the simplex form of the parameter integral.

Laurent coefficients of the Gamma-function expressions are taken with mpmath on a circle around eps = 0.
Lattice runs use the tent transform (reading C20): with t ~ y^2 of Eq. 21 the cancellation [g - g_0 - t g_1]/t^2 of a
variable with alpha = -2 loses four digits per decade of y (reading C28).
"""
import dataclasses

import mpmath as mp
import numpy as np
import pytest

import qmc_inputs as qi
from oracle import Oracle

mp.mp.dps = 30


def laurent(f, kmin, kmax, radius=0.25, npts=64):
    """Coefficients of eps^kmin .. eps^kmax of f, analytic on 0 < |eps| <= radius, by the trapezoidal rule on the circle."""
    vals = [f(radius * mp.e ** (2j * mp.pi * i / npts)) for i in range(npts)]
    return np.array([float((sum(v * mp.e ** (-2j * mp.pi * i * k / npts) for i, v in enumerate(vals)) / npts / radius ** k).real)
                     for k in range(kmin, kmax + 1)])


def lattice_estimate(o, N=65521, m=8, seed=5, transform=1):
    z = qi.good_vector(N, o.dim)
    sh = qi.splitmix64_shifts(seed, m, o.dim)
    S, A, cnt = o.integrate(N, z, sh, transform=transform)
    assert cnt[2] == 0
    c, e = o.totals(S)
    return c.real, e.real


def agree(got, err, want, nsigma=4.0):
    got, err, want = np.asarray(got), np.asarray(err), np.asarray(want)
    assert got.shape == want.shape, (got.shape, want.shape)
    tol = nsigma * err + 1e-11 * np.maximum(1.0, np.abs(want))
    assert np.all(np.abs(got - want) <= tol), (got, err, want, (got - want) / np.maximum(err, 1e-300))
    assert np.all(err <= 1e-3 * np.maximum(1.0, np.abs(want))), ("error bars too wide to pin anything", err)


ONE = [(1.0, (0,))]
ONE_PLUS_T = [(1.0, (0,)), (1.0, (1,))]


@pytest.mark.parametrize("wl", [qi.massless_box(), qi.double_box(), qi.triangle(), qi.bubble()], ids=lambda w: w.name)
def test_taylor_formula_reduces_to_the_double_sum_without_deep_variables(wl):
    o = Oracle.from_workload(wl)
    rng = np.random.default_rng(1)
    for s in rng.choice(o.n_sectors, size=min(o.n_sectors, 16), replace=False):
        t = rng.uniform(0.02, 0.98, o.dim)
        a = o.sector_integrand(int(s), t)
        b, mag = o.sector_integrand_taylor(int(s), t)
        assert np.all(a.imag == 0.0) and np.all(np.abs(a.real - b) <= 1e-14 * mag), (s, a.real, b)


def test_one_variable_binomial_closed_forms():
    # int t^(-2+eps) (1+t)^2 = 1/(-1+eps) + 2/eps + 1/(1+eps): eps^k coefficient -1 + (-1)^k for k >= 0, pole 2/eps
    o = Oracle.from_sector([-2], [1], ONE_PLUS_T, ONE, (2, 0), (0, 0), eps_order=2)
    assert (o.status, o.k_min, o.k_max) == (0, -1, 2)
    c, e = lattice_estimate(o)
    agree(c, e, [2.0, 0.0, -2.0, 0.0])
    # int t^(-3+2 eps) (1+t)^3 = 1/(-2+2e) + 3/(-1+2e) + 3/(2e) + 1/(1+2e): two non-pole Taylor terms
    o = Oracle.from_sector([-3], [2], ONE_PLUS_T, ONE, (3, 0), (0, 0), eps_order=1)
    c, e = lattice_estimate(o)
    agree(c, e, [1.5, -0.5 - 3.0 + 1.0, -0.5 - 6.0 - 2.0])
    # the same power through F with a negative integer exponent of the other polynomial switched off: (1+t)^2 as U^4 F^-2
    o = Oracle.from_sector([-2], [1], ONE_PLUS_T, ONE_PLUS_T, (4, 0), (-2, 0), eps_order=2)
    c, e = lattice_estimate(o)
    agree(c, e, [2.0, 0.0, -2.0, 0.0])


def test_one_variable_reciprocal_and_dirichlet_eta():
    # t^-2/(1+t) = 1/t^2 - 1/t + 1/(1+t):  1/(-1+eps) - 1/eps + sum_k (-eps)^k eta(k+1), eta(1) = ln 2, eta(s) = (1-2^(1-s)) zeta(s)
    o = Oracle.from_sector([-2], [1], ONE, ONE_PLUS_T, (0, 0), (-1, 0), eps_order=2)
    c, e = lattice_estimate(o)
    eta = [float(mp.log(2))] + [float((1 - mp.mpf(2) ** (1 - s)) * mp.zeta(s)) for s in (2, 3)]
    agree(c, e, [-1.0] + [-1.0 + (-1) ** k * eta[k] for k in range(3)])


def test_one_variable_eps_dependent_exponent_against_eulers_integral():
    # int_0^1 t^(s-1) (1+t)^e dt = 2F1(-e, s; s+1; -1) / s, continued to s = -1 + e; its eps^1 coefficient is -2 ln 2
    o = Oracle.from_sector([-2], [1], ONE_PLUS_T, ONE, (0, 1), (0, 0), eps_order=2)
    c, e = lattice_estimate(o)
    want = laurent(lambda x: mp.hyp2f1(-x, -1 + x, x, -1) / (-1 + x), -1, 2)
    assert abs(want[0]) < 1e-20 and abs(want[1]) < 1e-20 and abs(want[2] + 2 * np.log(2.0)) < 1e-14
    agree(c, e, want)


def test_two_variables_non_separable_polynomial():
    # t1^(-2+eps) t2^(-1+2 eps) (1+t1+t2)^2 (1+t1 t2): sum over the monomials t1^i t2^j of c_ij / ((i-1+eps)(j+2 eps))
    U = [(1.0, (0, 0)), (1.0, (1, 0)), (1.0, (0, 1))]
    F = [(1.0, (0, 0)), (1.0, (1, 1))]
    o = Oracle.from_sector([-2, -1], [1, 2], U, F, (2, 0), (1, 0), eps_order=1)
    assert (o.k_min, o.k_max) == (-2, 1)
    c, e = lattice_estimate(o)
    poly = {}
    for (i1, j1, c1) in ((0, 0, 1), (1, 0, 1), (0, 1, 1)):
        for (i2, j2, c2) in ((0, 0, 1), (1, 0, 1), (0, 1, 1)):
            for (i3, j3, c3) in ((0, 0, 1), (1, 1, 1)):
                key = (i1 + i2 + i3, j1 + j2 + j3)
                poly[key] = poly.get(key, 0) + c1 * c2 * c3
    want = laurent(lambda x: sum(cf / ((i - 1 + x) * (j + 2 * x)) for (i, j), cf in poly.items()), -2, 1)
    agree(c, e, want)
    assert abs(want[0] - 1.0) < 1e-14 and abs(want[1] - 13.0 / 3.0) < 1e-13


@pytest.mark.parametrize("nu", [(3, 1), (1, 3), (2, 1), (2, 2)])
def test_massless_propagator_with_powers_against_the_beta_function(nu):
    # textbook: int d^Dk/(i pi^(D/2)) 1/((-k^2)^a (-(k+p)^2)^b) = (-p^2)^(D/2-a-b) G(D/2-a) G(D/2-b) G(a+b-D/2)/(G(a) G(b) G(D-a-b));
    # without the prefactor G(a+b-D/2)/(G(a)G(b)) of Eq. 2: J = (-p^2)^(D/2-a-b) B(D/2-a, D/2-b)
    p2 = -1.7
    wl = dataclasses.replace(qi.bubble(p2, 0.0, 0.0), nu=nu, eps_order=1)
    o = Oracle.from_workload(wl, taylor=True)
    assert o.status == 0 and o.n_sectors == 2
    a, b = nu
    # sector x1 = 1: t^(b-1) F^(-(a+b-2)) with F = (-p^2) t, i.e. alpha = 1 - a; sector x2 = 1: alpha = 1 - b
    assert sorted(int(o.sector(s)["alpha"][0]) for s in range(o.n_sectors)) == sorted((1 - a, 1 - b))
    c, e = lattice_estimate(o)
    want = laurent(lambda x: (-p2) ** (2 - x - a - b) * mp.beta(2 - x - a, 2 - x - b), o.k_min, 1)
    agree(c, e, want)


@pytest.mark.parametrize("nu", [(2, 1, 1), (1, 1, 2), (1, 2, 1)])
def test_triangle_with_a_squared_propagator_against_the_dirichlet_integral(nu):
    # two light-like legs: F = (-s) x2 x3, and on the simplex U = 1, so that
    # J = (-s)^(D/2-N) G(nu1) G(nu2+D/2-N) G(nu3+D/2-N) / G(D-N),  N = nu1+nu2+nu3  (Dirichlet's integral)
    s = -2.0
    wl = dataclasses.replace(qi.triangle(s), nu=nu, eps_order=0)
    o = Oracle.from_workload(wl, taylor=True)
    cF, eF = o.graph_poly("F")
    assert o.status == 0 and len(cF) == 1 and tuple(eF[0]) == (0, 1, 1) and cF[0] == -s
    assert min(int(min(o.sector(k)["alpha"])) for k in range(o.n_sectors)) == -2     # a variable that needs the p = 1 term
    Nn = sum(nu)
    c, e = lattice_estimate(o, N=99991)
    want = laurent(lambda x: (-s) ** (2 - x - Nn) * mp.gamma(nu[0]) * mp.gamma(nu[1] + 2 - x - Nn) * mp.gamma(nu[2] + 2 - x - Nn)
                   / mp.gamma(4 - 2 * x - Nn), o.k_min, 0)
    agree(c, e, want)


def test_massive_bubble_with_a_squared_propagator_against_simplex_quadrature():
    # no singular variable: J = int_0^1 dx x^(nu1-1) (1-x)^(nu2-1) F(x)^(D/2-N), F = -p^2 x(1-x) + m1^2 x + m2^2 (1-x) (U = 1 on the simplex)
    p2, m1, m2 = -1.3, 1.0, 2.5
    for nu in ((2, 1), (1, 3)):
        wl = dataclasses.replace(qi.bubble(p2, m1, m2), nu=nu, eps_order=2)
        o = Oracle.from_workload(wl)                       # (no Taylor terms needed: every alpha_j >= 0)
        assert o.status == 0 and o.k_min == 0 and (o.aU0, o.aU1, o.aF0, o.aF1) == (sum(nu) - 4, 2, -(sum(nu) - 2), -1)
        c, e = lattice_estimate(o, N=10007, transform=0)
        F = lambda x: -p2 * x * (1 - x) + m1 * x + m2 * (1 - x)
        want = [float(mp.quad(lambda x: x ** (nu[0] - 1) * (1 - x) ** (nu[1] - 1) * F(x) ** (2 - sum(nu)) * (-mp.log(F(x))) ** k / mp.factorial(k),
                              [0, 1])) for k in range(3)]
        agree(c, e, want)


def test_deep_variables_are_refused_without_the_taylor_flag_and_on_the_complex_path():
    wl = dataclasses.replace(qi.bubble(-1.0, 0.0, 0.0), nu=(3, 1))
    assert Oracle.from_workload(wl).status == -3                       # reading C9 stays the default
    assert Oracle.from_workload(wl, taylor=True).status == 0
    assert Oracle.from_workload(wl, taylor=True, lam=0.5).status == -3  # the Taylor terms are real-path only
    with pytest.raises(ValueError):
        Oracle.from_workload(dataclasses.replace(qi.bubble(), nu=(0, 1)))
