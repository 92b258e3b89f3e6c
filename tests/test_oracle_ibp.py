"""Pins of the oracle's pole extraction by integration by parts (Eq. 13, reading C30).

IBP and the subtraction (Eqs. 11-12) are different integrands with the same integral, so nothing here compares the two
point by point: the pins are the closed forms of tests/test_oracle_taylor_terms.py and tests/test_oracle_closed_forms.py again
(monomial integrals, Dirichlet eta values, Euler's hypergeometric integral, Beta function, Dirichlet's integral, the massless
box), reached this time through sector_point_ibp, and the property the paper introduces IBP for: no large-number
cancellation, i.e. a cancellation factor A/|S| of order one where the subtraction has 1e5 .. 1e13.
All runs use the paper's own transform (Eq. 21): IBP has no 1/t to be squared by it.
"""
import dataclasses

import mpmath as mp
import numpy as np
import pytest

import qmc_inputs as qi
from oracle import Oracle

mp.mp.dps = 30


def laurent(f, kmin, kmax, radius=0.25, npts=64):
    vals = [f(radius * mp.e ** (2j * mp.pi * i / npts)) for i in range(npts)]
    return np.array([float((sum(v * mp.e ** (-2j * mp.pi * i * k / npts) for i, v in enumerate(vals)) / npts / radius ** k).real)
                     for k in range(kmin, kmax + 1)])


def lattice_estimate(o, N=65521, m=8, seed=5, transform=0):
    z = qi.good_vector(N, o.dim)
    sh = qi.splitmix64_shifts(seed, m, o.dim)
    S, A, cnt = o.integrate(N, z, sh, transform=transform)
    assert cnt[2] == 0
    c, e = o.totals(S)
    T, AT = S.sum(axis=0), A.sum(axis=0)
    kappa = np.where(np.abs(T) > 0, AT / np.maximum(np.abs(T), 1e-300), 0.0).max(axis=-1)
    return c.real, e.real, kappa


def agree(got, err, want, nsigma=4.0, floor=1e-9):
    got, err, want = np.asarray(got), np.asarray(err), np.asarray(want)
    assert got.shape == want.shape
    assert np.all(np.abs(got - want) <= nsigma * err + floor * np.maximum(1.0, np.abs(want))), (got, err, want, (got - want) / np.maximum(err, 1e-300))
    assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(want))), ("error bars too wide to pin anything", err)


ONE = [(1.0, (0,))]
ONE_PLUS_T = [(1.0, (0,)), (1.0, (1,))]


def test_one_variable_closed_forms_through_ibp():
    # int t^(-2+eps) (1+t)^2 = 1/(-1+eps) + 2/eps + 1/(1+eps)
    o = Oracle.from_sector([-2], [1], ONE_PLUS_T, ONE, (2, 0), (0, 0), eps_order=2, ibp=True)
    c, e, kappa = lattice_estimate(o)
    agree(c, e, [2.0, 0.0, -2.0, 0.0])
    # int t^(-3+2 eps) (1+t)^3: three partial integrations
    o = Oracle.from_sector([-3], [2], ONE_PLUS_T, ONE, (3, 0), (0, 0), eps_order=1, ibp=True)
    c, e, kappa = lattice_estimate(o)
    agree(c, e, [1.5, -2.5, -8.5])
    # t^-2/(1+t): 1/(-1+eps) - 1/eps + sum_k (-eps)^k eta(k+1)
    o = Oracle.from_sector([-2], [1], ONE, ONE_PLUS_T, (0, 0), (-1, 0), eps_order=2, ibp=True)
    c, e, kappa = lattice_estimate(o)
    eta = [float(mp.log(2))] + [float((1 - mp.mpf(2) ** (1 - s)) * mp.zeta(s)) for s in (2, 3)]
    agree(c, e, [-1.0] + [-1.0 + (-1) ** k * eta[k] for k in range(3)])
    # eps-dependent exponent: Euler's integral 2F1(-e, s; s+1; -1)/s at s = -1 + e
    o = Oracle.from_sector([-2], [1], ONE_PLUS_T, ONE, (0, 1), (0, 0), eps_order=2, ibp=True)
    c, e, kappa = lattice_estimate(o)
    agree(c, e, laurent(lambda x: mp.hyp2f1(-x, -1 + x, x, -1) / (-1 + x), -1, 2))
    # the plain alpha = -1 case: int t^(-1+eps) (1+t)^-1 = 1/eps - sum ... : f(1)/eps - (1/eps) int t^eps f'(t)
    o = Oracle.from_sector([-1], [1], ONE, ONE_PLUS_T, (0, 0), (-1, 0), eps_order=1, ibp=True)
    c, e, kappa = lattice_estimate(o)
    agree(c, e, [1.0, -eta[0], eta[1]])                    # 1/eps - int t^eps/(1+t) = 1/eps - ln 2 + eps pi^2/12 - ...


def test_two_variables_non_separable_through_ibp_without_cancellation():
    U = [(1.0, (0, 0)), (1.0, (1, 0)), (1.0, (0, 1))]
    F = [(1.0, (0, 0)), (1.0, (1, 1))]
    poly = {}
    for (i1, j1) in ((0, 0), (1, 0), (0, 1)):
        for (i2, j2) in ((0, 0), (1, 0), (0, 1)):
            for (i3, j3) in ((0, 0), (1, 1)):
                poly[(i1 + i2 + i3, j1 + j2 + j3)] = poly.get((i1 + i2 + i3, j1 + j2 + j3), 0) + 1
    want = laurent(lambda x: sum(cf / ((i - 1 + x) * (j + 2 * x)) for (i, j), cf in poly.items()), -2, 1)
    o = Oracle.from_sector([-2, -1], [1, 2], U, F, (2, 0), (1, 0), eps_order=1, ibp=True)
    c, e, kappa = lattice_estimate(o)
    agree(c, e, want)
    s = Oracle.from_sector([-2, -1], [1, 2], U, F, (2, 0), (1, 0), eps_order=1)
    cs, es, kappa_s = lattice_estimate(s)
    assert kappa.max() < 100.0 and kappa_s.max() > 1e6 * kappa.max(), (kappa, kappa_s)


@pytest.mark.parametrize("nu", [(1, 1), (2, 1), (3, 1), (2, 2)])
def test_massless_propagator_with_powers_through_ibp(nu):
    p2 = -1.7
    a, b = nu
    wl = dataclasses.replace(qi.bubble(p2, 0.0, 0.0), nu=nu, eps_order=1)
    o = Oracle.from_workload(wl, ibp=True)
    assert o.status == 0
    c, e, kappa = lattice_estimate(o)
    agree(c, e, laurent(lambda x: (-p2) ** (2 - x - a - b) * mp.beta(2 - x - a, 2 - x - b), o.k_min, 1))
    assert kappa.max() < 100.0


@pytest.mark.parametrize("nu", [(1, 1, 1), (2, 1, 1), (1, 1, 2)])
def test_triangle_through_ibp_against_the_dirichlet_integral(nu):
    s = -2.0
    wl = dataclasses.replace(qi.triangle(s), nu=nu, eps_order=0)
    o = Oracle.from_workload(wl, ibp=True)
    Nn = sum(nu)
    c, e, kappa = lattice_estimate(o, N=99991)
    want = laurent(lambda x: (-s) ** (2 - x - Nn) * mp.gamma(nu[0]) * mp.gamma(nu[1] + 2 - x - Nn) * mp.gamma(nu[2] + 2 - x - Nn)
                   / mp.gamma(4 - 2 * x - Nn), -2, 0)
    agree(c, e, want)
    assert kappa.max() < 100.0
    if nu != (1, 1, 1):    # the same graph through the subtraction: eleven orders of magnitude more cancellation
        cs, es, kappa_s = lattice_estimate(Oracle.from_workload(wl, taylor=True), N=99991)
        assert kappa_s.max() > 1e6 * kappa.max(), (kappa, kappa_s)


def test_massless_box_through_ibp_against_its_closed_form():
    # config 2 (s = -3, t = -2): the values of tests/test_oracle_closed_forms.py
    o = Oracle.from_workload(qi.massless_box(), ibp=True)
    c, e, kappa = lattice_estimate(o, N=32749)
    agree(c, e, [0.666666666666667, -1.2639198230760183, -1.2238036181980894])
    assert kappa.max() < 100.0


def test_ibp_is_real_path_only():
    with pytest.raises(ValueError):
        Oracle.from_workload(qi.massive_box(), ibp=True)
