"""Statistical pins of the oracle ("O9 statistics" and "cfg4 double box (v)"), CPU only.

1. The shifted-lattice estimator is unbiased and Eq. 20 is an unbiased estimate of its variance:
   over many seeds the pull (estimate - closed form) / error has mean ~ 0 and rms ~ 1 (for m shifts it follows a
   Student t distribution with m - 1 degrees of freedom: rms = sqrt((m-1)/(m-3))).
2. The Laurent coefficients of J do not depend on the decomposition strategy (reading C23): the double box decomposed
   U^-first (293 sectors, the rule of every config) and F^-first (522 sectors) gives the same totals within errors.
"""
import numpy as np
import pytest

import qmc_inputs as qi
from oracle import Oracle

N_SEEDS = 120


def pulls(o, exact, N, z, m, dim, orders):
    out = []
    for seed in range(1000, 1000 + N_SEEDS):
        S, A, cnt = o.integrate(N, z, qi.splitmix64_shifts(seed, m, dim))
        coeff, err = o.totals(S)
        out.append([(coeff[k].real - exact[k]) / err[k].real for k in orders])
    return np.array(out)


def check_pulls(P, m):
    t_rms = np.sqrt((m - 1.0) / (m - 3.0))
    mean, rms = P.mean(axis=0), np.sqrt((P ** 2).mean(axis=0))
    # 120 samples: the mean of a unit-variance pull scatters by 0.09 * t_rms, its rms by about 10 %
    assert np.all(np.abs(mean) < 0.4 * t_rms), (mean, rms)
    assert np.all(rms > 0.7 * t_rms) and np.all(rms < 1.45 * t_rms), (mean, rms)


def test_pull_distribution_bubble():
    """Config 1: J = 1 - 0.152044704820020194 eps + ... (closed form of BASELINE.json, tests/test_oracle_closed_forms.py)."""
    o = Oracle.from_workload(qi.bubble())
    N, m = 251, 8
    P = pulls(o, {1: 2.0 - np.sqrt(5.0) * np.log((np.sqrt(5.0) + 1.0) / (np.sqrt(5.0) - 1.0))}, N, np.array([1], dtype=np.uint64), m, 1, [1])
    check_pulls(P, m)


def test_pull_distribution_massless_box():
    """Config 2: the three coefficients eps^-2 .. eps^0 of the closed form."""
    o = Oracle.from_workload(qi.massless_box())
    exact = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    N, m = 1021, 8
    P = pulls(o, exact, N, qi.korobov_vector(N, 3, 331), m, 3, [0, 1, 2])
    check_pulls(P, m)


def test_double_box_totals_do_not_depend_on_the_decomposition_order():
    wl = qi.double_box()
    a = Oracle.from_workload(wl)             # U^ first: rule A.3
    b = Oracle.from_workload(wl, order=1)    # F^ first
    assert (a.n_sectors, b.n_sectors) == (293, 522) and a.status == 0 and b.status == 0
    N, m = 4093, 6
    z = qi.korobov_vector(N, 6, 1487)
    sh = qi.splitmix64_shifts(wl.seed, m, 6)
    (ca, ea), (cb, eb) = (o.totals(o.integrate(N, z, sh)[0]) for o in (a, b))
    for k in range(5):
        sig = np.hypot(ea[k].real, eb[k].real)
        assert abs(ca[k].real - cb[k].real) <= 4.0 * sig, (k, ca[k], cb[k], sig)
    # and both agree with the three analytic poles (tests/test_oracle_closed_forms.py)
    ex = [2.0 / 9.0, -0.8497687147780183, 0.003001503361321066]
    for c, e in ((ca, ea), (cb, eb)):
        assert np.all(np.abs(c.real[:3] - ex) <= 4.0 * e.real[:3])
