"""Worked-example pin: the paper's own Table 1 reproduced by the oracle.

Same graph as config 4 (Eq. 23) with two legs off-shell at s = t = u = -2/3; values stored
in tests/golden/paper_table1.txt.  P_i = coefficient of eps^-i of e^{2 eps gammaE} (-s)^{3+2eps}
Gamma(3+2eps) J(eps)  (Eq. 24 with the readings C1-C4 of DESIGN.md).  CPU only.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import qmc_inputs as qi
from oracle import Oracle

mp.mp.dps = 30
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_table1.txt")


def load_table():
    rows = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        legs, i, vegas, qmc = [x.strip() for x in line.split("|")]
        legs = tuple(float(x) for x in legs.split())
        rows.setdefault(legs, {})[int(i)] = (tuple(float(x) for x in vegas.split()), tuple(float(x) for x in qmc.split()))
    return rows


@pytest.mark.parametrize("legs", sorted(load_table()), ids=str)
def test_paper_table1(legs):
    table = load_table()[legs]
    s = t = -2.0 / 3.0
    wl = qi.double_box(s, t, p2=legs)
    o = Oracle.from_workload(wl)
    assert o.status == 0 and o.k_max == 0
    N, m = 16381, 6
    S, A, cnt = o.integrate(N, qi.good_vector(N, 6), qi.splitmix64_shifts(101, m, 6))
    assert not cnt.any()
    # prefactor series, then per-shift P_i so that the error bars include the correlations between orders
    pref = mp.taylor(lambda e: mp.exp(2 * e * mp.euler) * mp.mpf(-s) ** (3 + 2 * e) * mp.gamma(3 + 2 * e), 0, 4)
    pref = np.array([float(x) for x in pref])
    T = S.sum(axis=0).real                       # [K, m], orders k_min..0
    K = T.shape[0]
    full = np.zeros((5, m))                      # orders -4..0
    full[5 - K:] = T
    for i in range(5):                           # P_i: order -i
        k = 4 - i                                # index of eps^-i in `full`
        Pi = sum(pref[q] * full[k - q] for q in range(k + 1))
        mean, err = Pi.mean(), Pi.std(ddof=1) / np.sqrt(m)
        # the oracle's own error must be small enough for the comparison to mean something
        assert err <= max(2e-3 * abs(table[i][1][0]), 1e-5), (i, err)
        for val, perr in table[i]:               # both printed columns (Vegas/CPU and QMC/GPU)
            tol = 4.0 * np.hypot(err, perr) + 1e-5 * max(1.0, abs(val))
            assert abs(mean - val) <= tol, (legs, i, mean, err, val, perr)
