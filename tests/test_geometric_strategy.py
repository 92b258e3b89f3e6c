"""Geometric decomposition strategy (qmc_options.strategy = 1, reading C31): the strategy the paper says
it uses.  Host logic only (no GPU): the sectors it emits are evaluated by the ORACLE from the exported
tables, so what is pinned here is the decomposition -- every sector in the form of Eqs. 7-9 (a monomial times
polynomials with a constant term), and, since per-sector numbers depend on the strategy and totals do not (reading C23), the
totals against closed forms and against the iterated strategy of reading C7."""
import dataclasses

import numpy as np
import pytest

import qmc_inputs as qi
import paper_1508_02512_b200 as q
from oracle import Oracle

WORKLOADS = [qi.bubble(), qi.triangle(), qi.massless_box(), qi.massive_box(), qi.double_box(), qi.nonplanar_vertex(), qi.paper_IC(),
             qi.paper_ID(), qi.double_box(-2 / 3, -2 / 3, p2=(0, 0, -1, -1))]


def tables(wl, strategy, eps_order=None):
    return q.qmc_prepare(wl, eps_order=wl.eps_order if eps_order is None else eps_order, lam=wl.lam, strategy=strategy)


def totals(wl, strategy, N, m, transform=0):
    o = Oracle.from_tables(tables(wl, strategy).export())
    S, A, cnt = o.integrate(N, qi.good_vector(N, o.dim), qi.splitmix64_shifts(wl.seed, m, o.dim), transform=transform)
    assert not cnt.any()
    c, e = o.totals(S)
    return c, e


@pytest.mark.parametrize("wl", WORKLOADS, ids=lambda w: w.name)
def test_every_geometric_sector_has_the_form_of_eqs_7_to_9(wl):
    t = tables(wl, 1)
    o = Oracle.from_tables(t.export())
    it = Oracle.from_tables(tables(wl, 0).export())
    assert o.status == 0 and o.n_sectors >= wl.n_edges and (o.k_min, o.k_max) == (it.k_min, it.k_max)
    assert (o.aU0, o.aU1, o.aF0, o.aF1) == (it.aU0, it.aU1, it.aF0, it.aF1)
    primaries = set()
    for s in range(o.n_sectors):
        sec = o.sector(s)
        primaries.add(sec["primary"])
        for which in "UF":
            coeff, expo = sec[which]
            assert (expo.sum(axis=1) == 0).sum() == 1, (wl.name, s, which)        # exactly one constant term
            assert np.all(expo >= 0) and np.all(expo.min(axis=0) == 0)              # nothing left to factor out
        assert np.all(sec["alpha"] >= -1) and sec["n_sing"] <= 4
        assert np.all(sec["beta"][sec["alpha"] == -1] != 0)
    assert primaries == set(range(wl.n_edges))                                      # every primary sector of Eqs. 3-6 is covered


def test_sector_counts_of_the_geometric_strategy():
    # regression values of this implementation (the triangulation of a non-simplicial cone is not unique: another valid choice gives
    # other counts); the iterated rule of reading C7 gives 2 / 3 / 12 / 4 / 293 / 36 / 46 / 48
    got = {wl.name: Oracle.from_tables(tables(wl, 1).export()).n_sectors for wl in WORKLOADS[:8]}
    assert got == {"cfg1_bubble": 2, "triangle": 3, "cfg2_massless_box": 12, "cfg3_massive_box": 4, "cfg4_double_box": 266,
                   "cfg5_nonplanar_vertex": 36, "paper_IC_planar_double_box": 46, "paper_ID_nonplanar_double_box": 48}


def test_totals_against_closed_forms_and_against_the_iterated_strategy():
    # massless box: closed form through eps^0 (tests/test_oracle_closed_forms.py)
    c, e = totals(qi.massless_box(), 1, 32749, 8)
    ex = np.array([0.666666666666667, -1.2639198230760183, -1.2238036181980894])
    assert np.all(np.abs(c.real - ex) <= 4 * e.real)
    # double box: the three leading poles in closed form, all five orders against the iterated strategy
    cg, eg = totals(qi.double_box(), 1, 16381, 4)
    ci, ei = totals(qi.double_box(), 0, 16381, 4)
    ex4 = np.array([2.0 / 9.0, -0.8497687147780183, 0.003001503361321066])
    assert np.all(np.abs(cg.real[:3] - ex4) <= 4 * eg.real[:3]), (cg.real, eg.real)
    assert np.all(np.abs(cg.real - ci.real) <= 4 * np.hypot(eg.real, ei.real)), (cg.real, ci.real, eg.real, ei.real)
    assert np.all(eg.real <= 3e-2 * np.maximum(np.abs(cg.real), 1e-2))
    # complex path: the non-planar vertex of config 5 (36 sectors under both strategies, different ones)
    cg, eg = totals(qi.nonplanar_vertex(), 1, 16381, 6)
    ci, ei = totals(qi.nonplanar_vertex(), 0, 16381, 6)
    assert np.all(np.abs(cg.real - ci.real) <= 4 * np.hypot(eg.real, ei.real)) and np.all(np.abs(cg.imag - ci.imag) <= 4 * np.hypot(eg.imag, ei.imag))


def test_geometric_strategy_with_propagator_powers_and_other_options():
    import mpmath as mp
    # triangle with a squared propagator (a sector with alpha = -2): Dirichlet's integral, through IBP and Eq. 21's transform
    nu, s = (1, 1, 2), -2.0
    wl = dataclasses.replace(qi.triangle(s), nu=nu, eps_order=0)
    t = q.qmc_prepare(wl, eps_order=0, strategy=1, pole_extraction=1)
    o = Oracle.from_tables(t.export())
    S, A, cnt = o.integrate(99991, qi.good_vector(99991, 2), qi.splitmix64_shifts(3, 8, 2))
    c, e = o.totals(S)
    assert np.all(np.abs(c.real - [0.0, 0.5, -0.8465735902799727]) <= 4 * e.real + 1e-9), (c.real, e.real)
    with pytest.raises(q.QmcError) as err:
        q.qmc_prepare(qi.massless_box(), strategy=2)
    assert err.value.status == -1


def test_random_graphs_either_decompose_into_the_form_of_eqs_7_to_9_or_fail_with_a_status():
    """Robustness of the host code on inputs nobody chose: random connected multigraphs (2-5 vertices, up to 7 edges, up to six
    loops), random masses, Euclidean momenta with some light-like legs, random propagator powers, both strategies and both pole
    extractions.  Every call either returns tables whose sectors have the form of Eqs. 7-9 or a status (unsupported, depth cap);
    the geometric strategy never runs into the depth cap (it does not iterate), and its work budget keeps a call short."""
    import collections
    import time
    from qmc_inputs import Workload
    rng = np.random.default_rng(7)
    stat = collections.Counter()
    t_begin = time.time()
    for it in range(60):
        V = int(rng.integers(2, 6)); P = int(rng.integers(max(V, 2), 8))
        edges = [(int(rng.integers(0, v)), v) for v in range(1, V)]
        while len(edges) < P:
            a, b = int(rng.integers(0, V)), int(rng.integers(0, V))
            if a != b or rng.random() < 0.05:
                edges.append((a, b))
        masses = [float(rng.choice([0.0, 0.0, 1.0, 2.5])) for _ in edges]
        nl = int(rng.integers(2, min(V, 4) + 1))
        legs = [int(x) for x in rng.choice(V, size=nl, replace=False)]
        p = rng.normal(size=(nl, 4)); p[-1] = -p[:-1].sum(axis=0)
        gram = -(p @ p.T)
        if rng.random() < 0.3:
            for i in range(nl):
                if rng.random() < 0.5:
                    gram[i, i] = 0.0
        nu = None if rng.random() < 0.5 else [int(rng.choice([1, 1, 2, 3])) for _ in edges]
        wl = Workload("random", V, [(a, b, m) for (a, b), m in zip(edges, masses)], legs, gram)
        for strategy in (0, 1):
            for pole in (0, 1):
                t0 = time.time()
                try:
                    t = q.qmc_prepare(wl, eps_order=int(rng.integers(0, 3)), strategy=strategy, pole_extraction=pole, nu=nu, max_depth=12)
                except q.QmcError as e:
                    assert e.status in (-2, -3) and not (strategy == 1 and e.status == -2), (it, strategy, e.status)
                    stat[("status", strategy, e.status)] += 1
                    continue
                finally:
                    assert time.time() - t0 < 20.0, (it, strategy, "qmc_prepare took too long")
                o = Oracle.from_tables(t.export())
                for s in range(min(o.n_sectors, 30)):
                    sec = o.sector(s)
                    for which in "UF":
                        coeff, expo = sec[which]
                        assert (expo.sum(axis=1) == 0).sum() == 1 and np.all(expo.min(axis=0) == 0), (it, strategy, s, which)
                stat[("tables", strategy)] += 1
    assert stat[("tables", 0)] > 40 and stat[("tables", 1)] > 40, dict(stat)
    assert time.time() - t_begin < 240.0
