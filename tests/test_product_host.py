"""CPU-only checks of the product library: it loads, exports every symbol of include/qmc_feynman.h, and its
host stage (qmc_prepare: decomposer + tables) agrees with the independently written oracle.  No compute calls."""
import ctypes
import os
import re

import mpmath as mp
import numpy as np
import pytest

import qmc_inputs as qi
import paper_1508_02512_b200 as q
from oracle import Oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "qmc_feynman.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(qmc_[a-z0-9_]+)\s*\(", hdr)))
    assert {"qmc_prepare", "qmc_integrate", "qmc_integrate_ex", "qmc_tables_export", "qmc_tables_free",
            "qmc_tables_info", "qmc_workspace_bytes", "qmc_strerror"} <= set(names)
    L = q.lib()
    for n in names:
        assert hasattr(L, n), n
    assert q.strerror(0) == "ok" and "CUDA" in q.strerror(-4)


def parse_export(words):
    d = words.view(np.float64)
    assert words[0] == 0x514D4346 and words[1] == 1
    nsec, n = int(words[2]), int(words[3])
    hdr = dict(n_sectors=nsec, dim=n, k_min=int(words[4]), k_max=int(words[5]), is_complex=int(words[6]),
               a=tuple(int(x) for x in words[7:11]), lam=float(d[11]))
    p = 12
    secs = []
    for _ in range(nsec):
        primary = int(words[p]); p += 1
        alpha = words[p:p + n].copy(); p += n
        beta = words[p:p + n].copy(); p += n
        nU, nF = int(words[p]), int(words[p + 1]); p += 2
        polys = []
        for cnt in (nU, nF):
            mon = {}
            for _ in range(cnt):
                c = float(d[p]); e = tuple(int(x) for x in words[p + 1:p + 1 + n]); p += 1 + n
                mon[e] = c
            polys.append(mon)
        secs.append(dict(primary=primary, alpha=alpha, beta=beta, U=polys[0], F=polys[1]))
    assert p == len(words)
    return hdr, secs


WORKLOADS = qi.CONFIGS() + [qi.triangle(), qi.double_box(-2 / 3, -2 / 3, p2=(0, -1, 0, -1)),
                            qi.double_box(-2 / 3, -2 / 3, p2=(-1, 0, 0, -1))]


@pytest.mark.parametrize("wl", WORKLOADS, ids=lambda w: w.name + str(w.gram[0, 0]) + str(w.gram[1, 1]))
def test_prepare_matches_oracle_decomposition(wl):
    """Two independent decomposers (oracle: std::map + recursion + subset enumeration of forests; product: packed
    keys + explicit stack + deletion/contraction) must emit the same sectors in the same order."""
    t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
    o = Oracle.from_workload(wl)
    hdr, secs = parse_export(t.export())
    assert (t.n_sectors, t.dim, t.k_min, t.k_max) == (o.n_sectors, o.dim, o.k_min, o.k_max)
    assert hdr["a"] == (o.aU0, o.aU1, o.aF0, o.aF1) and hdr["lam"] == wl.lam and hdr["is_complex"] == (wl.lam > 0)
    for i, s in enumerate(secs):
        os_ = o.sector(i)
        assert s["primary"] == os_["primary"]
        assert np.array_equal(s["alpha"], os_["alpha"]) and np.array_equal(s["beta"], os_["beta"])
        for name in ("U", "F"):
            c, e = os_[name]
            want = {tuple(int(x) for x in ee): float(cc) for cc, ee in zip(c, e)}
            assert set(want) == set(s[name])
            for k in want:
                assert s[name][k] == pytest.approx(want[k], rel=1e-14, abs=0)


def test_exported_tables_drive_the_oracle():
    """qmc_tables_export -> Oracle.from_tables evaluates the same numbers as the oracle's own decomposition."""
    wl = qi.massless_box()
    t = q.qmc_prepare(wl, eps_order=0)
    o1 = Oracle.from_tables(t.export())
    o2 = Oracle.from_workload(wl)
    N = 1021
    z = qi.korobov_vector(N, 3, 331)
    sh = qi.splitmix64_shifts(5, 3, 3)
    S1, _, _ = o1.integrate(N, z, sh)
    S2, _, _ = o2.integrate(N, z, sh)
    assert np.allclose(S1, S2, rtol=1e-12, atol=1e-14)


def test_prepare_error_codes():
    wl = qi.massless_box()
    wl.edges = [(0, 1, 0.0), (0, 1, 0.0), (2, 3, 0.0), (2, 3, 0.0)]       # disconnected
    with pytest.raises(q.QmcError) as e:
        q.qmc_prepare(wl)
    assert e.value.status == -1
    wl = qi.massless_box()
    wl.leg_vertex = [0, 1, 2, 7]                                          # leg on a missing vertex
    with pytest.raises(q.QmcError) as e:
        q.qmc_prepare(wl)
    assert e.value.status == -1
    with pytest.raises(q.QmcError) as e:                                  # tree graph: L < 1
        q.qmc_prepare(n_vertices=3, edges=[(0, 1, 0.0), (1, 2, 0.0)], leg_vertex=[0, 2], gram=np.zeros((2, 2)))
    assert e.value.status == -1
    for bad in (dict(transform=3), dict(transform=-1), dict(lattice=2), dict(lam=-0.1)):
        with pytest.raises(q.QmcError) as e:                              # options out of range
            q.qmc_prepare(qi.massless_box(), **bad)
        assert e.value.status == -1
    with pytest.raises(q.QmcError) as e:
        q.qmc_prepare(qi.double_box(), max_depth=2)                       # depth cap
    assert e.value.status == -2
    with pytest.raises(q.QmcError) as e:
        q.qmc_prepare(qi.massless_box(), eps_order=5)                     # kernels instantiated up to eps^2
    assert e.value.status == -3


def test_shift_generator_matches_input_generator():
    assert np.array_equal(q.qmc_shifts(17, 20, 5), qi.splitmix64_shifts(17, 20, 5))


def test_prefactor_series_matches_mpmath():
    mp.mp.dps = 30
    s = -2.0 / 3.0
    got, lo = q.qmc_prefactor_series(2.0, -s, 3.0, 2.0, 3, 2.0, 5)        # e^{2 eps gE} (-s)^{3+2eps} Gamma(3+2eps)
    want = mp.taylor(lambda e: mp.exp(2 * e * mp.euler) * mp.mpf(-s) ** (3 + 2 * e) * mp.gamma(3 + 2 * e), 0, 4)
    assert lo == 0 and np.allclose(got, [float(x) for x in want], rtol=1e-13)
    got, lo = q.qmc_prefactor_series(1.0, 1.0, 0.0, 0.0, 0, 1.0, 4)       # e^{eps gE} Gamma(eps)  (bubble)
    want = mp.taylor(lambda e: e * mp.exp(e * mp.euler) * mp.gamma(e), 0, 3, singular=True)
    assert lo == -1 and np.allclose(got, [float(x) for x in want], rtol=1e-12)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    t = q.qmc_prepare(qi.bubble(), eps_order=1)
    with pytest.raises(q.QmcError) as e:
        q.qmc_integrate(t, 10007, 10, 1)
    assert e.value.status == -4
    # the raw C entry point refuses too (no device => QMC_ECUDA), it never computes on the host
    res = q.binding.qmc_result()
    rc = q.lib().qmc_integrate(t._h, 10007, 10, 1, None, None, 0, ctypes.byref(res))
    assert rc in (-4, -5)


# ---------------------------------------------------------------- component-by-component construction
@pytest.mark.parametrize("N,dim", [(3, 3), (89, 2), (251, 5), (1009, 6), (4093, 6), (8191, 3)])
def test_cbc_vector_matches_oracle_definition(N, dim):
    # product: FFT over the multiplicative group + exact re-evaluation of the closest candidates (qmc_cbc.cpp);
    # oracle: the O(N^2) definition (oracle/cbc.py).  Integer result: bit-exact.  Criterion: a difference of O(1 + e^2)
    # numbers in both, so compared on that scale.
    from oracle.cbc import cbc_vector
    z, e2 = q.qmc_cbc_vector(N, dim, with_criterion=True)
    zo, eo = cbc_vector(N, dim)
    assert np.array_equal(z, zo)
    assert np.all(np.abs(e2 - eo) <= 1e-13 * (1.0 + eo))


def test_cbc_vector_at_a_production_size_is_a_local_optimum():
    # N too large for the O(N^2) oracle: check what holds at any size -- range, coprimality, the reported criterion
    # against the oracle's one-pass definition, and that no sampled candidate for any component beats the chosen one
    from oracle.cbc import criterion
    N, dim = 65521, 6
    z, e2 = q.qmc_cbc_vector(N, dim, with_criterion=True)
    assert z[0] == 1 and np.all(z >= 1) and np.all(z <= (N - 1) // 2)
    for d in range(1, dim + 1):
        assert abs(criterion(N, z[:d]) - e2[d - 1]) <= 1e-12 * (1.0 + e2[d - 1])
    rng = np.random.default_rng(5)
    for d in range(2, dim + 1):
        for c in rng.integers(1, (N - 1) // 2 + 1, size=40):
            assert criterion(N, list(z[:d - 1]) + [int(c)]) >= e2[d - 1] - 1e-11 * (1.0 + e2[d - 1])
    assert np.all(np.diff(e2) > 0)          # every new factor (1 + omega) adds non-negative dual-lattice terms


def test_cbc_vector_error_codes():
    for N, dim in ((1, 2), (2, 2), (91, 3), (1 << 26, 2), (101, 0), (101, 17)):
        with pytest.raises(q.QmcError) as e:
            q.qmc_cbc_vector(N, dim)
        assert e.value.status == -1         # QMC_EINVAL


def test_every_workload_gets_table_driven_tables():
    """A graph the record builders cannot represent silently runs on the (correct, several times slower) generic kernel: the
    parity tests cannot see that.  Every config, the triangle, the Table-1 kinematics and the paper's I_C / I_D (the latter
    needs the larger slot budgets qmc_prepare retries with) must come out of qmc_prepare with table-driven chunks."""
    for wl in qi.CONFIGS() + [qi.triangle(), qi.double_box(-2 / 3, -2 / 3, p2=(0, 0, -1, -1)), qi.paper_IC(), qi.paper_ID()]:
        t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
        lines = t.describe().splitlines()[1:]
        kind = "complex chunk" if wl.lam > 0 else "chunk"
        assert lines and all(l.startswith(kind) for l in lines), (wl.name, t.describe()[:200])
    # a budget that is too small on purpose still falls back (and says so: no chunks)
    t = q.qmc_prepare(qi.double_box(), slot_budget=15, chunk_bytes=1000)
    assert len(t.describe().splitlines()) == 1


def test_propagator_powers_give_the_oracles_sectors_and_run_on_the_generic_kernel():
    """qmc_graph.edge_nu (Eq. 1): exponents of Eq. 6 with N_nu = sum nu_j, x_j^(nu_j - 1) in the integrand.  The
    product's sectors must be the ones of the oracle's own decomposition; the table-driven kernels are compiled for
    nu_j = 1 (exponents functions of n and L), so such tables carry no table images and run on the generic kernel."""
    import dataclasses
    from oracle import Oracle
    for wl in (dataclasses.replace(qi.bubble(-1.0, 1.0, 2.0), nu=(2, 1)),
               dataclasses.replace(qi.massive_box(), nu=(2, 1, 1, 1)),
               dataclasses.replace(qi.massive_box(), nu=(1, 3, 1, 2)),
               dataclasses.replace(qi.bubble(-1.0, 0.0, 0.0), nu=(2, 1)),
               dataclasses.replace(qi.nonplanar_vertex(), nu=(1, 2, 1, 1, 1, 1))):
        t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
        a, b = Oracle.from_tables(t.export()), Oracle.from_workload(wl)
        Nn, L = sum(wl.nu), b.L                      # (the exported tables do not carry the loop number)
        assert (a.aU0, a.aU1, a.aF0, a.aF1) == (Nn - 2 * (L + 1), L + 1, -(Nn - 2 * L), -L) == (b.aU0, b.aU1, b.aF0, b.aF1)
        assert (a.n_sectors, a.k_min, a.k_max) == (b.n_sectors, b.k_min, b.k_max)
        for s in range(a.n_sectors):
            x, y = a.sector(s), b.sector(s)
            assert np.array_equal(x["alpha"], y["alpha"]) and np.array_equal(x["beta"], y["beta"])
            for w in "UF":
                assert np.array_equal(x[w][1], y[w][1]) and np.allclose(x[w][0], y[w][0], rtol=1e-15, atol=0.0)
        d = t.describe()
        assert "real-path tables 0 B" in d and "chunks 0" in d, d
    # the same call with the powers as an argument instead of a workload field
    t = q.qmc_prepare(qi.bubble(-1.0, 1.0, 2.0), eps_order=1, nu=(2, 1))
    assert Oracle.from_tables(t.export()).aF0 == -1
    # sectors that end with alpha = -2, -3 (the p >= 1 Taylor terms of Eq. 11): accepted on the real path, same sectors as the oracle's
    for wl in (dataclasses.replace(qi.bubble(-1.0, 0.0, 0.0), nu=(3, 1)), dataclasses.replace(qi.triangle(), nu=(1, 1, 2)),
               dataclasses.replace(qi.triangle(), nu=(1, 1, 3)), dataclasses.replace(qi.massless_box(), nu=(2, 1, 1, 1))):
        t = q.qmc_prepare(wl, eps_order=wl.eps_order)
        a, b = Oracle.from_tables(t.export()), Oracle.from_workload(wl, taylor=True)
        assert a.status == 0 and b.status == 0 and (a.n_sectors, a.k_min, a.k_max) == (b.n_sectors, b.k_min, b.k_max)
        lowest = 0
        for s in range(a.n_sectors):
            x, y = a.sector(s), b.sector(s)
            assert np.array_equal(x["alpha"], y["alpha"]) and np.array_equal(x["beta"], y["beta"]) and x["n_sing"] == y["n_sing"]
            lowest = min(lowest, int(x["alpha"].min()))
        assert lowest <= -2 and "real-path tables 0 B" in t.describe()
    # refused: alpha = -4, and any alpha <= -2 on the complex path
    for wl, lam in ((dataclasses.replace(qi.bubble(-1.0, 0.0, 0.0), nu=(5, 1)), 0.0),
                    (dataclasses.replace(qi.bubble(-1.0, 0.0, 0.0), nu=(3, 1)), 0.5)):
        with pytest.raises(q.QmcError) as e:
            q.qmc_prepare(wl, lam=lam)
        assert e.value.status == -3
    for bad in ((0, 1), (9, 1), (-1, 1)):
        with pytest.raises(q.QmcError) as e:
            q.qmc_prepare(qi.bubble(), nu=bad)
        assert e.value.status == -1
    with pytest.raises(ValueError):
        q.qmc_prepare(qi.bubble(), nu=(1, 1, 1))
