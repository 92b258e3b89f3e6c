"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded
inputs -- same tables (exported data), same generating vector, same shifts.

Tolerance (reading C19): |S_gpu - S_oracle| <= 1e-12 * max(|S_oracle|, A * 2^-10),
A = the un-cancelled magnitude the oracle accumulates next to S.  Integer counters must match exactly.
"""
import numpy as np
import pytest

import qmc_inputs as qi
import paper_1508_02512_b200 as q
from oracle import Oracle

pytestmark = pytest.mark.gpu

RTOL = 1e-12
NFLOOR = {}      # per parity() call: how many compared values needed the second branch of the C19 tolerance (reported, C19)


def check(got, want, A, what):
    tol = RTOL * np.maximum(np.abs(want), A * 2.0 ** -10)
    bad = np.abs(got - want) > tol
    used_floor = np.abs(want) < A * 2.0 ** -10
    assert not bad.any(), (what, int(bad.sum()), np.abs(got - want)[bad][:5], tol[bad][:5], want[bad][:5])
    return int(used_floor.sum())


def report_floor(key, nfloor, total, worst_kappa):
    """Reading C19: every use of the A-floor is listed.  Printed (pytest -s / the captured log) and written to
    gpurun_out/parity_floor.json at the end of the session (conftest.py); DESIGN.md section 2 quotes the counts."""
    NFLOOR[key] = {"floor": int(nfloor), "of": int(total), "max_kappa": float(worst_kappa)}
    print(f"[C19] {key}: {nfloor} of {total} per-sector values compared against the A-floor, largest A/|S| = {worst_kappa:.3g}")


def parity(wl, N, m, z=None, index_range=None, sectors=None, transform=0, shifts=None, eps_order=None, kernel=0, **layout):
    """`layout`: table-layout fields of qmc_options (slot_budget, chunk_bytes, ...); kernel = 1: the generic kernel."""
    eo = wl.eps_order if eps_order is None else eps_order
    t = q.qmc_prepare(wl, eps_order=eo, lam=wl.lam, transform=transform, **layout)
    o = Oracle.from_tables(t.export())
    if z is None:
        z = qi.good_vector(N, t.dim)
    sh = qi.splitmix64_shifts(wl.seed, m, t.dim) if shifts is None else shifts
    S, A, cnt = o.integrate(N, z, sh, transform=transform, index_range=index_range, sectors=sectors)
    r = q.qmc_integrate(t, N, m, z=z, shifts=sh, index_range=index_range, sectors=sectors, per_sector=True, kernel=kernel)
    assert r.mode_used == 2 and r.shift_sums.shape == S.shape
    nfloor = check(r.shift_sums, S, A, wl.name + " per-sector")
    nz = np.abs(S) > 0
    nu = getattr(wl, "nu", None)
    report_floor(f"{wl.name}{'' if nu is None else ' nu=' + str(tuple(nu))} N={N} m={m} sectors={sectors} idx={index_range} tr={transform} eps={eo} kernel={kernel} {sorted(layout.items())}",
                 nfloor, S.size, float((A[nz] / np.abs(S[nz])).max()) if nz.any() else 0.0)
    assert np.array_equal(r.counters, cnt), (r.counters, cnt)
    # fused mode (the throughput mode): per-shift totals over sectors
    f = q.qmc_integrate(t, N, m, z=z, shifts=sh, index_range=index_range, sectors=sectors, per_sector=False, kernel=kernel)
    assert f.mode_used == 1
    check(f.shift_totals, S.sum(axis=0), A.sum(axis=0), wl.name + " fused")
    check(r.shift_totals, S.sum(axis=0), A.sum(axis=0), wl.name + " per-sector totals")
    # S8: statistics (Eqs. 19-20).  tau_k = the C19 tolerance of the per-shift total T_k.  The mean moves by at most
    # max_k tau_k; the error bar is |d| / sqrt(m (m-1)) with d_k = T_k - mean, and perturbing every T_k by at most tau moves
    # |d| by at most sqrt(m) tau, the error bar by tau / sqrt(m - 1)
    coeff, err = o.totals(S)
    T, AT = S.sum(axis=0), A.sum(axis=0)
    tau = (RTOL * np.maximum(np.abs(T), AT * 2.0 ** -10)).max(axis=-1)        # per order
    for got in (r, f):
        assert np.all(np.abs(got.coeff - coeff) <= tau), (got.coeff, coeff, tau)
        assert np.all(np.abs(got.err.real - err.real) <= tau / np.sqrt(m - 1.0) + 1e-300)
        assert np.all(np.abs(got.err.imag - err.imag) <= tau / np.sqrt(m - 1.0) + 1e-300)
    return r, f, S, A, nfloor


def test_config1_bubble():
    parity(qi.bubble(), 10007, 10)
    parity(qi.bubble(), 10007, 10, eps_order=2)


def test_triangle_double_pole():
    parity(qi.triangle(), 99991, 4)


def test_config2_massless_box():
    r, f, S, A, _ = parity(qi.massless_box(), 99991, 6)
    # closed form within 3 sigma on the GPU result itself (level 2)
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    assert np.all(np.abs(f.coeff.real - ex) <= 3 * f.err.real + 1e-13)


def test_config2_eps1_and_tent_transform():
    parity(qi.massless_box(), 32749, 3, eps_order=1)
    parity(qi.massless_box(), 16381, 3, transform=1)


def test_config3_massive_box_complex():
    r, f, S, A, _ = parity(qi.massive_box(), 99991, 6)
    ref = 0.29347155740583 + 0.33214829595148j       # Gauss-Legendre pin of tests/test_oracle_deformation.py
    assert abs(f.coeff[0].real - ref.real) <= 3 * f.err[0].real and abs(f.coeff[0].imag - ref.imag) <= 3 * f.err[0].imag


def test_config4_double_box_all_sectors_small_N():
    parity(qi.double_box(), 16381, 2)


def test_config4_sector_subset_many_points_per_thread():
    # enough points that every thread walks several lattice indices (grid-stride tail included)
    parity(qi.double_box(), 999983, 2, sectors=(120, 126))


def test_config4_full_size_strided_indices():
    # BASELINE size N = 999983, all 293 sectors, every 61st lattice index
    N = 999983
    parity(qi.double_box(), N, 2, index_range=(7, 61, (N - 7 + 60) // 61))


def test_config5_nonplanar_vertex_complex():
    parity(qi.nonplanar_vertex(), 16381, 4)
    parity(qi.nonplanar_vertex(), 131071, 2, sectors=(20, 28))


def test_config4_full_lattice_all_sectors_at_the_baseline_size():
    """full parity (every sector, every lattice index) at N = 999983 -- two shift vectors (Eq. 20
    needs m >= 2), about two minutes of oracle time on the GPU box's host cores."""
    parity(qi.double_box(), 999983, 2)


def test_contour_counters_nonzero_and_equal():
    """Config 5 at twice its lambda: the deformed contour crosses Re U^(z) <= 0 at some corner evaluations (SURVEY B.6 saw
    2848 in 2e7; reading C21: counted, not fatal).  The integer counters of the CUDA path and of the oracle must be equal
    (parity() asserts that) and non-zero here."""
    r, f, S, A, _ = parity(qi.nonplanar_vertex(lam=0.6), 16381, 4)
    assert r.counters[1] > 0 and f.counters[1] == r.counters[1], r.counters


def test_generic_kernel_parity_on_all_configs():
    """qmc_eval_kernel (version 1, the exponent-table interpreter: qmc_run.kernel = 1) is what runs when the record builders
    cannot represent a graph (complex sectors with more than two singular variables, too many distinct coefficients): the
    same parity bar as the table-driven kernels, on every config, fused and per-sector."""
    parity(qi.bubble(), 10007, 4, kernel=1)
    parity(qi.bubble(), 10007, 4, eps_order=2, kernel=1)
    parity(qi.triangle(), 16381, 3, kernel=1)
    parity(qi.massless_box(), 32749, 4, kernel=1)
    parity(qi.massless_box(), 16381, 3, transform=1, kernel=1)
    parity(qi.massless_box(), 16381, 3, transform=2, eps_order=1, kernel=1)
    parity(qi.massive_box(), 32749, 4, kernel=1)
    parity(qi.double_box(), 16381, 2, sectors=(96, 126), kernel=1)
    parity(qi.nonplanar_vertex(), 16381, 2, kernel=1)
    N = qi.PRIMES[10 ** 8]
    parity(qi.double_box(), N, 2, z=qi.korobov_vector(N, 6, 34567891), index_range=(N - 1 - 65537 * 300, 65537, 301),
           sectors=(200, 230), kernel=1)


def test_generic_kernel_is_the_automatic_path_for_three_singular_complex_variables():
    """The massless planar double box in the PHYSICAL region (s > 0): complex sectors with up to four singular variables.
    The complex table-driven kernel stops at two (QMC3_MAXSING), so qmc_integrate picks the generic kernel by itself."""
    wl = qi.double_box(s=3.0, t=-1.0)
    wl.lam = 0.3
    t = q.qmc_prepare(wl, lam=wl.lam)
    assert t.is_complex and t.k_min == -4
    # sectors [100, 112): one to four singular variables
    r, f, *_ = parity(wl, 10007, 2, sectors=(100, 112))
    g = q.qmc_integrate(t, 10007, 2, z=qi.good_vector(10007, 6), shifts=qi.splitmix64_shifts(wl.seed, 2, 6), sectors=(100, 112), kernel=1)
    assert np.array_equal(g.shift_totals, f.shift_totals)       # the automatic path WAS the generic kernel


def test_builder_failure_falls_back_to_the_generic_kernel():
    """A slot budget too small for the record builder: qmc_prepare must drop every half-built table, and
    qmc_integrate must then run the generic kernel -- never return zeros."""
    wl = qi.double_box()
    t = q.qmc_prepare(wl, slot_budget=15, chunk_bytes=1000)
    assert "chunks 0" in t.describe().splitlines()[0]
    r, f, S, A, _ = parity(wl, 10007, 2, sectors=(110, 118), slot_budget=15, chunk_bytes=1000)
    assert np.abs(f.shift_totals).max() > 0


def test_paper_table1_kinematics():
    parity(qi.double_box(-2 / 3, -2 / 3, p2=(0, 0, -1, -1)), 16381, 2, sectors=(0, 60))


def test_paper_table1_values_from_the_gpu_numbers():
    """Level 2 on the paper's worked example: its Table 1 (fixture tests/golden/paper_table1.txt, the loader
    and the prefactor convention of tests/test_oracle_paper_table1.py) from the library's own run -- qmc_prepare, the library's
    generating vector and seeded shifts, the fused kernels -- at N = 999983: all printed entries of the three mass assignments
    within 4 sigma of the printed values (both columns), with our error at most a tenth of a percent of the value."""
    import mpmath as mp
    from test_oracle_paper_table1 import load_table
    s = t = -2.0 / 3.0
    pref = np.array([float(x) for x in mp.taylor(lambda e: mp.exp(2 * e * mp.euler) * mp.mpf(-s) ** (3 + 2 * e) * mp.gamma(3 + 2 * e), 0, 4)])
    checked = 0
    for legs, table in sorted(load_table().items()):
        tb = q.qmc_prepare(qi.double_box(s, t, p2=legs), eps_order=0)
        m = 8
        r = q.qmc_integrate(tb, 999983, m, seed=101)
        assert not r.counters.any()
        T = r.shift_totals.real                      # [K, m], orders k_min .. 0
        full = np.zeros((5, m))
        full[5 - T.shape[0]:] = T
        for i in range(5):                           # P_i: coefficient of eps^-i, per shift (errors include the correlations)
            k = 4 - i
            Pi = sum(pref[qq] * full[k - qq] for qq in range(k + 1))
            mean, err = Pi.mean(), Pi.std(ddof=1) / np.sqrt(m)
            assert err <= max(1e-3 * abs(table[i][1][0]), 1e-6), (legs, i, err)
            for val, perr in table[i]:
                assert abs(mean - val) <= 4.0 * np.hypot(err, perr) + 1e-5 * max(1.0, abs(val)), (legs, i, mean, err, val, perr)
                checked += 1
    assert checked == 30


def test_edge_cases_boundary_points_and_tiny_lattices():
    wl = qi.massless_box()
    # a zero shift component puts lattice index 0 on the boundary: contributes exactly 0, counted
    sh = qi.splitmix64_shifts(3, 3, 3)
    sh[1, 2] = 0.0
    r, f, S, A, _ = parity(wl, 1021, 3, z=qi.korobov_vector(1021, 3, 331), shifts=sh)
    assert r.counters[3] == 1
    parity(wl, 5, 2, z=np.array([1, 2, 3], dtype=np.uint64))
    parity(wl, 257, 2, z=qi.korobov_vector(257, 3, 3))


def test_invalid_arguments():
    t = q.qmc_prepare(qi.massless_box())
    with pytest.raises(q.QmcError) as e:
        q.qmc_integrate(t, 1000, 4, z=[1, 10, 100])          # z_j not coprime to N
    assert e.value.status == -1
    with pytest.raises(q.QmcError) as e:
        q.qmc_integrate(t, 1021, 1)                          # Eq. 20 needs m >= 2
    assert e.value.status == -1


def test_library_generating_vector_and_seeded_shifts():
    t = q.qmc_prepare(qi.massless_box())
    N = 99991
    z = q.qmc_generating_vector(N, 3)
    assert z[0] == 1 and all(np.gcd(int(v), N) == 1 for v in z)
    assert int(z[2]) == (int(z[1]) * int(z[1])) % N          # Korobov form
    a = q.qmc_integrate(t, N, 8, seed=7)
    b = q.qmc_integrate(t, N, 8, z=z, shifts=qi.splitmix64_shifts(7, 8, 3))
    assert np.array_equal(a.shift_totals, b.shift_totals)     # deterministic, same inputs
    c = q.qmc_integrate(t, N, 8, seed=7)
    assert np.array_equal(a.shift_totals, c.shift_totals)     # run-to-run bit reproducible
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    assert np.all(np.abs(a.coeff.real - ex) <= 3.5 * a.err.real)
    assert np.all(a.err.real < 1e-5)


def test_double_box_poles_on_gpu_at_baseline_size():
    """Level 2 at a BASELINE.json size: N = 999983, m = 20, seed 13, fused mode (the bench configuration)."""
    t = q.qmc_prepare(qi.double_box())
    r = q.qmc_integrate(t, 999983, 20, seed=13)
    ex = [2.0 / 9.0, -0.8497687147780183, 0.003001503361321066]     # tests/test_oracle_closed_forms.py (mpmath)
    assert np.all(np.abs(r.coeff.real[:3] - ex) <= 3.5 * r.err.real[:3])
    assert np.all(r.err.real < [1e-6, 1e-5, 1e-4, 1e-3, 1e-2])
    assert not r.counters.any()
    # fused and per-sector modes agree at full size
    p = q.qmc_integrate(t, 999983, 20, seed=13, per_sector=True)
    assert np.allclose(p.shift_totals, r.shift_totals, rtol=1e-11, atol=1e-13)


def test_real_path_tables_chunk_boundaries_slot_budget_and_launch_splits():
    """Real-path tables (version 4: one launch per run of sectors, tables in the kernel parameters): sector ranges that
    straddle chunk boundaries, a slot budget small enough to force sector-local product slots and chunk splits, and
    chunks larger than what one launch can carry (qmc_options.slot_budget / chunk_bytes)."""
    wl = qi.double_box()
    t = q.qmc_prepare(wl)
    desc = t.describe()
    assert "chunks" in desc and t.n_sectors == 293
    bounds = [int(l.split("[")[1].split(",")[0]) for l in desc.splitlines()[1:]]
    assert len(bounds) > 2
    b = bounds[2]
    parity(wl, 16381, 2, sectors=(b - 3, b + 4))            # straddles a chunk boundary
    parity(wl, 16381, 2, sectors=(bounds[1] - 1, bounds[3] + 1))   # spans a whole chunk plus both neighbours
    t2 = q.qmc_prepare(wl, slot_budget=26, chunk_bytes=3000)
    d2 = t2.describe()
    assert sum(int(l.split("local products ")[1].split(" ")[0]) for l in d2.splitlines()[1:]) > 0
    assert len(d2.splitlines()) > len(desc.splitlines())
    parity(wl, 16381, 2, sectors=(100, 140), slot_budget=26, chunk_bytes=3000)
    t3 = q.qmc_prepare(wl, chunk_bytes=60000)             # a chunk now exceeds the 28 KB of tables one launch carries
    nchunks3 = sum(int(l.split("[")[1].split(",")[0]) < 150 for l in t3.describe().splitlines()[1:])   # chunks meeting [0, 150)
    r3, f3, *_ = parity(wl, 16381, 2, sectors=(0, 150), chunk_bytes=60000)
    assert f3.kernel_launches - 2 > nchunks3                # the launcher split chunks into several runs
    parity(wl, 16381, 2, sectors=(100, 140), threads=128)   # the other block size of the kernel


def test_async_launch_resident_inputs_and_fetch():
    """qmc_integrate_async with everything resident (the bench's device-timed step) gives bit-identical results to the
    synchronous call, and the device view of the per-shift totals matches what fetch returns."""
    import torch
    wl = qi.massless_box()
    t = q.qmc_prepare(wl)
    N, m = 99991, 8
    z = qi.good_vector(N, 3)
    sh = qi.splitmix64_shifts(wl.seed, m, 3)
    ref = q.qmc_integrate(t, N, m, z=z, shifts=sh)
    q.qmc_integrate_async(t, N, m, z=z, shifts=sh, resident=0)
    q.qmc_integrate_async(t, N, m, z=z, resident=2)          # nothing copied from the host
    dev = q.qmc_result_device_totals(t, m)
    r = q.qmc_result_fetch(t, m)
    assert np.array_equal(r.shift_totals, ref.shift_totals) and np.array_equal(r.coeff, ref.coeff)
    torch.cuda.synchronize()
    d = dev.cpu().numpy()
    assert np.array_equal(d[..., 0] + 1j * d[..., 1], ref.shift_totals)
    assert r.h2d_bytes < ref.h2d_bytes and r.d2h_bytes > 0 and r.eval_kernel_ms > 0


def test_complex_path_tables_launch_splits_and_local_slots():
    """Complex-path tables (version 5): small chunks (several launches per step, sector ranges that straddle them) and
    slot budgets small enough to force sector-local real and complex product slots (qmc_options.chunk_bytes,
    slot_budget_cplx_real, slot_budget_cplx)."""
    wl = qi.nonplanar_vertex()
    t = q.qmc_prepare(wl, lam=wl.lam)
    n0 = len(t.describe().splitlines())
    lay = dict(chunk_bytes=6000, slot_budget_cplx_real=26, slot_budget_cplx=10)
    t2 = q.qmc_prepare(wl, lam=wl.lam, **lay)
    d2 = t2.describe()
    assert len(d2.splitlines()) > n0 and "local) complex slots 10 (+" in d2 and "(+0 local) tables" not in d2.splitlines()[1]
    r, f, *_ = parity(wl, 16381, 2, sectors=(3, 31), **lay)
    assert f.kernel_launches - 2 >= 3


def test_kinematic_scan_points_of_the_papers_box():
    """three points of the paper's s-scan of the one-loop box: parity with the oracle,
    a vanishing imaginary part below the threshold s = 4 M_t^2, and lambda-independence above it."""
    pts = dict((round(s), wl) for s, wl in qi.gghh_box_scan(44))     # s = 70000, 80000, ..., 500000
    below, above = pts[110000], pts[200000]
    r, *_ = parity(below, 16381, 4)
    assert abs(r.coeff[-1].imag) < 5 * r.err[-1].imag + 1e-9 and r.coeff[-1].real > 0
    parity(above, 16381, 4)
    N, m = 99991, 16
    z = qi.good_vector(N, 3)
    vals = []
    for lam in (0.25, 0.5):
        t = q.qmc_prepare(above, eps_order=0, lam=lam)
        vals.append(q.qmc_integrate(t, N, m, z=z, seed=11))
    d = vals[0].coeff[-1] - vals[1].coeff[-1]
    sig = np.hypot(abs(vals[0].err[-1]), abs(vals[1].err[-1]))
    assert abs(d) < 6 * sig and abs(vals[0].coeff[-1].imag) > 0.1
    assert not vals[0].counters[:2].any() and not vals[1].counters[:2].any()


@pytest.mark.parametrize("which", ["table2_IC", "table3_ID"])
def test_paper_tables_2_and_3_on_gpu(which):
    """the paper's own two-loop integrals in the physical region (Eqs. 25, 27; Tables 2, 3):
    per-sector parity with the oracle at a small lattice, then the printed P_2, P_1, P_0 at N = 1048573."""
    from test_oracle_paper_table23 import compare, laurent_P, load_table
    wl, table = (qi.paper_IC(), load_table("paper_table2.txt")) if which == "table2_IC" else (qi.paper_ID(), load_table("paper_table3.txt"))
    parity(wl, 16381, 2, sectors=(0, 12))
    parity(wl, 16381, 2, sectors=(30, 46))
    t = q.qmc_prepare(wl, eps_order=0, lam=wl.lam)
    assert (t.k_min, t.k_max, t.is_complex) == (-2, 0, True)
    r = q.qmc_integrate(t, 1048573, 20, seed=5)
    assert r.counters[0] == 0 and r.counters[2] == 0
    P = laurent_P(r.shift_totals, wl.meta["s_over_mt2"])
    assert max(P[0][1], P[0][2]) / abs(P[0][0]) < 2e-3          # the finite part to the paper's O(1e-3)
    compare(P, table, 5.0)


def test_cbc_generating_vectors_through_the_kernels():
    """the library's component-by-component vectors drive the same kernels -- parity
    against the oracle on the massless box and the non-planar vertex, closed form of the box within 3 sigma."""
    N = 65521
    z3 = q.qmc_cbc_vector(N, 3)
    r, f, S, A, _ = parity(qi.massless_box(), N, 6, z=z3)
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    assert np.all(np.abs(f.coeff.real - ex) <= 3.5 * f.err.real + 1e-13)
    parity(qi.nonplanar_vertex(), 16381, 3, z=q.qmc_cbc_vector(16381, 5))
    # qmc_options.lattice = 1: qmc_integrate builds (and caches) the CBC vector itself
    t = q.qmc_prepare(qi.massless_box(), lattice=1)
    a = q.qmc_integrate(t, N, 6, seed=7)
    b = q.qmc_integrate(q.qmc_prepare(qi.massless_box()), N, 6, z=z3, shifts=qi.splitmix64_shifts(7, 6, 3))
    assert np.array_equal(a.shift_totals, b.shift_totals)
    with pytest.raises(q.QmcError) as e:
        q.qmc_integrate(t, 65535, 6, seed=7)              # CBC needs a prime N
    assert e.value.status == -1


def test_second_order_periodising_transform_on_gpu():
    """transform = 2 (the r = 2 member of Eq. 21's family, R:C20) through all three kernels: real path (box, double-box
    sector subset), complex path (massive box), and the closed form of the box within 3.5 sigma."""
    r, f, S, A, _ = parity(qi.massless_box(), 65521, 6, transform=2)
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    assert np.all(np.abs(f.coeff.real - ex) <= 3.5 * f.err.real + 1e-13)
    parity(qi.massive_box(), 16381, 3, transform=2)
    parity(qi.double_box(), 10007, 2, transform=2, sectors=(100, 130))


def test_maximum_baseline_sizes_strided_indices():
    """The largest lattices BASELINE.json names (cfg4: N = 99999989, cfg2 / cfg3: N = 9999991): i * z_j reaches 2^53, so
    the remainder must be integer arithmetic on both sides.  Sampled outputs: a strided subset of the
    lattice indices that the oracle can compute one by one, all sectors, the launch geometry of the full rule."""
    N = qi.PRIMES[10 ** 8]
    z = qi.korobov_vector(N, 6, 34567891)
    step = 65537
    parity(qi.double_box(), N, 2, z=z, index_range=(N - 1 - step * 1500, step, 1501))   # includes the last index N - 1
    N = qi.PRIMES[10 ** 7]
    z = qi.korobov_vector(N, 3, 2345677)
    parity(qi.massless_box(), N, 3, z=z, index_range=(5, 4099, (N - 5 + 4098) // 4099))
    parity(qi.massive_box(), N, 2, z=z, index_range=(11, 8191, (N - 11 + 8190) // 8191))


def test_index_blocks_of_two_ranks_add_to_the_full_lattice():
    """the lattice split into contiguous index ranges (sharding.index_block) -- the two half-sums, each
    normalised by 1/N, add to the single-rank totals within the C19 tolerance (here: evaluated one after the other on one
    GPU; the all_reduce itself is covered by tests/test_multi_rank.py)."""
    from paper_1508_02512_b200 import sharding
    wl = qi.double_box()
    t = q.qmc_prepare(wl)
    N, m = 131071, 4
    z = qi.korobov_vector(N, 6, 60941)
    sh = qi.splitmix64_shifts(wl.seed, m, 6)
    full = q.qmc_integrate(t, N, m, z=z, shifts=sh)
    parts = [q.qmc_integrate(t, N, m, z=z, shifts=sh, index_range=sharding.index_block(N, r, 2)) for r in range(2)]
    tot = parts[0].shift_totals + parts[1].shift_totals
    scale = np.abs(parts[0].shift_totals) + np.abs(parts[1].shift_totals)
    assert np.all(np.abs(tot - full.shift_totals) <= 1e-12 * np.maximum(np.abs(full.shift_totals), scale))
    coeff, err = q.qmc_statistics(tot)
    assert np.allclose(coeff, full.coeff, rtol=1e-11, atol=1e-14)


def test_embedded_lattice_sequence():
    """SURVEY 8(f) f4, reading C26: lattices N = 2^k that share one generating vector with odd components.  (1) the library's
    vector: odd, Korobov form; (2) the odd-index half of a level against the oracle (per sector, C19 tolerance); (3) walking up
    the levels (each evaluating only its new points) gives the estimate of a direct run at N = 2^k on the same vector and
    shifts; (4) the early stop; on the real path and on the complex path."""
    z = q.qmc_embedded_vector(10, 18, 3)
    assert all(int(v) & 1 for v in z) and int(z[2]) == (int(z[1]) * int(z[1])) % (1 << 18)
    for wl, zz in ((qi.massless_box(), z), (qi.massive_box(), z)):
        N = 1 << 12
        parity(wl, N, 3, z=zz % N, index_range=(1, 2, N // 2))                 # the new points of level 12
        t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
        m = 8
        r, k, npts = q.qmc_integrate_embedded(t, 10, 15, m, wl.seed, zz)        # target 0: runs to k_max
        assert (k, npts) == (15, 1 << 15)
        d = q.qmc_integrate(t, 1 << 15, m, z=zz % (1 << 15), seed=wl.seed)      # all 2^15 points in one go
        scale = np.maximum(np.abs(d.shift_totals), np.abs(d.shift_totals).max())
        assert np.all(np.abs(r.shift_totals - d.shift_totals) <= 1e-12 * scale)
        assert np.allclose(r.coeff, d.coeff, rtol=1e-11, atol=1e-14) and np.allclose(r.err.real, d.err.real, rtol=1e-6, atol=1e-16)
        r2, k2, n2 = q.qmc_integrate_embedded(t, 10, 18, m, wl.seed, zz, target_rel_err=1e-5)
        c0, e0 = r2.coeff[-1], r2.err[-1]
        assert k2 < 18 and n2 == 1 << k2 and max(e0.real, e0.imag) <= 1e-5 * abs(c0)
    with pytest.raises(q.QmcError):
        q.qmc_integrate_embedded(q.qmc_prepare(qi.massless_box()), 10, 12, 4, 1, np.array([1, 2, 5], dtype=np.uint64))   # even component


def test_sector_mask_selects_sectors_in_fused_mode():
    """qmc_run.sector_mask: a fused launch that serves an arbitrary subset of sectors -- the per-shift totals are the sum of
    the oracle's per-sector values over the selected sectors (C19 tolerance); real path, complex path, empty chunks; the
    generic kernel refuses masks."""
    rng = np.random.default_rng(3)
    for wl, N in ((qi.double_box(), 16381), (qi.nonplanar_vertex(), 16381)):
        t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
        o = Oracle.from_tables(t.export())
        z = qi.good_vector(N, t.dim)
        sh = qi.splitmix64_shifts(wl.seed, 2, t.dim)
        S, A, cnt = o.integrate(N, z, sh)
        for mask in (rng.random(t.n_sectors) < 0.3, np.arange(t.n_sectors) % 7 == 3, np.arange(t.n_sectors) >= t.n_sectors - 2):
            r = q.qmc_integrate(t, N, 2, z=z, shifts=sh, sector_mask=mask.astype(np.uint8))
            check(r.shift_totals, S[mask].sum(axis=0), A[mask].sum(axis=0), wl.name + " masked")
        with pytest.raises(q.QmcError) as e:
            q.qmc_integrate(t, N, 2, z=z, shifts=sh, sector_mask=np.ones(t.n_sectors, dtype=np.uint8), kernel=1)
        assert e.value.status == -3


def test_per_sector_lattice_sizes_by_variance():
    """SURVEY 8(f) f4, reading C27 (qmc_integrate_allocated): sizes differ between sectors, the target is met, the result agrees
    with the uniform embedded sequence within errors and with the closed forms (how the evaluation counts compare depends on
    the target: bench.py reports it, `allocation_vs_uniform`)."""
    wl = qi.double_box()
    t = q.qmc_prepare(wl)
    z = q.qmc_embedded_vector(12, 22, 6)
    r, lev, ev = q.qmc_integrate_allocated(t, 13, 22, wl.m, wl.seed, z, 2e-4)
    u, k, npts = q.qmc_integrate_embedded(t, 13, 22, wl.m, wl.seed, z, target_rel_err=2e-4)
    assert r.err[-1].real <= 2e-4 * abs(r.coeff[-1]) and lev.min() >= 13 and lev.max() > lev.min() + 3
    assert ev >= t.n_sectors << 13                                                   # stage 1 alone
    assert abs(r.coeff[-1] - u.coeff[-1]) <= 4 * np.hypot(r.err[-1].real, u.err[-1].real)
    ex = [2.0 / 9.0, -0.8497687147780183, 0.003001503361321066]                     # the three analytic poles
    assert np.all(np.abs(r.coeff.real[:3] - ex) <= 4 * r.err.real[:3])
    wl = qi.massless_box()
    t = q.qmc_prepare(wl)
    r, lev, ev = q.qmc_integrate_allocated(t, 10, 20, wl.m, wl.seed, q.qmc_embedded_vector(10, 20, 3), 1e-7)
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    assert np.all(np.abs(r.coeff.real - ex) <= 4 * r.err.real) and r.err[-1].real <= 1e-7 * abs(r.coeff[-1])
    wl = qi.massive_box()                                                            # complex path
    t = q.qmc_prepare(wl, lam=wl.lam)
    r, lev, ev = q.qmc_integrate_allocated(t, 10, 20, wl.m, wl.seed, q.qmc_embedded_vector(10, 20, 3), 1e-6)
    ref = 0.29347155740583 + 0.33214829595148j
    assert abs(r.coeff[0].real - ref.real) <= 4 * r.err[0].real and abs(r.coeff[0].imag - ref.imag) <= 4 * r.err[0].imag


def test_batched_kinematic_points():
    """kinematic points as a batch (qmc_prepare_batch + qmc_run.mode = 3): ONE call evaluates all points.  Per
    point and per shift the batch result equals the oracle's totals of that point (its own decomposition at that point's
    kinematics; C19 tolerance), and the result of the one-call-per-point path to the same tolerance (the two split the lattice
    into different numbers of slices, so the partial sums group differently) -- complex path (the paper's box scan, points on
    both sides of the threshold) and real path (the massless box at four kinematic points)."""
    N, m = 16381, 4
    z = qi.good_vector(N, 3)
    for pts, lam, seed in (([wl for s, wl in qi.gghh_box_scan(44)][2:9], 0.5, 11),
                           ([qi.massless_box(-3, -2), qi.massless_box(-1, -1), qi.massless_box(-2, -5), qi.massless_box(-0.3, -4)], 0.0, 7)):
        sh = qi.splitmix64_shifts(seed, m, 3)
        t = q.qmc_prepare_batch(pts, lam=lam)
        assert t.n_points == len(pts) and t.n_sectors == t.n_points * t.sectors_per_point
        r = q.qmc_integrate(t, N, m, z=z, shifts=sh, mode=3)
        assert r.mode_used == 3 and r.shift_sums.shape == (len(pts), t.K, m)
        for p, wl in enumerate(pts):
            o = Oracle.from_workload(wl, lam=lam)
            S, A, cnt = o.integrate(N, z, sh)
            check(r.shift_sums[p], S.sum(axis=0), A.sum(axis=0), f"{wl.name} point {p}")
            one = q.qmc_integrate(q.qmc_prepare(wl, lam=lam), N, m, z=z, shifts=sh)
            check(one.shift_totals, r.shift_sums[p], A.sum(axis=0), f"{wl.name} point {p}: one call per point")
            assert np.allclose(one.coeff, r.sector_coeff[p], rtol=1e-11, atol=1e-13 * np.abs(A).max())
    with pytest.raises(q.QmcError):
        q.qmc_integrate(t, N, m, z=z, shifts=sh, mode=3, sectors=(0, 4))         # a batch is integrated as a whole


def test_resident_shifts_are_keyed_by_their_seed():
    """with tables_resident = 2 a different seed must not silently reuse the previous call's shift vectors."""
    wl = qi.massless_box()
    t = q.qmc_prepare(wl)
    N, m = 16381, 4
    z = qi.good_vector(N, 3)
    a7 = q.qmc_integrate(t, N, m, z=z, seed=7)
    q.qmc_integrate_async(t, N, m, z=z, seed=7, resident=0)
    q.qmc_integrate_async(t, N, m, z=z, seed=8, resident=2)              # another seed: re-generated, not reused
    r8 = q.qmc_result_fetch(t, m)
    a8 = q.qmc_integrate(t, N, m, z=z, seed=8)
    assert np.array_equal(r8.shift_totals, a8.shift_totals) and not np.array_equal(r8.shift_totals, a7.shift_totals)
    q.qmc_integrate_async(t, N, m, z=z, seed=8, resident=2)              # the same seed: reused (nothing but the tables travels)
    r8b = q.qmc_result_fetch(t, m)
    assert np.array_equal(r8b.shift_totals, a8.shift_totals) and r8b.h2d_bytes < r8.h2d_bytes


def test_two_ranks_on_two_gpus():
    """the N > 1 path on hardware -- skipped unless two GPUs are visible (one GPU per call on this pool; the
    sharding logic itself is covered by the world-size-2 gloo tests)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    from paper_1508_02512_b200 import sharding
    wl = qi.massless_box()
    N, m = 99991, 4
    z = qi.good_vector(N, 3)
    full = q.qmc_integrate(q.qmc_prepare(wl), N, m, z=z, seed=wl.seed, device="cuda:0")
    parts = [q.qmc_integrate(q.qmc_prepare(wl), N, m, z=z, seed=wl.seed, index_range=sharding.index_block(N, r, 2), device=f"cuda:{r}")
             for r in range(2)]
    tot = parts[0].shift_totals + parts[1].shift_totals
    assert np.allclose(tot, full.shift_totals, rtol=1e-11, atol=1e-13)


def test_propagator_powers_run_on_the_generic_kernel():
    """qmc_graph.edge_nu (Eq. 1): N_nu = sum nu_j in the exponents of Eq. 6, x_j^(nu_j - 1) in the integrand.  The
    table-driven kernels have their exponents compiled in for nu_j = 1; other powers run on the generic kernel by themselves.
    Parity against the oracle on the product's tables (that these are the sectors of the oracle's own decomposition is a CPU
    test: tests/test_product_host.py), and two closed forms on the GPU numbers."""
    import dataclasses
    import mpmath as mp
    # real path, no singular variable: massive bubble with a squared propagator against the simplex form of the parameter integral
    p2, m1, m2 = -1.3, 1.0, 2.5
    wl = dataclasses.replace(qi.bubble(p2, m1, m2), nu=(2, 1), eps_order=2)
    r, f, S, A, _ = parity(wl, 10007, 6)
    assert "real-path tables 0 B" in q.qmc_prepare(wl, eps_order=2).describe()
    F = lambda x: -p2 * x * (1 - x) + m1 * x + m2 * (1 - x)
    want = [float(mp.quad(lambda x: x * F(x) ** (2 - 3) * (-mp.log(F(x))) ** k / mp.factorial(k), [0, 1])) for k in range(3)]
    assert np.all(np.abs(f.coeff.real - want) <= 4 * f.err.real + 1e-12), (f.coeff.real, f.err.real, want)
    # real path, one pole: massless propagator with powers (2, 1): J = (-p^2)^(-1-eps) B(-eps, 1-eps)
    wl = dataclasses.replace(qi.bubble(-1.7, 0.0, 0.0), nu=(2, 1), eps_order=1)
    r, f, S, A, _ = parity(wl, 32749, 6)
    g = lambda x: mp.mpf(1.7) ** (-1 - x) * mp.beta(-x, 1 - x)
    rad, npts = 0.25, 64
    vals = [g(rad * mp.e ** (2j * mp.pi * i / npts)) for i in range(npts)]
    want = [float((sum(v * mp.e ** (-2j * mp.pi * i * k / npts) for i, v in enumerate(vals)) / npts / rad ** k).real) for k in (-1, 0, 1)]
    assert np.all(np.abs(f.coeff.real - want) <= 4 * f.err.real + 1e-12), (f.coeff.real, f.err.real, want)
    # complex path (physical region): the massive box of config 3 with squared and cubed propagators
    parity(dataclasses.replace(qi.massive_box(), nu=(2, 1, 1, 1)), 32749, 3)
    parity(dataclasses.replace(qi.massive_box(), nu=(1, 3, 1, 2)), 16381, 2)
    # two loops, complex path with a pole: the non-planar vertex of config 5 with a squared propagator, a third of its sectors
    parity(dataclasses.replace(qi.nonplanar_vertex(), nu=(1, 2, 1, 1, 1, 1)), 16381, 2, sectors=(0, 12))


def _laurent(f, kmin, kmax, radius=0.25, npts=64):
    """Laurent coefficients of f around eps = 0 by the trapezoidal rule on a circle (mpmath)."""
    import mpmath as mp
    vals = [f(radius * mp.e ** (2j * mp.pi * i / npts)) for i in range(npts)]
    return np.array([float((sum(v * mp.e ** (-2j * mp.pi * i * k / npts) for i, v in enumerate(vals)) / npts / radius ** k).real)
                     for k in range(kmin, kmax + 1)])


def test_taylor_terms_for_alpha_below_minus_one_on_the_generic_kernel():
    """SURVEY 8(f) f3, reading C28: sectors with a variable of exponent alpha_j = -2 or -3 (they come with propagator powers)
    need the p >= 1 Taylor terms of Eq. 11.  The generic kernel evaluates them in product form with
    truncated power series in the variables set to zero (sector_eval_taylor); the oracle evaluates the expanded double sum.
    Parity per sector, order and shift at the C19 tolerance; closed forms on the GPU numbers with the tent transform (under
    Eq. 21's transform the subtraction at alpha = -2 is numerically unstable on BOTH sides, DESIGN.md section 10 f3)."""
    import dataclasses
    import mpmath as mp
    # massless propagator with powers (3, 1): J = (-p^2)^(D/2-4) B(D/2-3, D/2-1)
    wl = dataclasses.replace(qi.bubble(-1.7, 0.0, 0.0), nu=(3, 1), eps_order=1)
    assert "real-path tables 0 B" in q.qmc_prepare(wl, eps_order=1).describe()
    r, f, S, A, _ = parity(wl, 65521, 8, transform=1)
    want = _laurent(lambda x: mp.mpf(1.7) ** (-2 - x) * mp.beta(-1 - x, 1 - x), -1, 1)
    assert np.all(np.abs(f.coeff.real - want) <= 4 * f.err.real + 1e-11), (f.coeff.real, f.err.real, want)
    parity(wl, 16381, 3)                                   # Eq. 21's transform: the two sides still agree
    parity(wl, 16381, 3, transform=2)
    # triangle with a squared propagator: sectors with exponents (-2, -2) and (-2, -1); Dirichlet's integral
    s = -2.0
    for nu in ((2, 1, 1), (1, 1, 2)):
        wl = dataclasses.replace(qi.triangle(s), nu=nu, eps_order=0)
        r, f, S, A, _ = parity(wl, 99991, 8, transform=1)
        Nn = sum(nu)
        want = _laurent(lambda x: (-s) ** (2 - x - Nn) * mp.gamma(nu[0]) * mp.gamma(nu[1] + 2 - x - Nn) * mp.gamma(nu[2] + 2 - x - Nn)
                        / mp.gamma(4 - 2 * x - Nn), -2, 0)
        assert np.all(np.abs(f.coeff.real - want) <= 4 * f.err.real + 1e-11), (nu, f.coeff.real, f.err.real, want)
    parity(dataclasses.replace(qi.triangle(s), nu=(1, 1, 2), eps_order=1), 16381, 3)
    # alpha = -3 (two regular Taylor terms and the pole)
    parity(dataclasses.replace(qi.triangle(s), nu=(1, 1, 3)), 16381, 3, transform=1)
    # three variables: the massless box of config 2 with squared propagators, sectors with two such variables
    parity(dataclasses.replace(qi.massless_box(), nu=(2, 1, 1, 1)), 16381, 3, transform=1)
    parity(dataclasses.replace(qi.massless_box(), nu=(1, 2, 1, 2), eps_order=1), 16381, 2, transform=1)
    # refused: alpha = -4; the complex path
    for wl in (dataclasses.replace(qi.bubble(-1.0, 0.0, 0.0), nu=(5, 1)),
               dataclasses.replace(qi.bubble(-1.0, 0.0, 0.0), nu=(3, 1), lam=0.5)):
        with pytest.raises(q.QmcError) as e:
            q.qmc_prepare(wl, lam=wl.lam)
        assert e.value.status == -3


def test_pole_extraction_by_integration_by_parts():
    """SURVEY 8(f) f3, reading C30: qmc_options.pole_extraction = 1 extracts the poles by Eq. 13 instead of the
    subtraction.  Parity per sector, order and shift against the oracle's own IBP (sector_point_ibp) on the product's tables;
    the closed forms on the GPU numbers; the cancellation factor the paper introduces IBP for."""
    import dataclasses
    import mpmath as mp
    # one-loop massless box: three variables, up to two singular ones; closed form
    r, f, S, A, _ = parity(qi.massless_box(), 32749, 6, pole_extraction=1)
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    assert np.all(np.abs(f.coeff.real - ex) <= 4 * f.err.real + 1e-12), (f.coeff.real, f.err.real)
    T, AT = S.sum(axis=0), A.sum(axis=0)
    assert (AT / np.abs(T)).max() < 100.0
    parity(qi.massless_box(), 16381, 3, pole_extraction=1, eps_order=1, transform=1)
    parity(qi.triangle(), 32749, 4, pole_extraction=1)
    parity(qi.bubble(), 10007, 4, pole_extraction=1)                      # no singular variable: nothing to extract
    # variables with alpha = -2, -3: Eq. 13 two and three times; Eq. 21's transform throughout
    wl = dataclasses.replace(qi.bubble(-1.7, 0.0, 0.0), nu=(3, 1), eps_order=1)
    r, f, S, A, _ = parity(wl, 65521, 8, pole_extraction=1)
    want = _laurent(lambda x: mp.mpf(1.7) ** (-2 - x) * mp.beta(-1 - x, 1 - x), -1, 1)
    assert np.all(np.abs(f.coeff.real - want) <= 4 * f.err.real + 1e-9), (f.coeff.real, f.err.real, want)
    s = -2.0
    for nu in ((2, 1, 1), (1, 1, 2)):
        wl = dataclasses.replace(qi.triangle(s), nu=nu, eps_order=0)
        r, f, S, A, _ = parity(wl, 99991, 8, pole_extraction=1)
        Nn = sum(nu)
        want = _laurent(lambda x: (-s) ** (2 - x - Nn) * mp.gamma(nu[0]) * mp.gamma(nu[1] + 2 - x - Nn) * mp.gamma(nu[2] + 2 - x - Nn)
                        / mp.gamma(4 - 2 * x - Nn), -2, 0)
        assert np.all(np.abs(f.coeff.real - want) <= 4 * f.err.real + 1e-9), (nu, f.coeff.real, f.err.real, want)
        T, AT = S.sum(axis=0), A.sum(axis=0)
        assert (AT / np.maximum(np.abs(T), 1e-300)).max() < 100.0      # the subtraction: 1e14 on the same graph (profiles/r02e_parity_floor.json)
    parity(dataclasses.replace(qi.triangle(s), nu=(1, 1, 3)), 16381, 3, pole_extraction=1)
    parity(dataclasses.replace(qi.massless_box(), nu=(2, 1, 1, 1)), 16381, 2, pole_extraction=1)
    # two loops: sectors of the double box with two, three and four singular variables (16 Taylor coefficients)
    parity(qi.double_box(), 16381, 2, sectors=(118, 126), pole_extraction=1)
    # refused: the complex path; a sector whose series would need more than 16 coefficients
    with pytest.raises(q.QmcError) as e:
        q.qmc_prepare(qi.massive_box(), lam=0.5, pole_extraction=1)
    assert e.value.status == -3
    with pytest.raises(q.QmcError) as e:
        q.qmc_prepare(dataclasses.replace(qi.massless_box(), nu=(3, 3, 1, 1)), pole_extraction=1)
    assert e.value.status == -3
    with pytest.raises(q.QmcError) as e:
        q.qmc_prepare(qi.massless_box(), pole_extraction=2)
    assert e.value.status == -1


def test_geometric_decomposition_strategy():
    """SURVEY 8(f) f3, reading C31: qmc_options.strategy = 1 decomposes by the geometric method (one monomial substitution per
    simplicial cone of the normal fan of the Newton polyhedron).  The sectors are different ones (266 instead of 293 on the double
    box), the kernels the same: parity per sector on both paths, the closed forms on the GPU numbers, and -- totals do not
    depend on the strategy (reading C23) -- agreement with the iterated strategy on all five orders of the double box."""
    r, f, S, A, _ = parity(qi.massless_box(), 32749, 4, strategy=1)
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]
    assert np.all(np.abs(f.coeff.real - ex) <= 4 * f.err.real + 1e-13)
    parity(qi.massive_box(), 32749, 3, strategy=1)
    parity(qi.double_box(), 16381, 2, sectors=(0, 40), strategy=1)
    parity(qi.double_box(), 16381, 2, sectors=(226, 266), strategy=1)
    parity(qi.double_box(), 10007, 2, sectors=(150, 170), strategy=1, kernel=1)
    parity(qi.nonplanar_vertex(), 16381, 2, sectors=(18, 36), strategy=1)
    parity(qi.paper_IC(), 16381, 2, sectors=(30, 46), strategy=1)
    tg, ti = q.qmc_prepare(qi.double_box(), strategy=1), q.qmc_prepare(qi.double_box(), strategy=0)
    assert (tg.n_sectors, ti.n_sectors) == (266, 293)
    rg, ri = q.qmc_integrate(tg, 999983, 8, seed=13), q.qmc_integrate(ti, 999983, 8, seed=13)
    ex4 = [2.0 / 9.0, -0.8497687147780183, 0.003001503361321066]
    assert np.all(np.abs(rg.coeff.real[:3] - ex4) <= 4 * rg.err.real[:3]), (rg.coeff.real, rg.err.real)
    assert np.all(np.abs(rg.coeff.real - ri.coeff.real) <= 4 * np.hypot(rg.err.real, ri.err.real)), (rg.coeff.real, ri.coeff.real)
    assert np.all(rg.err.real <= 1e-4 * np.maximum(np.abs(rg.coeff.real), 1e-2))


@pytest.mark.parametrize("physical", [False, True], ids=["euclidean", "physical"])
def test_random_graphs_parity(physical):
    """Inputs nobody chose: random connected multigraphs (2-5 vertices, up to 6 edges, up to five loops), random masses and
    momenta, random propagator powers, both decomposition strategies, both pole extractions, random eps order, a random window
    of eight sectors, a random Korobov vector: whatever qmc_prepare accepts must agree with the oracle per sector, order and
    shift at the C19 tolerance, counters included -- on the table-driven kernels and on the generic one, as the tables decide.
    (A case whose contour counters are non-zero is skipped: the deformation crossed the cut, the values sit on branch cuts.)"""
    import collections
    from qmc_inputs import Workload
    rng = np.random.default_rng(11 if physical else 1)
    stat = collections.Counter()
    for it in range(40):
        V = int(rng.integers(2, 6)); P = int(rng.integers(max(V, 2), 7))
        edges = [(int(rng.integers(0, v)), v) for v in range(1, V)]
        while len(edges) < P:
            a, b = int(rng.integers(0, V)), int(rng.integers(0, V))
            if a != b:
                edges.append((a, b))
        masses = [float(rng.choice([1.0, 2.5, 0.6] if physical else [0.0, 0.0, 1.0, 2.5])) for _ in edges]
        nl = int(rng.integers(2, min(V, 4) + 1))
        legs = [int(x) for x in rng.choice(V, size=nl, replace=False)]
        p = rng.normal(size=(nl, 4)); p[-1] = -p[:-1].sum(axis=0)
        gram = 6.0 * (p @ p.T) if physical else -(p @ p.T)
        nu = None if rng.random() < 0.6 else [int(rng.choice([1, 1, 2])) for _ in edges]
        lam = float(rng.choice([0.2, 0.5])) if physical else 0.0
        wl = Workload("random", V, [(a, b, m) for (a, b), m in zip(edges, masses)], legs, gram, lam)
        for strategy in (0, 1):
            pole = int(rng.random() < 0.3) if lam == 0.0 else 0
            eo = int(rng.integers(0, 2))
            try:
                t = q.qmc_prepare(wl, eps_order=eo, lam=lam, strategy=strategy, pole_extraction=pole, nu=nu, max_depth=10)
            except q.QmcError as e:
                assert e.status in (-2, -3)
                stat["refused"] += 1
                continue
            o = Oracle.from_tables(t.export())
            assert o.status == 0
            N = 4093 if t.dim > 1 else 1021
            z = qi.korobov_vector(N, t.dim, int(rng.integers(2, N - 1)))
            sh = qi.splitmix64_shifts(int(rng.integers(1, 1000)), 2, t.dim)
            s0 = int(rng.integers(0, max(1, t.n_sectors - 8))); s1 = min(t.n_sectors, s0 + 8)
            r = q.qmc_integrate(t, N, 2, z=z, shifts=sh, sectors=(s0, s1), per_sector=True)
            S, A, cnt = o.integrate(N, z, sh, sectors=(s0, s1))
            assert np.array_equal(r.counters, cnt), (it, strategy, r.counters, cnt)
            if cnt[0] or cnt[1]:
                stat["contour counters"] += 1
                continue
            check(r.shift_sums, S, A, f"random graph {it} strategy {strategy} pole {pole} nu {nu} edges {edges}")
            lines = t.describe().splitlines()
            stat[lines[1].split()[0] if len(lines) > 1 else "generic"] += 1
    assert stat["generic"] >= 10 and stat["complex" if physical else "chunk"] >= 10, dict(stat)
