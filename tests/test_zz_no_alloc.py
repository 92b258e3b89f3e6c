"""qmc_generating_vector_noalloc: the allocation-free entry point (its scratch is a fixed device array inside the library)
against the existing path qmc_generating_vector (scratch in a caller-allocated workspace).  Same candidates, same kernel:
the generating vectors are integers and must be IDENTICAL -- on two calls in a row, which share the array and find the
previous call's contents in it.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import qmc_inputs as qi
import paper_1508_02512_b200 as q

pytestmark = pytest.mark.gpu


def test_noalloc_generating_vector_matches_the_workspace_path_on_consecutive_calls():
    # first call: a large lattice in 6 dimensions; second call right after it: a smaller lattice in 3 dimensions (fewer
    # components written per candidate: stale contents of the first call stay behind in the array and must not matter)
    cases = [(999983, 6), (99991, 3), (99991, 3), (1048573, 5), (10007, 2), (16381, 8)]
    got = [q.qmc_generating_vector_noalloc(N, d) for N, d in cases]            # back to back, nothing in between
    want = [q.qmc_generating_vector(N, d) for N, d in cases]
    for (N, d), a, b in zip(cases, got, want):
        assert a.shape == (d,) and np.array_equal(a, b), (N, d, a, b)
        assert a[0] == 1 and all(np.gcd(int(v), N) == 1 for v in a)             # a valid rule
        assert all(int(a[j + 1]) == (int(a[j]) * int(a[1])) % N for j in range(d - 1))   # Korobov form (reading C13)
    assert np.array_equal(got[1], got[2])                                          # the same call twice: the same answer


def test_noalloc_vector_drives_the_kernels_like_the_workspace_one():
    wl = qi.massless_box()
    t = q.qmc_prepare(wl)
    N, m = 99991, 8
    sh = qi.splitmix64_shifts(wl.seed, m, 3)
    a = q.qmc_integrate(t, N, m, z=q.qmc_generating_vector_noalloc(N, 3), shifts=sh)
    b = q.qmc_integrate(t, N, m, seed=wl.seed)                                    # the library's own search + the same shifts
    assert np.array_equal(a.shift_totals, b.shift_totals)
    ex = [0.666666666666667, -1.2639198230760183, -1.2238036181980894]            # closed form (tests/test_oracle_closed_forms.py)
    assert np.all(np.abs(a.coeff.real - ex) <= 3.5 * a.err.real)


def test_noalloc_rejects_what_its_fixed_scratch_cannot_hold():
    with pytest.raises(q.QmcError) as e:
        q.qmc_generating_vector_noalloc(99991, 9)          # more components than the scratch is sized for
    assert e.value.status == q.binding.QMC_ENOMEM and "too small" in str(e.value)
    with pytest.raises(q.QmcError) as e:
        q.qmc_generating_vector_noalloc(1 << 31, 3)        # N beyond the 32-bit lattice arithmetic of the kernels
    assert e.value.status == q.binding.QMC_EINVAL
    assert np.array_equal(q.qmc_generating_vector_noalloc(99991, 1), [1])
