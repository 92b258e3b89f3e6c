"""Pins for oracle/cbc.py (component-by-component construction; reading C25) -- no GPU.

Each pin checks the oracle against something other than itself: closed forms, the Fourier-side (dual lattice) form of
the criterion, exhaustive search in pure Python loops, and the Fibonacci lattices.
"""
import math

import numpy as np
import pytest

from oracle.cbc import cbc_vector, criterion, omega_from_remainder


def test_omega_closed_form_values():
    # omega(x) = 2 pi^2 B_2(x) = sum_{h != 0} e^{2 pi i h x} / h^2:  omega(0) = 2 zeta(2) = pi^2/3,
    # omega(1/2) = 2 sum (-1)^h / h^2 = -pi^2/6, mean over the N-point grid = (2 pi^2 / N) B_2(0) / N = pi^2 / (3 N^2)
    N = 1000
    assert omega_from_remainder(0, N) == pytest.approx(math.pi ** 2 / 3, rel=1e-15)
    assert omega_from_remainder(N // 2, N) == pytest.approx(-math.pi ** 2 / 6, rel=1e-14)
    assert omega_from_remainder(np.arange(N), N).mean() == pytest.approx(math.pi ** 2 / (3 * N * N), rel=1e-9)
    # truncated Fourier series at a generic point, tail bounded by 2/H
    x, H = 0.3, 200000
    h = np.arange(1, H + 1, dtype=np.float64)
    series = 2.0 * np.sum(np.cos(2 * np.pi * h * x) / h ** 2)
    assert omega_from_remainder(3, 10) == pytest.approx(series, abs=2.0 / H)


@pytest.mark.parametrize("N", [3, 101, 10007])
def test_one_dimensional_closed_form(N):
    # e^2(1) = (2 pi^2 / N) sum_i B_2(i/N) = (2 pi^2 / N) B_2(0) / N = pi^2 / (3 N^2)   (multiplication theorem of B_2)
    assert criterion(N, [1]) == pytest.approx(math.pi ** 2 / (3.0 * N * N), rel=1e-9)
    z, e2 = cbc_vector(N, 1)
    assert list(z) == [1] and e2[0] == pytest.approx(math.pi ** 2 / (3.0 * N * N), rel=1e-9)


def dual_lattice_criterion(N, z):
    """e^2(z) = sum over h in Z^s \\ {0} with h.z = 0 (mod N) of prod_j r(h_j), r(0) = 1, r(h) = 1/h^2, summed exactly
    per residue class: A(a) = sum_{h = a mod N} r(h) = (pi/N)^2 / sin^2(pi a / N) (a != 0), A(0) = 1 + pi^2 / (3 N^2)."""
    A = [1.0 + math.pi ** 2 / (3.0 * N * N)] + [(math.pi / N) ** 2 / math.sin(math.pi * a / N) ** 2 for a in range(1, N)]
    s = len(z)
    total = 0.0
    # all residue vectors (a_1..a_{s-1}) free, a_s fixed by the congruence
    zs_inv = pow(int(z[-1]), -1, N)
    import itertools
    for a in itertools.product(range(N), repeat=s - 1):
        last = (-sum(ai * int(zi) for ai, zi in zip(a, z[:-1])) * zs_inv) % N
        p = A[last]
        for ai in a:
            p *= A[ai]
        total += p
    return total - 1.0   # the term h = 0


@pytest.mark.parametrize("N,z", [(7, (1, 3)), (13, (1, 5)), (31, (1, 12)), (11, (1, 3, 5)), (13, (2, 5, 6))])
def test_criterion_equals_dual_lattice_sum(N, z):
    assert criterion(N, z) == pytest.approx(dual_lattice_criterion(N, z), rel=1e-10)


def test_two_dimensions_exhaustive_pure_python():
    # z_1 = 1 loses nothing in two dimensions (z -> z * unit gives the same point set), so the CBC vector must attain
    # the minimum over ALL pairs; criterion retyped with x = r/N and the B_2 polynomial in plain Python floats
    N = 31
    def e2(z1, z2):
        acc = 0.0
        for i in range(N):
            p = 1.0
            for zz in (z1, z2):
                x = ((i * zz) % N) / N
                p *= 1.0 + 2.0 * math.pi ** 2 * (x * x - x + 1.0 / 6.0)
            acc += p
        return acc / N - 1.0
    table = {(a, b): e2(a, b) for a in range(1, N) for b in range(1, N)}
    best = min(table.values())
    z, e = cbc_vector(N, 2)
    assert z[0] == 1
    assert e[1] == pytest.approx(best, rel=1e-12)
    attained = [b for b in range(1, (N - 1) // 2 + 1) if table[(1, b)] <= best + 1e-11 * (1 + best)]   # tie rule, R:C25
    assert int(z[1]) == min(attained)


@pytest.mark.parametrize("N,f", [(89, 55), (233, 144), (1597, 987)])
def test_fibonacci_lattices(N, f):
    # N = F_k prime: the two-dimensional Fibonacci lattice (1, F_{k-1}) is the best rank-1 rule; CBC must return a
    # member of its equivalence class {f, N-f, f^-1, N-f^-1} (the smallest one, by the tie rule)
    inv = pow(f, -1, N)
    cls = {f, N - f, inv, N - inv}
    z, _ = cbc_vector(N, 2)
    assert int(z[1]) == min(cls)


def test_cbc_steps_are_argmins_and_reported_values_consistent():
    N, s = 251, 4
    z, e2 = cbc_vector(N, s)
    assert np.all(z >= 1) and np.all(z <= (N - 1) // 2)
    for d in range(1, s + 1):
        assert criterion(N, z[:d]) == pytest.approx(e2[d - 1], rel=1e-12)
    for d in range(2, s + 1):           # no other candidate is better at any step; equal ones are larger
        for c in range(1, (N - 1) // 2 + 1):
            v = criterion(N, list(z[:d - 1]) + [c])
            assert v >= e2[d - 1] * (1 - 1e-12)
