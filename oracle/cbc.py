"""CPU oracle of the component-by-component (CBC) construction of the generating vector -- TEST INFRASTRUCTURE ONLY.

PAPER.md:172 (section 3, below Eq. 20): "the convergence rate can be improved to O(n^-1) [29, 30] if the
generating vector is obtained by the component-by-component construction".  The paper prints neither the
criterion nor the weights; reading C25 fixes them the way reading C13 fixed the Korobov search:

    e^2(z_1..z_d) = -1 + (1/N) sum_{i=0}^{N-1} prod_{j=1}^{d} (1 + omega({i z_j / N})),
    omega(x) = 2 pi^2 B_2(x) = 2 pi^2 (x^2 - x + 1/6)                       (the P_2 figure of merit, weights 1)

    z_1 = 1;  for d = 2..s:  z_d = argmin over z in {1, .., (N-1)/2} of e^2(z_1, .., z_{d-1}, z),  ties -> smaller z
    (N an odd prime; omega(x) = omega(1-x) makes z and N-z exactly equivalent, so only the lower half is searched).
    A tie is a value within TIE_TOL * (1 + minimum) of the minimum: e^2 is the difference of two O(1 + e^2) numbers, so
    the mathematically exact ties of the construction (z and its inverse give the same rule in two dimensions) come out
    of any floating-point evaluation with rounding noise of about 1e-15 (1 + e^2) and must not be decided by it.

This file is the DEFINITION written out: every candidate's criterion is the plain O(N) sum, O(N^2) per component.
No FFT, no primitive roots, no reuse across candidates beyond the running product over the components already fixed.
omega is evaluated from the integer remainder r = i z mod N as 2 pi^2 (1/6 - r (N - r) / N^2): r (N - r) is an exact
integer below 2^53 for N < 9e7, which is what makes the z <-> N-z tie exact.

Pins (tests/test_oracle_cbc.py): closed form e^2(1) = pi^2 / (3 N^2) in one dimension; omega against its Fourier
series values at 0 and 1/2 and its zero mean; the dual-lattice form of e^2 by brute force; exhaustive search over ALL
pairs (z_1, z_2) for small N in pure Python loops; the Fibonacci lattices in two dimensions.
"""
from __future__ import annotations

import numpy as np


TIE_TOL = 1e-11


def omega_from_remainder(r, N: int):
    """omega(r / N) for integer remainders r in [0, N)."""
    r = np.asarray(r, dtype=np.int64)
    return 2.0 * np.pi ** 2 * (1.0 / 6.0 - (r * (N - r)).astype(np.float64) / (float(N) * float(N)))


def criterion(N: int, z) -> float:
    """e^2(z) by its definition: one pass over the N lattice points."""
    i = np.arange(N, dtype=np.int64)
    prod = np.ones(N)
    for zj in z:
        prod = prod * (1.0 + omega_from_remainder((i * int(zj)) % N, N))
    return float(-1.0 + prod.sum() / N)


def cbc_vector(N: int, s: int, chunk: int = 256):
    """(z[s], e2[s]): the CBC vector and the criterion after each component."""
    if N < 3 or N % 2 == 0:
        raise ValueError("N must be an odd prime")
    i = np.arange(N, dtype=np.int64)
    z = [1]
    prod = 1.0 + omega_from_remainder(i % N, N)          # running product over the fixed components, per lattice point
    e2 = [float(-1.0 + prod.sum() / N)]
    half = (N - 1) // 2
    for _ in range(1, s):
        vals = np.empty(half)                                # vals[c - 1] = e^2(z_1..z_{d-1}, c)
        for c0 in range(1, half + 1, chunk):
            cand = np.arange(c0, min(c0 + chunk, half + 1), dtype=np.int64)
            r = (cand[:, None] * i[None, :]) % N             # [candidates, lattice points]
            vals[c0 - 1:c0 - 1 + len(cand)] = -1.0 + ((1.0 + omega_from_remainder(r, N)) * prod[None, :]).sum(axis=1) / N
        best = float(vals.min())
        best_z = int(np.nonzero(vals <= best + TIE_TOL * (1.0 + best))[0][0]) + 1   # smallest z among the ties
        z.append(best_z)
        prod = prod * (1.0 + omega_from_remainder((i * best_z) % N, N))
        e2.append(float(-1.0 + prod.sum() / N))
    return np.array(z, dtype=np.uint64), np.array(e2)
