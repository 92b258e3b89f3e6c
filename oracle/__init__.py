"""CPU oracle of the arXiv:1508.02512 hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports the CUDA product and shares no code with it.

`build()` compiles oracle/qmc_oracle.cpp with g++ (-O2 -fopenmp) into oracle/libqmc_oracle.so;
`Oracle` is a thin ctypes wrapper (argument marshalling only; all arithmetic is in the C++ file).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qmc_oracle.cpp")
_LIB = os.path.join(_HERE, "libqmc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_build.restype = C.c_void_p
        L.orc_from_tables.restype = C.c_void_p
        L.orc_integrate.restype = C.c_int
        L.orc_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def max_threads() -> int:
    return int(_load().orc_max_threads())


def statistics(T: np.ndarray):
    """Eqs. 19-20.  T[K, m] complex -> mean[K], err[K] (complex: Re/Im errors)."""
    T = np.ascontiguousarray(T, dtype=np.complex128)
    K, m = T.shape
    mean = np.zeros(K, dtype=np.complex128)
    err = np.zeros(K, dtype=np.complex128)
    _load().orc_statistics(_p(T.view(np.float64), C.c_double), C.c_int(K), C.c_int(m),
                           _p(mean.view(np.float64), C.c_double), _p(err.view(np.float64), C.c_double))
    return mean, err


def lattice(N: int, z: Sequence[int], i0: int, count: int, shift: Sequence[float], transform: int = 0):
    z = np.ascontiguousarray(z, dtype=np.uint64)
    n = len(z)
    shift = np.ascontiguousarray(shift, dtype=np.float64)
    y = np.zeros((count, n)); t = np.zeros((count, n)); w = np.zeros(count)
    inside = np.zeros(count, dtype=np.int32)
    _load().orc_lattice(C.c_uint64(N), _p(z, C.c_uint64), C.c_int(n), C.c_uint64(i0), C.c_uint64(count),
                        _p(shift, C.c_double), C.c_int(transform), _p(y, C.c_double), _p(t, C.c_double),
                        _p(w, C.c_double), _p(inside, C.c_int))
    return y, t, w, inside


class Oracle:
    """One (graph, kinematics, lambda, eps_order) problem, decomposed into sectors."""

    def __init__(self, handle):
        if not handle:
            raise ValueError("oracle: invalid graph / tables")
        self._h = C.c_void_p(handle)
        info = np.zeros(12, dtype=np.int32)
        _load().orc_info(self._h, _p(info, C.c_int))
        (self.status, self.L, self.dim, self.n_sectors, self.k_min, self.k_max,
         self.aU0, self.aU1, self.aF0, self.aF1, self.n_terms_U, self.n_terms_F) = (int(v) for v in info)
        self.K = self.k_max - self.k_min + 1

    @classmethod
    def from_workload(cls, wl, lam: Optional[float] = None, eps_order: Optional[int] = None, max_depth: int = 64,
                      order: int = 0, taylor: bool = False, ibp: bool = False):
        """order = 0: decomposition rule A.3 (U^ first); 1: F^ first (only to pin strategy independence of the totals).
        wl.nu: propagator powers (None = all 1).  taylor: accept alpha_j <= -2 on the real path (the p >= 1 Taylor terms of
        Eq. 11) instead of status -3.  ibp: pole extraction by integration by parts
        (Eq. 13) instead of the subtraction; real path only."""
        eu, ev, m2, lv, gram = wl.arrays()
        nu = getattr(wl, "nu", None)
        nu_arr = None if nu is None else np.ascontiguousarray(nu, dtype=np.int32)
        if nu_arr is not None and nu_arr.size != wl.n_edges:
            raise ValueError("oracle: one propagator power per edge")
        L = _load()
        L.orc_build_nu.restype = C.c_void_p
        h = L.orc_build_nu(C.c_int(wl.n_vertices), C.c_int(wl.n_edges), C.c_int(len(lv)), _p(eu, C.c_int),
                           _p(ev, C.c_int), _p(m2, C.c_double), _p(lv, C.c_int), _p(gram, C.c_double),
                           C.c_double(wl.lam if lam is None else lam),
                           C.c_int(wl.eps_order if eps_order is None else eps_order), C.c_int(max_depth), C.c_int(order),
                           None if nu_arr is None else _p(nu_arr, C.c_int), C.c_int((1 if taylor else 0) | (2 if ibp else 0)))
        o = cls(h)
        o.n_edges = wl.n_edges
        return o

    @classmethod
    def from_sector(cls, alpha, beta, U, F, aU, aF, eps_order: int = 0, ibp: bool = False):
        """ONE explicit real sector prod_j t_j^(alpha_j + beta_j eps) U(t)^(aU[0] + aU[1] eps) F(t)^(aF[0] + aF[1] eps) on the
        unit cube (the form of Eq. 9), Taylor terms enabled.  U, F: lists of (coefficient, exponent tuple),
        each with a constant term."""
        alpha = np.ascontiguousarray(alpha, dtype=np.int32); beta = np.ascontiguousarray(beta, dtype=np.int32)
        n = alpha.size
        def flat(Q):
            c = np.ascontiguousarray([q[0] for q in Q], dtype=np.float64)
            e = np.ascontiguousarray([q[1] for q in Q], dtype=np.int32).reshape(len(Q), n)
            return c, e
        cU, eU = flat(U); cF, eF = flat(F)
        L = _load()
        L.orc_from_sector.restype = C.c_void_p
        h = L.orc_from_sector(C.c_int(n), _p(alpha, C.c_int), _p(beta, C.c_int), C.c_int(len(U)), _p(cU, C.c_double),
                              _p(eU, C.c_int), C.c_int(len(F)), _p(cF, C.c_double), _p(eF, C.c_int), C.c_int(aU[0]),
                              C.c_int(aU[1]), C.c_int(aF[0]), C.c_int(aF[1]), C.c_int(eps_order), C.c_int(1 if ibp else 0))
        o = cls(h)
        o.n_edges = n + 1
        return o

    @classmethod
    def from_tables(cls, words: np.ndarray):
        words = np.ascontiguousarray(words, dtype=np.int64)
        h = _load().orc_from_tables(_p(words, C.c_int64), C.c_size_t(words.size))
        return cls(h)

    def __del__(self):
        try:
            if self._h:
                _load().orc_free(self._h)
                self._h = None
        except Exception:
            pass

    # ---- inspection (pins) ------------------------------------------------------------
    def graph_poly(self, which: str):
        nt = self.n_terms_U if which == "U" else self.n_terms_F
        coeff = np.zeros(nt); expo = np.zeros((nt, self.n_edges), dtype=np.int32)
        _load().orc_graph_poly(self._h, C.c_int(0 if which == "U" else 1), _p(coeff, C.c_double), _p(expo, C.c_int))
        return coeff, expo

    def sector(self, s: int):
        meta = np.zeros(4, dtype=np.int32)
        alpha = np.zeros(self.dim, dtype=np.int32); beta = np.zeros(self.dim, dtype=np.int32)
        jac = np.zeros(self.dim, dtype=np.int32)
        L = _load()
        L.orc_sector_meta(self._h, C.c_int(s), _p(meta, C.c_int), _p(alpha, C.c_int), _p(beta, C.c_int), _p(jac, C.c_int))
        out = {"primary": int(meta[0]), "n_sing": int(meta[3]), "alpha": alpha, "beta": beta, "jac": jac}
        for name, which, nt in (("U", 0, int(meta[1])), ("F", 1, int(meta[2]))):
            coeff = np.zeros(nt); expo = np.zeros((nt, self.dim), dtype=np.int32)
            L.orc_sector_poly(self._h, C.c_int(s), C.c_int(which), _p(coeff, C.c_double), _p(expo, C.c_int))
            out[name] = (coeff, expo)
        return out

    def deform(self, s: int, t: Sequence[float]):
        t = np.ascontiguousarray(t, dtype=np.float64)
        z = np.zeros(self.dim, dtype=np.complex128); det = np.zeros(1, dtype=np.complex128)
        _load().orc_deform(self._h, C.c_int(s), _p(t, C.c_double), _p(z.view(np.float64), C.c_double),
                           _p(det.view(np.float64), C.c_double))
        return z, det[0]

    def sector_integrand(self, s: int, t: Sequence[float]):
        """c_k(t), k = -n_sing(s)..k_max, at one real point (no lattice weight)."""
        t = np.ascontiguousarray(t, dtype=np.float64)
        out = np.zeros(self.K + 8, dtype=np.complex128)
        _load().orc_sector_integrand(self._h, C.c_int(s), _p(t, C.c_double), _p(out.view(np.float64), C.c_double))
        ns = self.sector(s)["n_sing"]
        return out[: self.k_max + ns + 1]

    def sector_integrand_taylor(self, s: int, t: Sequence[float]):
        """The same c_k(t) through the Taylor-term formula (sector_point_taylor), whatever the sector; real path only.
        Returns (c, sum of |terms|)."""
        t = np.ascontiguousarray(t, dtype=np.float64)
        out = np.zeros(self.K + 8); ab = np.zeros(self.K + 8)
        rc = _load().orc_sector_integrand_taylor(self._h, C.c_int(s), _p(t, C.c_double), _p(out, C.c_double), _p(ab, C.c_double))
        if rc != 0:
            raise RuntimeError(f"oracle: Taylor-term formula is real-path only ({rc})")
        ns = self.sector(s)["n_sing"]
        return out[: self.k_max + ns + 1], ab[: self.k_max + ns + 1]

    # ---- the path ---------------------------------------------------------------------
    def integrate(self, N: int, z, shifts, transform: int = 0, index_range=None, sectors=None, threads: int = 0):
        """Level-1 oracle: S[sector, k-k_min, shift] (complex), A (un-cancelled magnitude, R:C19), counters."""
        z = np.ascontiguousarray(z, dtype=np.uint64)
        shifts = np.ascontiguousarray(shifts, dtype=np.float64)
        m = shifts.shape[0]
        assert shifts.shape[1] == self.dim and z.size == self.dim
        i0, step, cnt = index_range if index_range is not None else (0, 1, N)
        s0, s1 = sectors if sectors is not None else (0, self.n_sectors)
        S = np.zeros((s1 - s0, self.K, m), dtype=np.complex128)
        A = np.zeros((s1 - s0, self.K, m))
        counters = np.zeros(4, dtype=np.int64)
        rc = _load().orc_integrate(self._h, C.c_uint64(N), _p(z, C.c_uint64), C.c_int(m), _p(shifts, C.c_double),
                                   C.c_int(transform), C.c_uint64(i0), C.c_uint64(step), C.c_uint64(cnt),
                                   C.c_int(s0), C.c_int(s1), C.c_int(threads), _p(S.view(np.float64), C.c_double),
                                   _p(A, C.c_double), _p(counters, C.c_int64))
        if rc != 0:
            raise RuntimeError(f"oracle integrate failed: {rc}")
        return S, A, counters

    def totals(self, S: np.ndarray):
        """Level 2: per-shift totals over sectors, then Eqs. 19-20.  Returns (coeff[K], err[K])."""
        return statistics(S.sum(axis=0))
