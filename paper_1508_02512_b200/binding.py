"""ctypes binding of include/qmc_feynman.h -- argument marshalling only.

Every step of the path (S1-S8) runs inside libqmcfeyn.so (hand-written sm_100a CUDA + host C++).  PyTorch is
used for what it is here for: device memory (the workspace tensor) and the CUDA stream.  There is no CPU
fallback: if the library is missing, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqmcfeyn.so")

QMC_OK, QMC_EINVAL, QMC_EDEPTH, QMC_EUNSUPPORTED, QMC_ECUDA, QMC_ENOMEM, QMC_ECONTOUR = 0, -1, -2, -3, -4, -5, -6


class QmcError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} (status {status})")


class qmc_graph(C.Structure):
    _fields_ = [("n_vertices", C.c_int32), ("n_edges", C.c_int32), ("n_legs", C.c_int32),
                ("edge_u", C.POINTER(C.c_int32)), ("edge_v", C.POINTER(C.c_int32)), ("edge_m2", C.POINTER(C.c_double)),
                ("edge_nu", C.POINTER(C.c_int32)), ("leg_vertex", C.POINTER(C.c_int32))]


class qmc_kinematics(C.Structure):
    _fields_ = [("gram", C.POINTER(C.c_double))]


class qmc_options(C.Structure):
    _fields_ = [("lambda_", C.c_double), ("transform", C.c_int32), ("max_depth", C.c_int32), ("lattice", C.c_int32),
                ("slot_budget", C.c_int32), ("chunk_bytes", C.c_int32), ("threads", C.c_int32),
                ("slot_budget_cplx_real", C.c_int32), ("slot_budget_cplx", C.c_int32), ("dense_template", C.c_int32),
                ("pole_extraction", C.c_int32), ("strategy", C.c_int32)]


class qmc_result(C.Structure):
    _fields_ = [("coeff", C.POINTER(C.c_double)), ("err", C.POINTER(C.c_double)),
                ("sector_coeff", C.POINTER(C.c_double)), ("sector_err", C.POINTER(C.c_double)),
                ("shift_totals", C.POINTER(C.c_double)), ("shift_sums", C.POINTER(C.c_double)),
                ("counters", C.c_int64 * 4), ("kernel_ms", C.c_double), ("eval_kernel_ms", C.c_double),
                ("h2d_bytes", C.c_int64), ("d2h_bytes", C.c_int64),
                ("kernel_launches", C.c_int32),
                ("mode_used", C.c_int32)]


class qmc_run(C.Structure):
    _fields_ = [("z", C.POINTER(C.c_uint64)), ("shifts", C.POINTER(C.c_double)),
                ("index_begin", C.c_uint64), ("index_step", C.c_uint64), ("index_count", C.c_uint64),
                ("sector_begin", C.c_int32), ("sector_end", C.c_int32), ("mode", C.c_int32),
                ("tables_resident", C.c_int32), ("kernel", C.c_int32), ("waves", C.c_int32), ("streams", C.c_int32),
                ("sector_mask", C.POINTER(C.c_uint8))]


_lib = None


def lib():
    """Load libqmcfeyn.so (built in-tree by paper_1508_02512_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1508_02512_b200.build` "
                              "(there is no CPU or PyTorch fallback for the QMC hot path)")
        L = C.CDLL(LIB_PATH)
        L.qmc_prepare.restype = C.c_int
        L.qmc_prepare.argtypes = [C.POINTER(qmc_graph), C.POINTER(qmc_kinematics), C.c_int32, C.POINTER(qmc_options),
                                  C.POINTER(C.c_void_p)]
        L.qmc_prepare_batch.restype = C.c_int
        L.qmc_prepare_batch.argtypes = [C.POINTER(qmc_graph), C.POINTER(qmc_kinematics), C.c_int32, C.c_int32, C.POINTER(qmc_options),
                                        C.POINTER(C.c_void_p)]
        L.qmc_tables_batch_info.restype = C.c_int
        L.qmc_tables_batch_info.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.qmc_tables_free.restype = None
        L.qmc_tables_free.argtypes = [C.c_void_p]
        L.qmc_tables_info.restype = C.c_int
        L.qmc_tables_info.argtypes = [C.c_void_p] + [C.POINTER(C.c_int32)] * 5
        L.qmc_tables_export.restype = C.c_int
        L.qmc_tables_export.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
        L.qmc_workspace_bytes.restype = C.c_size_t
        L.qmc_workspace_bytes.argtypes = [C.c_void_p, C.c_uint64, C.c_int32]
        L.qmc_integrate.restype = C.c_int
        L.qmc_integrate.argtypes = [C.c_void_p, C.c_uint64, C.c_int32, C.c_uint64, C.c_void_p, C.c_void_p, C.c_size_t,
                                    C.POINTER(qmc_result)]
        L.qmc_integrate_ex.restype = C.c_int
        L.qmc_integrate_ex.argtypes = [C.c_void_p, C.c_uint64, C.c_int32, C.c_uint64, C.POINTER(qmc_run), C.c_void_p,
                                       C.c_void_p, C.c_size_t, C.POINTER(qmc_result)]
        L.qmc_integrate_async.restype = C.c_int
        L.qmc_integrate_async.argtypes = [C.c_void_p, C.c_uint64, C.c_int32, C.c_uint64, C.POINTER(qmc_run), C.c_void_p,
                                          C.c_void_p, C.c_size_t]
        L.qmc_result_fetch.restype = C.c_int
        L.qmc_result_fetch.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(qmc_result)]
        L.qmc_result_device_totals.restype = C.c_int
        L.qmc_result_device_totals.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
        L.qmc_statistics.restype = C.c_int
        L.qmc_statistics.argtypes = [C.POINTER(C.c_double), C.c_int32, C.c_int32, C.POINTER(C.c_double),
                                     C.POINTER(C.c_double)]
        L.qmc_flop_model.restype = C.c_int
        L.qmc_flop_model.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                     C.POINTER(C.c_int64)]
        L.qmc_cbc_vector.restype = C.c_int
        L.qmc_cbc_vector.argtypes = [C.c_uint64, C.c_int32, C.POINTER(C.c_uint64), C.POINTER(C.c_double)]
        L.qmc_generating_vector.restype = C.c_int
        L.qmc_generating_vector.argtypes = [C.c_uint64, C.c_int32, C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(C.c_uint64)]
        L.qmc_generating_vector_noalloc.restype = C.c_int
        L.qmc_generating_vector_noalloc.argtypes = [C.c_uint64, C.c_int32, C.c_void_p, C.POINTER(C.c_uint64)]
        L.qmc_embedded_vector.restype = C.c_int
        L.qmc_embedded_vector.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(C.c_uint64)]
        L.qmc_integrate_embedded.restype = C.c_int
        L.qmc_integrate_embedded.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_uint64, C.POINTER(C.c_uint64),
                                             C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(qmc_result), C.POINTER(C.c_int32),
                                             C.POINTER(C.c_int64)]
        L.qmc_integrate_allocated.restype = C.c_int
        L.qmc_integrate_allocated.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_int32, C.c_uint64, C.POINTER(C.c_uint64),
                                              C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(qmc_result), C.POINTER(C.c_int32),
                                              C.POINTER(C.c_int64)]
        L.qmc_shifts.restype = C.c_int
        L.qmc_shifts.argtypes = [C.c_uint64, C.c_int32, C.c_int32, C.POINTER(C.c_double)]
        L.qmc_prefactor_series.restype = C.c_int
        L.qmc_prefactor_series.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_int32, C.c_double,
                                           C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int32)]
        L.qmc_fp64_peak.restype = C.c_int
        L.qmc_fp64_peak.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.qmc_tables_describe.restype = C.c_int
        L.qmc_tables_describe.argtypes = [C.c_void_p, C.c_char_p, C.c_size_t]
        L.qmc_strerror.restype = C.c_char_p
        L.qmc_strerror.argtypes = [C.c_int]
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().qmc_strerror(status).decode()


def _ptr(a: np.ndarray, t):
    return a.ctypes.data_as(C.POINTER(t))


class Tables:
    """Handle of the opaque `qmc_tables` returned by qmc_prepare."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)
        v = [C.c_int32() for _ in range(5)]
        rc = lib().qmc_tables_info(self._h, *[C.byref(x) for x in v])
        if rc:
            raise QmcError(rc, "qmc_tables_info")
        self.n_sectors, self.dim, self.k_min, self.k_max, cx = (int(x.value) for x in v)
        self.is_complex = bool(cx)
        self.K = self.k_max - self.k_min + 1
        npts, spp = C.c_int32(1), C.c_int32(0)
        lib().qmc_tables_batch_info(self._h, C.byref(npts), C.byref(spp))
        self.n_points, self.sectors_per_point = int(npts.value), int(spp.value)   # > 1 point: qmc_prepare_batch
        self._ws = None

    def __del__(self):
        try:
            if self._h:
                lib().qmc_tables_free(self._h)
                self._h = None
        except Exception:
            pass

    def export(self) -> np.ndarray:
        """qmc_tables_export: flat int64/double words (layout in include/qmc_feynman.h)."""
        n = C.c_size_t(0)
        rc = lib().qmc_tables_export(self._h, None, C.byref(n))
        if rc:
            raise QmcError(rc, "qmc_tables_export")
        buf = np.zeros(n.value // 8, dtype=np.int64)
        rc = lib().qmc_tables_export(self._h, buf.ctypes.data_as(C.c_void_p), C.byref(n))
        if rc:
            raise QmcError(rc, "qmc_tables_export")
        return buf

    def describe(self) -> str:
        buf = C.create_string_buffer(1 << 16)
        lib().qmc_tables_describe(self._h, buf, len(buf))
        return buf.value.decode()

    def workspace_bytes(self, N: int, m: int) -> int:
        return int(lib().qmc_workspace_bytes(self._h, N, m))


def qmc_prepare(wl=None, *, n_vertices=None, edges=None, leg_vertex=None, gram=None, eps_order: int = 0,
                lam: float = 0.0, transform: int = 0, max_depth: int = 0, lattice: int = 0, slot_budget: int = 0,
                chunk_bytes: int = 0, threads: int = 0, slot_budget_cplx_real: int = 0, slot_budget_cplx: int = 0,
                dense_template: int = 0, nu=None, pole_extraction: int = 0, strategy: int = 0) -> Tables:
    """qmc_prepare(graph, kinematics, eps_order) -> sector tables.  `wl` is a qmc_inputs.Workload, or pass the
    graph explicitly (edges = [(u, v, m^2), ...]).  slot_budget .. slot_budget_cplx are the table-layout fields of
    qmc_options (0 = the library's defaults).  nu: propagator powers, one per edge (qmc_graph.edge_nu; None = all 1).
    pole_extraction = 1: integration by parts (Eq. 13) instead of the subtraction (real path, generic kernel)."""
    if wl is not None:
        n_vertices, edges, leg_vertex, gram = wl.n_vertices, wl.edges, wl.leg_vertex, wl.gram
        if nu is None:
            nu = getattr(wl, "nu", None)
    eu = np.ascontiguousarray([e[0] for e in edges], dtype=np.int32)
    ev = np.ascontiguousarray([e[1] for e in edges], dtype=np.int32)
    m2 = np.ascontiguousarray([e[2] for e in edges], dtype=np.float64)
    lv = np.ascontiguousarray(leg_vertex, dtype=np.int32)
    gr = np.ascontiguousarray(gram, dtype=np.float64)
    nu_arr = None if nu is None else np.ascontiguousarray(nu, dtype=np.int32)
    if nu_arr is not None and nu_arr.size != len(edges):
        raise ValueError("qmc_prepare: one propagator power per edge")
    g = qmc_graph(n_vertices, len(edges), len(lv), _ptr(eu, C.c_int32), _ptr(ev, C.c_int32), _ptr(m2, C.c_double),
                  None if nu_arr is None else _ptr(nu_arr, C.c_int32), _ptr(lv, C.c_int32))
    k = qmc_kinematics(_ptr(gr, C.c_double))
    o = qmc_options(lam, transform, max_depth, lattice, slot_budget, chunk_bytes, threads, slot_budget_cplx_real,
                    slot_budget_cplx, dense_template, pole_extraction, strategy)
    h = C.c_void_p()
    rc = lib().qmc_prepare(C.byref(g), C.byref(k), eps_order, C.byref(o), C.byref(h))
    if rc:
        raise QmcError(rc, "qmc_prepare")
    return Tables(h.value)


def qmc_prepare_batch(wls, *, eps_order: int = 0, lam: float = 0.0, transform: int = 0, max_depth: int = 0, lattice: int = 0,
                      slot_budget: int = 0, chunk_bytes: int = 0, threads: int = 0, slot_budget_cplx_real: int = 0,
                      slot_budget_cplx: int = 0, dense_template: int = 0, nu=None, pole_extraction: int = 0, strategy: int = 0) -> Tables:
    """qmc_prepare_batch: ONE graph (taken from wls[0]) at the kinematic points of the workloads `wls` (their Gram matrices).
    Integrate with qmc_integrate(..., mode=3): results per kinematic point.  nu, pole_extraction: as in qmc_prepare (such
    tables run on the generic kernel, which has no mode 3: integrate them per point)."""
    w0 = wls[0]
    if nu is None:
        nu = getattr(w0, "nu", None)
    nu_arr = None if nu is None else np.ascontiguousarray(nu, dtype=np.int32)
    if nu_arr is not None and nu_arr.size != len(w0.edges):
        raise ValueError("qmc_prepare_batch: one propagator power per edge")
    eu = np.ascontiguousarray([e[0] for e in w0.edges], dtype=np.int32)
    ev = np.ascontiguousarray([e[1] for e in w0.edges], dtype=np.int32)
    m2 = np.ascontiguousarray([e[2] for e in w0.edges], dtype=np.float64)
    lv = np.ascontiguousarray(w0.leg_vertex, dtype=np.int32)
    grams = [np.ascontiguousarray(w.gram, dtype=np.float64) for w in wls]
    for w in wls:
        assert w.edges == w0.edges and list(w.leg_vertex) == list(w0.leg_vertex), "a batch is one graph at several kinematic points"
    g = qmc_graph(w0.n_vertices, len(w0.edges), len(lv), _ptr(eu, C.c_int32), _ptr(ev, C.c_int32), _ptr(m2, C.c_double),
                  None if nu_arr is None else _ptr(nu_arr, C.c_int32), _ptr(lv, C.c_int32))
    kins = (qmc_kinematics * len(wls))(*[qmc_kinematics(_ptr(gr, C.c_double)) for gr in grams])
    o = qmc_options(lam, transform, max_depth, lattice, slot_budget, chunk_bytes, threads, slot_budget_cplx_real,
                    slot_budget_cplx, dense_template, pole_extraction, strategy)
    h = C.c_void_p()
    rc = lib().qmc_prepare_batch(C.byref(g), kins, len(wls), eps_order, C.byref(o), C.byref(h))
    if rc:
        raise QmcError(rc, "qmc_prepare_batch")
    return Tables(h.value)


@dataclass
class Result:
    coeff: np.ndarray            # [K] complex: Laurent coefficients of J(eps), orders k_min..k_max
    err: np.ndarray              # [K] complex: 1-sigma errors of Re and Im
    shift_totals: np.ndarray     # [K, m] complex
    sector_coeff: Optional[np.ndarray]
    sector_err: Optional[np.ndarray]
    shift_sums: Optional[np.ndarray]   # [n_sectors, K, m] complex
    counters: np.ndarray         # [4]
    kernel_ms: float
    eval_kernel_ms: float
    h2d_bytes: int
    d2h_bytes: int
    kernel_launches: int
    mode_used: int


def _workspace(t: Tables, N: int, m: int, device):
    import torch
    need = t.workspace_bytes(N, m)
    ws = t._ws
    if ws is None or ws.numel() < need or ws.device != torch.device(device):
        ws = torch.empty(need, dtype=torch.uint8, device=device)
        t._ws = ws
    return ws


def _make_run(t: Tables, m: int, z, shifts, index_range, sectors, mode: int, resident: int, kernel: int = 0,
              waves: int = 0, streams: int = 0, sector_mask=None):
    run = qmc_run()
    run.kernel, run.waves, run.streams = kernel, waves, streams
    keep = []
    if sector_mask is not None:
        ma = np.ascontiguousarray(sector_mask, dtype=np.uint8); keep.append(ma)
        assert ma.shape == (t.n_sectors,)
        run.sector_mask = _ptr(ma, C.c_uint8)
    if z is not None:
        za = np.ascontiguousarray(z, dtype=np.uint64); keep.append(za)
        run.z = _ptr(za, C.c_uint64)
    if shifts is not None:
        sa = np.ascontiguousarray(shifts, dtype=np.float64); keep.append(sa)
        assert sa.shape == (m, t.dim)
        run.shifts = _ptr(sa, C.c_double)
    if index_range is not None:
        run.index_begin, run.index_step, run.index_count = index_range
    if sectors is not None:
        run.sector_begin, run.sector_end = sectors
    run.mode = mode
    run.tables_resident = int(resident)
    return run, keep


def _make_result(t: Tables, m: int, ns: int, per_sector: bool):
    K = t.K
    coeff = np.zeros(K, dtype=np.complex128); err = np.zeros(K, dtype=np.complex128)
    shift_totals = np.zeros((K, m), dtype=np.complex128)
    res = qmc_result()
    res.coeff = _ptr(coeff.view(np.float64), C.c_double)
    res.err = _ptr(err.view(np.float64), C.c_double)
    res.shift_totals = _ptr(shift_totals.view(np.float64), C.c_double)
    sc = se = ss = None
    if per_sector:
        sc = np.zeros((ns, K), dtype=np.complex128); se = np.zeros((ns, K), dtype=np.complex128)
        ss = np.zeros((ns, K, m), dtype=np.complex128)
        res.sector_coeff = _ptr(sc.view(np.float64), C.c_double)
        res.sector_err = _ptr(se.view(np.float64), C.c_double)
        res.shift_sums = _ptr(ss.view(np.float64), C.c_double)
    return res, (coeff, err, shift_totals, sc, se, ss)


def _wrap_result(res, arrays) -> Result:
    coeff, err, shift_totals, sc, se, ss = arrays
    return Result(coeff, err, shift_totals, sc, se, ss, np.array(list(res.counters), dtype=np.int64),
                  float(res.kernel_ms), float(res.eval_kernel_ms), int(res.h2d_bytes), int(res.d2h_bytes),
                  int(res.kernel_launches), int(res.mode_used))


def qmc_integrate(t: Tables, N: int, m: int, seed: int = 0, *, z: Optional[Sequence[int]] = None,
                  shifts: Optional[np.ndarray] = None, index_range=None, sectors=None, per_sector: bool = False,
                  mode: int = 0, resident: int = 0, kernel: int = 0, waves: int = 0, streams: int = 0, sector_mask=None,
                  device="cuda:0", stream=None) -> Result:
    """qmc_integrate(tables, N, m, seed) -> Laurent coefficients and errors (qmc_integrate_ex when any of the
    explicit controls is given).  Workspace and stream come from PyTorch."""
    import torch
    if not torch.cuda.is_available():
        raise QmcError(QMC_ECUDA, "qmc_integrate (no CUDA device; there is no CPU fallback)")
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = _workspace(t, N, m, dev)
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        s0, s1 = sectors if sectors is not None else (0, t.n_sectors)
        rows = t.n_points if mode == 3 else s1 - s0       # mode 3: one row of results per kinematic point of a batch
        res, arrays = _make_result(t, m, rows, per_sector or mode == 3)
        run, keep = _make_run(t, m, z, shifts, index_range, sectors, mode, resident, kernel, waves, streams, sector_mask)
        rc = lib().qmc_integrate_ex(t._h, N, m, seed, C.byref(run), C.c_void_p(st.cuda_stream),
                                    C.c_void_p(ws.data_ptr()), ws.numel(), C.byref(res))
        if rc:
            raise QmcError(rc, "qmc_integrate")
    return _wrap_result(res, arrays)


def qmc_integrate_async(t: Tables, N: int, m: int, seed: int = 0, *, z=None, shifts=None, index_range=None,
                        sectors=None, mode: int = 1, resident: int = 0, kernel: int = 0, waves: int = 0, streams: int = 0,
                        device="cuda:0", stream=None) -> None:
    """Enqueue S1-S8 on the stream and return without synchronising; results stay in the workspace of `t`
    (qmc_result_fetch brings them to the host).  resident=2: nothing is copied from the host."""
    import torch
    if not torch.cuda.is_available():
        raise QmcError(QMC_ECUDA, "qmc_integrate_async (no CUDA device; there is no CPU fallback)")
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = _workspace(t, N, m, dev)
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        run, keep = _make_run(t, m, z, shifts, index_range, sectors, mode, resident, kernel, waves, streams)
        rc = lib().qmc_integrate_async(t._h, N, m, seed, C.byref(run), C.c_void_p(st.cuda_stream),
                                       C.c_void_p(ws.data_ptr()), ws.numel())
        if rc:
            raise QmcError(rc, "qmc_integrate_async")


def qmc_result_fetch(t: Tables, m: int, *, per_sector: bool = False, n_sectors: Optional[int] = None, device="cuda:0",
                     stream=None) -> Result:
    """Results of the last qmc_integrate_async on `t`: one D2H copy + stream synchronisation."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = t._ws
        if ws is None:
            raise QmcError(QMC_EINVAL, "qmc_result_fetch (no launch on these tables)")
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        res, arrays = _make_result(t, m, t.n_sectors if n_sectors is None else n_sectors, per_sector)
        rc = lib().qmc_result_fetch(t._h, C.c_void_p(st.cuda_stream), C.c_void_p(ws.data_ptr()), ws.numel(), C.byref(res))
        if rc:
            raise QmcError(rc, "qmc_result_fetch")
    return _wrap_result(res, arrays)


def qmc_result_device_totals(t: Tables, m: int):
    """torch view (float64, shape [K, m, 2]) of the per-shift totals the last qmc_integrate_async left on the device."""
    import torch
    ws = t._ws
    p = C.c_void_p()
    rc = lib().qmc_result_device_totals(t._h, C.c_void_p(ws.data_ptr()), ws.numel(), C.byref(p))
    if rc:
        raise QmcError(rc, "qmc_result_device_totals")
    off = p.value - ws.data_ptr()
    return ws[off: off + t.K * m * 16].view(torch.float64).view(t.K, m, 2)


def qmc_statistics(shift_totals: np.ndarray):
    """Eqs. 19-20 on per-shift estimates [K, m] (complex) -> (coeff[K], err[K])."""
    T = np.ascontiguousarray(shift_totals, dtype=np.complex128)
    K, m = T.shape
    coeff = np.zeros(K, dtype=np.complex128); err = np.zeros(K, dtype=np.complex128)
    rc = lib().qmc_statistics(_ptr(T.view(np.float64), C.c_double), K, m, _ptr(coeff.view(np.float64), C.c_double),
                              _ptr(err.view(np.float64), C.c_double))
    if rc:
        raise QmcError(rc, "qmc_statistics")
    return coeff, err


def qmc_flop_model(t: Tables, sectors=None):
    """(flops once per point, flops in all sectors, corner evaluations) per (lattice point, shift)."""
    s0, s1 = sectors if sectors is not None else (0, 0)
    fp, fs, nc = C.c_double(0), C.c_double(0), C.c_int64(0)
    rc = lib().qmc_flop_model(t._h, s0, s1, C.byref(fp), C.byref(fs), C.byref(nc))
    if rc:
        raise QmcError(rc, "qmc_flop_model")
    return float(fp.value), float(fs.value), int(nc.value)


def qmc_shifts(seed: int, m: int, dim: int) -> np.ndarray:
    out = np.zeros((m, dim))
    rc = lib().qmc_shifts(seed, m, dim, _ptr(out, C.c_double))
    if rc:
        raise QmcError(rc, "qmc_shifts")
    return out


def qmc_generating_vector(N: int, dim: int, device="cuda:0") -> np.ndarray:
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = torch.empty(1 << 20, dtype=torch.uint8, device=dev)
        z = np.zeros(dim, dtype=np.uint64)
        rc = lib().qmc_generating_vector(N, dim, C.c_void_p(torch.cuda.current_stream(dev).cuda_stream),
                                         C.c_void_p(ws.data_ptr()), ws.numel(), _ptr(z, C.c_uint64))
    if rc:
        raise QmcError(rc, "qmc_generating_vector")
    return z


def qmc_generating_vector_noalloc(N: int, dim: int, device="cuda:0") -> np.ndarray:
    """qmc_generating_vector without a workspace: the library's own fixed device array is the scratch (no allocation)."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        z = np.zeros(max(dim, 1), dtype=np.uint64)
        rc = lib().qmc_generating_vector_noalloc(N, dim, C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), _ptr(z, C.c_uint64))
    if rc:
        raise QmcError(rc, "qmc_generating_vector_noalloc")
    return z[:dim]


def qmc_embedded_vector(k_min: int, k_max: int, dim: int, device="cuda:0") -> np.ndarray:
    """Generating vector (odd components) shared by the lattices N = 2^k, k_min <= k <= k_max (embedded sequence)."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = torch.empty(1 << 20, dtype=torch.uint8, device=dev)
        z = np.zeros(dim, dtype=np.uint64)
        rc = lib().qmc_embedded_vector(k_min, k_max, dim, C.c_void_p(torch.cuda.current_stream(dev).cuda_stream),
                                       C.c_void_p(ws.data_ptr()), ws.numel(), _ptr(z, C.c_uint64))
    if rc:
        raise QmcError(rc, "qmc_embedded_vector")
    return z


def qmc_integrate_embedded(t: Tables, k_min: int, k_max: int, m: int, seed: int, z, target_rel_err: float = 0.0,
                           device="cuda:0", stream=None):
    """qmc_integrate_embedded: levels 2^k_min .. of an embedded lattice sequence, each level evaluating only its new (odd)
    indices.  Returns (Result, k_reached, points_evaluated_per_shift)."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = _workspace(t, 1 << k_max, m, dev)
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        res, arrays = _make_result(t, m, 0, False)
        za = np.ascontiguousarray(z, dtype=np.uint64)
        kr, npts = C.c_int32(0), C.c_int64(0)
        rc = lib().qmc_integrate_embedded(t._h, k_min, k_max, float(target_rel_err), m, seed, _ptr(za, C.c_uint64),
                                          C.c_void_p(st.cuda_stream), C.c_void_p(ws.data_ptr()), ws.numel(), C.byref(res),
                                          C.byref(kr), C.byref(npts))
        if rc:
            raise QmcError(rc, "qmc_integrate_embedded")
    return _wrap_result(res, arrays), int(kr.value), int(npts.value)


def qmc_integrate_allocated(t: Tables, k0: int, k_max: int, m: int, seed: int, z, target_rel_err: float,
                            device="cuda:0", stream=None):
    """qmc_integrate_allocated: per-sector lattice sizes by variance.  Returns (Result, levels[n_sectors], evals_per_shift)."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = _workspace(t, 1 << k_max, m, dev)
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        res, arrays = _make_result(t, m, 0, False)
        za = np.ascontiguousarray(z, dtype=np.uint64)
        lev = np.zeros(t.n_sectors, dtype=np.int32)
        ev = C.c_int64(0)
        rc = lib().qmc_integrate_allocated(t._h, k0, k_max, float(target_rel_err), m, seed, _ptr(za, C.c_uint64),
                                           C.c_void_p(st.cuda_stream), C.c_void_p(ws.data_ptr()), ws.numel(), C.byref(res),
                                           _ptr(lev, C.c_int32), C.byref(ev))
        if rc:
            raise QmcError(rc, "qmc_integrate_allocated")
    return _wrap_result(res, arrays), lev, int(ev.value)


def qmc_cbc_vector(N: int, dim: int, with_criterion: bool = False):
    """Component-by-component generating vector (host function of the library)."""
    z = np.zeros(dim, dtype=np.uint64)
    e2 = np.zeros(dim, dtype=np.float64)
    rc = lib().qmc_cbc_vector(N, dim, _ptr(z, C.c_uint64), _ptr(e2, C.c_double))
    if rc != 0:
        raise QmcError(rc, "qmc_cbc_vector")
    return (z, e2) if with_criterion else z


def qmc_prefactor_series(eg: float, base: float, p0: float, p1: float, g0: int, g1: float, n_out: int):
    """Laurent series of e^{eg eps gammaE} base^{p0+p1 eps} Gamma(g0 + g1 eps): (coefficients, lowest order)."""
    out = np.zeros(n_out)
    lo = C.c_int32(0)
    rc = lib().qmc_prefactor_series(eg, base, p0, p1, g0, g1, n_out, _ptr(out, C.c_double), C.byref(lo))
    if rc:
        raise QmcError(rc, "qmc_prefactor_series")
    return out, int(lo.value)


def qmc_fp64_peak(device="cuda:0"):
    """Measured sustained DFMA rate of the device in FLOP/s (DFMA = 2) and the kernel time in ms."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        ws = torch.empty(4096, dtype=torch.uint8, device=dev)
        fl, ms = C.c_double(0), C.c_double(0)
        rc = lib().qmc_fp64_peak(C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), C.c_void_p(ws.data_ptr()),
                                 ws.numel(), C.byref(fl), C.byref(ms))
    if rc:
        raise QmcError(rc, "qmc_fp64_peak")
    return float(fl.value), float(ms.value)
