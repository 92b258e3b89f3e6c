"""bench.py -- FP64 integrand evaluations per second of the QMC hot path (arXiv:1508.02512) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--N 999983] [--impl reference]

One "step" = one pass of the whole hot path S1-S8 (lattice points, shifts, periodising transform, all sectors with
their subtraction corners / contour deformation, per-shift reduction, statistics) over one batch: N lattice
points x m shifts x all sectors of the workload.  One evaluation = one (lattice point, shift, sector) triple
(BASELINE.md M1).  Prints ONE JSON line (rank 0).  DESIGN.md "Measurement" explains every key.

N > 1 GPUs (torchrun): weak scaling over shift vectors -- every rank integrates its own block of m shift vectors of
the one SplitMix64 stream (per-GPU work fixed), the per-shift totals are all-gathered (NCCL), Eqs. 19-20 run over all
m x N_gpus estimates.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import qmc_inputs as qi  # noqa: E402  (seeded input generators only)

METRIC = "fp64_integrand_evals_per_sec_all_sectors"
UNIT = "evals/s"

# default lattice size per config for the timed step (primes from BASELINE.md).  cfg4: the middle one of the three sizes
# BASELINE.json lists (a step is ~1.8 s, so the driver's 25 device-timed + 20 end-to-end steps take ~1.5 min); the largest,
# 99999989 (~18 s per step), is timed once beside it (`largest_size`)
DEFAULT_N = {1: 10007, 2: 9999991, 3: 9999991, 4: 9999991, 5: 1048573}
LARGEST_N = {4: 99999989}


def workload(cfg: int):
    return qi.CONFIGS()[cfg - 1]


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML every 100 ms while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag = index, threading.Event()
        self.mhz, self.reasons, self.max_mhz, self.power = [], set(), None, []

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                     "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
            while not self.stop_flag.is_set():
                self.mhz.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                except Exception:
                    pass
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                time.sleep(0.1)
        except Exception as e:  # NVML missing: report that, never fail the bench
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def summary(self):
        self.stop_flag.set()
        self.join(timeout=2.0)
        return {"sm_mhz": float(np.median(self.mhz)) if self.mhz else None, "sm_max_mhz": self.max_mhz,
                "power_w_max": max(self.power) if self.power else None, "samples": len(self.mhz),
                "reasons": sorted(self.reasons)}


def host_cores() -> int:
    """Threads the oracle is run with, set explicitly (an inherited OMP_NUM_THREADS=1 made the two arms differ in round 1)."""
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except Exception:
        return max(1, os.cpu_count() or 1)


def config_of(wl, N, n_sectors, world):
    """The `config` object: the same keys in the product arm and in the reference arm."""
    return {"workload": wl.name, "N": int(N), "m": int(wl.m), "seed": int(wl.seed), "n_sectors": int(n_sectors), "dim": int(wl.dim),
            "lambda": float(wl.lam), "parallelism": f"shift-sharded x{world}",
            "l2": "flushed between steps (256 MiB fill, outside the event pairs); the tables (<= 300 KB) travel in the kernel parameters, nothing else is read"}


def oracle_sample(wl, N, z, shifts, target_s: float):
    """Time the oracle (as it stands, all host cores) on a bounded sample of the same workload: the first `count`
    lattice indices of the rule, all sectors, the first m_s shift vectors.  Returns (evals/s, cores, description)."""
    import oracle
    o = oracle.Oracle.from_workload(wl)       # the oracle's own decomposition: no product code on this path
    cores = host_cores()
    m_s = min(2, shifts.shape[0])
    count = max(cores * 4, 64)
    t0 = time.perf_counter()
    o.integrate(N, z, shifts[:m_s], index_range=(0, 1, count), threads=cores)
    dt = time.perf_counter() - t0
    rate = count * m_s * o.n_sectors / dt
    count = int(min(N, max(count, target_s * rate / (m_s * o.n_sectors))))
    t0 = time.perf_counter()
    o.integrate(N, z, shifts[:m_s], index_range=(0, 1, count), threads=cores)
    dt = time.perf_counter() - t0
    val = count * m_s * o.n_sectors / dt
    c1 = max(64, count // (4 * cores))
    t0 = time.perf_counter()
    o.integrate(N, z, shifts[:m_s], index_range=(0, 1, c1), threads=1)
    oracle_sample.single_thread = c1 * m_s * o.n_sectors / (time.perf_counter() - t0)
    return val, cores, (f"{wl.name}: lattice indices 0..{count - 1} of N={N}, all {o.n_sectors} sectors, {m_s} shifts, "
                        f"{dt:.1f} s on {cores} threads (OpenMP), g++ -O2")


def test_vector(N: int, dim: int) -> np.ndarray:
    """A valid generating vector without a GPU (reference arm): tabulated Korobov multiplier, else a fixed one."""
    if dim == 1 or (N, dim) in qi.GOOD_KOROBOV:
        return qi.good_vector(N, dim)
    return qi.korobov_vector(N, dim, 76 if N > 76 else 2)


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the same workload / metric; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = workload(args.config)
    N = args.N or DEFAULT_N[args.config]
    z = test_vector(N, wl.dim)
    shifts = qi.splitmix64_shifts(wl.seed, wl.m, wl.dim)
    import oracle
    oracle.build()
    per_step = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    vals, desc, cores = [], "", 0
    for i in range(args.warmup + args.steps):
        v, cores, desc = oracle_sample(wl, N, z, shifts, per_step)
        if i >= args.warmup:
            vals.append(v)
    val = float(np.mean(vals))
    n_sectors = oracle.Oracle.from_workload(wl).n_sectors
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * N * wl.m * n_sectors / val, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_of(wl, N, n_sectors, 1),
            "note": "ms_per_step extrapolated from the bounded sample (cost is linear in N*m)",
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def time_to_accuracy(q, wl, torch, target=1e-3, max_N=2 ** 27, transform=0):
    """M2: raise N through the primes below 2^k until the relative error of the eps^0 coefficient of J is <= target
    (reading C17); wall time of everything the user waits for after qmc_prepare: generating-vector search, uploads,
    kernels, downloads, statistics, summed over the N tried.  `rel_err` is the ESTIMATED standard error of Eq. 20 over the
    coefficient (what the paper calls accuracy), not a deviation from a known value."""
    t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam, transform=transform)
    q.qmc_integrate(t, 16381, wl.m, seed=wl.seed)          # context / module warm-up, not timed
    tried = []
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    rel = None
    for N in qi.primes_below_pow2(14, 27):
        if N > max_N:
            break
        r = q.qmc_integrate(t, N, wl.m, seed=wl.seed)
        c0, e0 = r.coeff[-1 - wl.eps_order], r.err[-1 - wl.eps_order]
        rel = max(e0.real, e0.imag) / abs(c0)
        tried.append(N)
        if rel <= target:
            break
    dt = time.perf_counter() - t0
    return {"workload": wl.name, "transform": transform, "target_rel_err": target, "wall_s": dt, "N_reached": tried[-1], "N_tried": len(tried),
            "rel_err": rel, "coeff_eps0": [c0.real, c0.imag], "err_eps0": [e0.real, e0.imag], "m": wl.m}


def time_to_accuracy_embedded(q, wl, torch, target=1e-5, k_min=14, k_max=22, transform=0):
    """M2 with an embedded lattice sequence (reading C26): N = 2^k with one odd generating vector; every level
    evaluates only its new points (qmc_integrate_embedded), where `time_to_accuracy` starts again at every N.  Wall time of
    everything after qmc_prepare, the vector search over all levels included (`search_s`)."""
    t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam, transform=transform)
    q.qmc_integrate(t, 16381, wl.m, seed=wl.seed)          # context / module warm-up, not timed
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    z = q.qmc_embedded_vector(k_min, k_max, t.dim)
    t1 = time.perf_counter()
    r, k, npts = q.qmc_integrate_embedded(t, k_min, k_max, wl.m, wl.seed, z, target_rel_err=target)
    dt = time.perf_counter() - t0
    c0, e0 = r.coeff[-1], r.err[-1]
    return {"workload": wl.name, "transform": transform, "target_rel_err": target, "wall_s": dt, "search_s": t1 - t0,
            "N_reached": 1 << k, "levels": k - k_min + 1, "points_evaluated_per_shift": npts,
            "points_if_restarted_per_level": (1 << (k + 1)) - (1 << k_min), "rel_err": float(max(e0.real, e0.imag) / abs(c0)),
            "coeff_eps0": [c0.real, c0.imag], "err_eps0": [e0.real, e0.imag], "m": wl.m, "z": [int(v) for v in z]}


def allocation_vs_uniform(q, torch, target=1e-5):
    """SURVEY 8(f) f4, reading C27: per-sector lattice sizes by variance (qmc_integrate_allocated) against the uniform embedded
    sequence at the same target, same vector and shifts: wall time and integrand evaluations per shift vector."""
    out = []
    for wl in (qi.double_box(), qi.nonplanar_vertex()):
        t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
        z = q.qmc_embedded_vector(13, 24, t.dim)
        q.qmc_integrate(t, 16381, wl.m, seed=wl.seed)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r, lev, ev = q.qmc_integrate_allocated(t, 13, 24, wl.m, wl.seed, z, target)
        ta = time.perf_counter() - t0
        t0 = time.perf_counter()
        u, k, npts = q.qmc_integrate_embedded(t, 13, 24, wl.m, wl.seed, z, target_rel_err=target)
        tu = time.perf_counter() - t0
        rel = lambda x: float(max(x.err[-1].real, x.err[-1].imag) / abs(x.coeff[-1]))
        out.append({"workload": wl.name, "target_rel_err": target, "m": wl.m,
                    "allocated": {"wall_s": ta, "rel_err": rel(r), "evals_per_shift": ev, "launches": r.kernel_launches,
                                  "sectors_per_level": {int(a): int(b) for a, b in zip(*np.unique(lev, return_counts=True))}},
                    "uniform": {"wall_s": tu, "rel_err": rel(u), "evals_per_shift": npts * t.n_sectors, "N": 1 << k},
                    "difference_in_sigma": float(abs(r.coeff[-1] - u.coeff[-1]) / np.hypot(abs(r.err[-1]), abs(u.err[-1])))})
    return out


def convergence(q, wl, transform=0, k_lo=14, k_hi=20):
    """error estimate of the eps^0 coefficient of J against N over the primes below 2^k, and the
    least-squares slope of log(error) against log(N) (the paper claims "close to O(n^-1)")."""
    t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam, transform=transform)
    Ns, rels = [], []
    for N in qi.primes_below_pow2(k_lo, k_hi):
        r = q.qmc_integrate(t, N, wl.m, seed=wl.seed)
        c0, e0 = r.coeff[-1 - wl.eps_order], r.err[-1 - wl.eps_order]
        Ns.append(int(N))
        rels.append(float(max(e0.real, e0.imag) / abs(c0)))
    slope = float(np.polyfit(np.log(Ns), np.log(rels), 1)[0])
    return {"workload": wl.name, "transform": transform, "m": wl.m, "N": Ns, "rel_err_eps0": rels, "fitted_exponent": slope}


def cbc_vs_korobov(q, dev):
    """error estimate of the eps^0 coefficient with the component-by-component vector the paper names
    (host construction, timed) next to the Korobov-form vector of the P_2 search (reading C13), same N,
    shifts and kernels."""
    out = []
    for wl, N in ((qi.massless_box(), 1048573), (qi.double_box(), 262139), (qi.nonplanar_vertex(), 262139)):
        t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
        t0 = time.perf_counter()
        zc = q.qmc_cbc_vector(N, t.dim)
        t_cbc = time.perf_counter() - t0
        zk = q.qmc_generating_vector(N, t.dim, device=dev)
        sh = qi.splitmix64_shifts(wl.seed, wl.m, t.dim)
        row = {"workload": wl.name, "N": N, "m": wl.m, "cbc_construction_s": t_cbc}
        for name, z in (("cbc", zc), ("korobov", zk)):
            r = q.qmc_integrate(t, N, wl.m, z=z, shifts=sh, device=dev)
            c0, e0 = r.coeff[-1 - wl.eps_order], r.err[-1 - wl.eps_order]
            row[name] = {"z": [int(v) for v in z], "coeff_eps0": [c0.real, c0.imag],
                         "rel_err_eps0": float(max(e0.real, e0.imag) / abs(c0))}
        out.append(row)
    return out


def closed_form_check(q, dev):
    """ACTUAL deviations from known values (next to the estimated errors): the massless box through eps^0 (closed form,
    tests/test_oracle_closed_forms.py) and the three leading poles of the double box (mpmath values of the same file)."""
    out = []
    for wl, N, exact in ((qi.massless_box(), 999983, [0.666666666666667, -1.2639198230760183, -1.2238036181980894]),
                         (qi.double_box(), 999983, [2.0 / 9.0, -0.8497687147780183, 0.003001503361321066])):
        t = q.qmc_prepare(wl, eps_order=wl.eps_order)
        r = q.qmc_integrate(t, N, wl.m, seed=wl.seed, device=dev)
        k = len(exact)
        out.append({"workload": wl.name, "N": N, "m": wl.m, "orders": list(range(t.k_min, t.k_min + k)),
                    "exact": exact, "value": [float(x) for x in r.coeff.real[:k]], "estimated_err": [float(x) for x in r.err.real[:k]],
                    "deviation_in_sigma": [float(abs(v - e) / max(s, 1e-300)) for v, e, s in zip(r.coeff.real[:k], exact, r.err.real[:k])]})
    return out


def pole_extraction_comparison(q, dev):
    """SURVEY 8(f) f3 (not part of the timed path): subtraction (Eqs. 11-12) against integration by parts (Eq. 13,
    qmc_options.pole_extraction = 1), both on the generic kernel, same lattice and shifts, Eq. 21's transform: the massless box
    of config 2 (every alpha_j >= -1) and the triangle with a squared propagator (a variable with alpha_j = -2, which needs the
    p = 1 Taylor term of Eq. 11), with the ACTUAL deviation from the closed forms (massless box: tests/test_oracle_closed_forms.py;
    triangle: Dirichlet's integral 2^(-2-eps) Gamma(-1-eps) Gamma(-eps) / Gamma(-2 eps), tests/test_oracle_taylor_terms.py)."""
    import dataclasses
    tri = dataclasses.replace(qi.triangle(-2.0), nu=(1, 1, 2), eps_order=0)
    out = []
    for wl, N, exact in ((qi.massless_box(), 99991, [0.666666666666667, -1.2639198230760183, -1.2238036181980894]),
                         (tri, 99991, [0.0, 0.5, -0.8465735902799727])):
        for pe in (0, 1):
            t = q.qmc_prepare(wl, eps_order=wl.eps_order, pole_extraction=pe, nu=getattr(wl, "nu", None))
            z = q.qmc_generating_vector(N, t.dim, device=dev)
            sh = qi.splitmix64_shifts(wl.seed, 16, t.dim)
            q.qmc_integrate(t, N, 16, z=z, shifts=sh, device=dev, kernel=1)
            r = q.qmc_integrate(t, N, 16, z=z, shifts=sh, device=dev, kernel=1)
            out.append({"workload": wl.name, "nu": list(getattr(wl, "nu", None) or []), "pole_extraction": pe, "N": N, "m": 16,
                        "exact": exact, "value": [float(x) for x in r.coeff.real], "estimated_err": [float(x) for x in r.err.real],
                        "deviation_in_sigma": [float(abs(v - e) / max(s, 1e-300)) for v, e, s in zip(r.coeff.real, exact, r.err.real)],
                        "eval_kernel_ms": float(r.eval_kernel_ms)})
    return out


def strategy_comparison(q, dev):
    """SURVEY 8(f) f3 (not part of the timed path, whose config says "iterated"): the geometric decomposition strategy
    (qmc_options.strategy = 1, reading C31) against the iterated rule on the same lattice and shifts: sectors, kernel
    time of a step, error estimate of the finite part, and the difference of the two totals in units of their combined error."""
    out = []
    for wl, N in ((qi.double_box(), 999983), (qi.nonplanar_vertex(), 1048573)):
        res = []
        for st in (0, 1):
            t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam, strategy=st)
            q.qmc_integrate(t, N, wl.m, seed=wl.seed, device=dev)
            r = q.qmc_integrate(t, N, wl.m, seed=wl.seed, device=dev)
            res.append((t.n_sectors, r))
        (n0, r0), (n1, r1) = res
        comb = np.maximum(np.hypot(np.abs(r0.err.real), np.abs(r1.err.real)), 1e-300)
        out.append({"workload": wl.name, "N": N, "m": wl.m, "sectors": [n0, n1],
                    "eval_kernel_ms": [float(r0.eval_kernel_ms), float(r1.eval_kernel_ms)],
                    "err_finite_part": [float(abs(r0.err[-1].real)), float(abs(r1.err[-1].real))],
                    "difference_in_sigma": [float(x) for x in np.abs(r0.coeff.real - r1.coeff.real) / comb]})
    return out


def per_sector_mode(q, t, N, m, z, shifts, dev, torch):
    """the per-sector (parity) mode of the kernel next to the fused (throughput) mode the headline times."""
    q.qmc_integrate(t, N, m, z=z, shifts=shifts, per_sector=True, device=dev)
    r = q.qmc_integrate(t, N, m, z=z, shifts=shifts, per_sector=True, device=dev)
    f = q.qmc_integrate(t, N, m, z=z, shifts=shifts, device=dev)
    tot = r.shift_sums.sum(axis=0)
    scale = np.abs(r.shift_sums).sum(axis=0)
    return {"eval_kernel_ms": float(r.eval_kernel_ms), "fused_eval_kernel_ms": float(f.eval_kernel_ms),
            "max_rel_diff_of_totals": float(np.max(np.abs(tot - f.shift_totals) / np.maximum(scale, 1e-300)))}


def kinematic_scan(q, torch, n_points=1000, N=99991, m=16, batch=250):
    """the paper's 1000-point s-scan of the one-loop box I_A (Fig. 2).  Batched: the kinematic
    points go through qmc_prepare_batch in groups of `batch` and ONE qmc_integrate(mode=3) call per group (graph fixed,
    coefficients change); host wall clock of everything, preparation included.  `per_point_calls` = the same scan with one
    qmc_prepare + qmc_integrate per kinematic point (round 1's way)."""
    z = qi.good_vector(N, 3)
    pts = list(qi.gghh_box_scan(n_points))
    t_w = q.qmc_prepare_batch([w for _, w in pts[:8]], lam=pts[0][1].lam)
    q.qmc_integrate(t_w, N, m, z=z, seed=11, mode=3)               # module / context warm-up, not timed
    torch.cuda.synchronize()
    rel, worst, bad_contour, kernel_ms = [], (0.0, None), 0, 0.0
    t0 = time.perf_counter()
    for b0 in range(0, n_points, batch):
        grp = pts[b0:b0 + batch]
        t = q.qmc_prepare_batch([w for _, w in grp], lam=grp[0][1].lam)
        r = q.qmc_integrate(t, N, m, z=z, seed=11, mode=3)
        kernel_ms += r.kernel_ms
        bad_contour += int(r.counters[0] > 0 or r.counters[1] > 0)
        for (s_phys, _), c, e in zip(grp, r.sector_coeff[:, -1], r.sector_err[:, -1]):
            rr = max(e.real, e.imag) / abs(c)
            rel.append(rr)
            if rr > worst[0]:
                worst = (rr, s_phys)
    dt = time.perf_counter() - t0
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    n_single = min(n_points, 200)
    for s_phys, wl in pts[:n_single]:
        t = q.qmc_prepare(wl, eps_order=0, lam=wl.lam)
        q.qmc_integrate(t, N, m, z=z, seed=11)
    dt_single = (time.perf_counter() - t1) / n_single
    rel = np.array(rel)
    return {"workload": "gghh_box_scan: s in [70000, 500000], t = -6000, M_t = 172, M_H = 125 (units of M_t^2, lambda 0.5)",
            "points": n_points, "N": N, "m": m, "points_per_call": batch, "ms_per_point": dt * 1e3 / n_points, "wall_s": dt,
            "kernel_ms_per_point": kernel_ms / n_points, "per_point_calls": {"ms_per_point": dt_single * 1e3, "points": n_single},
            "rel_err_median": float(np.median(rel)), "rel_err_max": float(rel.max()), "rel_err_max_at_s": worst[1],
            "frac_rel_err_le_1e-3": float((rel <= 1e-3).mean()), "frac_rel_err_le_1e-4": float((rel <= 1e-4).mean()),
            "calls_with_contour_counter": bad_contour,
            "paper_context": "83 ms per point on one Tesla K20, relative error <= 1e-3, mostly <= 1e-4, against LoopTools (PAPER.md:206)"}


def run_product(args):
    import torch
    import torch.distributed as dist
    import paper_1508_02512_b200 as q

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the QMC hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    wl = workload(args.config)
    N = args.N or DEFAULT_N[args.config]
    m = wl.m
    t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
    geo = dict(waves=args.waves, streams=args.streams)           # launch geometry (0 = the library's defaults)
    z = q.qmc_generating_vector(N, t.dim, device=dev)           # Korobov P2 search on the device, outside the timed steps
    from paper_1508_02512_b200 import sharding
    shifts = sharding.shift_block(wl.seed, m, t.dim, rank, world)
    fp, fs, corners = q.qmc_flop_model(t)
    flops_step = (fp + fs) * N * m
    evals_step = N * m * t.n_sectors

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    gathered = torch.zeros(world, t.K, m, 2, dtype=torch.float64, device=dev)

    def step(resident):
        q.qmc_integrate_async(t, N, m, z=z, shifts=None if resident == 2 else shifts, resident=resident, device=dev, **geo)
        if world > 1:
            dist.all_gather_into_tensor(gathered, q.qmc_result_device_totals(t, m).contiguous())

    # ---- device-timed steps: inputs resident in HBM, CUDA events on the launching stream ---------------------
    step(0)
    for _ in range(max(args.warmup, 3) - 1):
        step(2)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    eval_ms = []
    torch.cuda.synchronize()
    for a, b in ev:
        flush.fill_(1)                                          # L2 flush, outside the event pair
        a.record()
        step(2)
        b.record()
        b.synchronize()
        eval_ms.append(q.qmc_result_fetch(t, m, device=dev).eval_kernel_ms)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.summary()
    ms_local = sum(a.elapsed_time(b) for a, b in ev)
    res = q.qmc_result_fetch(t, m, device=dev)
    msT = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(msT, op=dist.ReduceOp.MAX)
    ms_per_step = float(msT.item()) / args.steps
    value = evals_step * world / (ms_per_step * 1e-3)

    # ---- end to end through the public call with HOST buffers: H2D of tables + shifts, kernels, D2H, every step ----
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r_e2e = q.qmc_integrate(t, N, m, z=z, shifts=shifts, resident=0, device=dev, **geo)
        if world > 1:
            loc = torch.from_numpy(np.ascontiguousarray(r_e2e.shift_totals).view(np.float64).reshape(t.K, m, 2)).to(dev)
            sharding.combine(loc)
    torch.cuda.synchronize()
    e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e_val = evals_step * world * args.steps / float(e2e_s.item())
    h2d, d2h = r_e2e.h2d_bytes, r_e2e.d2h_bytes             # counted by the library from the copies it made

    # ---- combine the shifts of all ranks (Eqs. 19-20 over m*world estimates) --------------------------------
    if world > 1:
        coeff, err, _ = sharding.combine(q.qmc_result_device_totals(t, m))
    else:
        coeff, err = res.coeff, res.err

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (qmc_eval_kernel): plain FP64 ALU bound -----------------------------
    peak_flops, _ = q.qmc_fp64_peak(device=dev)
    mean_eval_ms = float(np.mean(eval_ms))
    achieved = flops_step / (mean_eval_ms * 1e-3) / 1e12
    nominal = 148 * 64 * 2 * 1.965e9 / 1e12
    roofline = {"bound": "alu", "kernel": EVAL_KERNEL_NOTE if not t.is_complex else EVAL_KERNEL_NOTE.replace("qmc4", "qmc5"), "achieved": achieved, "peak": peak_flops / 1e12,
                "unit": "TFLOP/s", "frac": achieved / (peak_flops / 1e12), "traffic": _traffic_from_profiles(),
                "peak_source": "DFMA chain microbenchmark (qmc_fp64_peak) measured in this run; MEASURED_PEAKS.json has no FP64 entry",
                "peak_nominal": nominal, "frac_of_nominal": achieved / nominal, "kernel_ms": mean_eval_ms,
                "kernel_share_of_step": mean_eval_ms / ms_per_step, "eval_launches_per_step": int(res.kernel_launches) - 2,
                "flops_per_point_shift": fp + fs, "corners_per_point": corners, "algorithmic_bytes_per_launch": 0}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_of(wl, N, t.n_sectors, world),
            "workload_info": {"orders": [t.k_min, t.k_max], "complex": t.is_complex, "corners_per_point": corners,
                              "m_per_gpu": m, "tables": t.describe().splitlines()[0]},
            "corner_evals_per_sec": corners * N * m * world / (ms_per_step * 1e-3),
            "result": {"coeff_re": [float(x) for x in coeff.real], "coeff_im": [float(x) for x in coeff.imag],
                       "err_re": [float(x) for x in err.real], "err_im": [float(x) for x in err.imag],
                       "counters": [int(x) for x in res.counters]},
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "note": "qmc_integrate with host buffers each step: tables + shifts H2D (pageable staging), kernels, statistics D2H, host wall clock"},
            "gpu_launches": int(res.kernel_launches) * args.steps * world, "clocks": clocks, "roofline": roofline}

    if world == 1 and not args.no_extras and args.config in LARGEST_N and N != LARGEST_N[args.config]:
        # the largest lattice BASELINE.json lists for this config: one device-timed step (inputs resident), same kernels
        NL = LARGEST_N[args.config]
        zl = q.qmc_generating_vector(NL, t.dim, device=dev)
        q.qmc_integrate_async(t, NL, m, z=zl, shifts=shifts, resident=0, device=dev, **geo)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        flush.fill_(1)
        a.record()
        q.qmc_integrate_async(t, NL, m, z=zl, resident=2, device=dev, **geo)
        b.record()
        b.synchronize()
        rl = q.qmc_result_fetch(t, m, device=dev)
        msl = a.elapsed_time(b)
        line["largest_size"] = {"N": NL, "steps": 1, "ms_per_step": msl, "value": NL * m * t.n_sectors / (msl * 1e-3), "unit": UNIT,
                                "roofline_frac": (fp + fs) * NL * m / (rl.eval_kernel_ms * 1e-3) / peak_flops,
                                "coeff_re": [float(x) for x in rl.coeff.real], "err_re": [float(x) for x in rl.err.real]}
    if world == 1 and not args.no_extras:
        line["closed_form_check"] = closed_form_check(q, dev)
        z_o = test_vector(N, wl.dim)
        v, cores, desc = oracle_sample(wl, N, z_o, qi.splitmix64_shifts(wl.seed, m, wl.dim), 15.0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                "single_thread_value": oracle_sample.single_thread}
        def extra(fn, *a, **k):       # the context numbers must not take the headline line down with them
            try:
                return fn(*a, **k)
            except Exception as e:    # noqa: BLE001
                return {"error": f"{type(e).__name__}: {e}"}
        # M2 on the two-loop configs, then on the paper's own two-loop integrals of the physical region
        # (Tables 2-3: 19 s and 20 s on a K20)
        line["time_to_1e-3"] = [extra(time_to_accuracy, q, w, torch)
                                for w in (qi.double_box(), qi.nonplanar_vertex(), qi.paper_IC(), qi.paper_ID())]
        # transform 0 = the paper's Eq. 21; transform 2 = the next member of its family (reading C20)
        line["time_to_1e-5"] = [extra(time_to_accuracy, q, w, torch, target=1e-5, max_N=2 ** 24, transform=tr)
                                for w in (qi.double_box(), qi.nonplanar_vertex()) for tr in (0, 2)]
        line["time_to_1e-6"] = [extra(time_to_accuracy, q, w, torch, target=1e-6, max_N=2 ** 24, transform=tr)
                                for w, tr in ((qi.nonplanar_vertex(), 0), (qi.nonplanar_vertex(), 2), (qi.double_box(), 2))]
        line["time_to_1e-5_embedded"] = [extra(time_to_accuracy_embedded, q, w, torch, target=1e-5, transform=tr)
                                         for w in (qi.double_box(), qi.nonplanar_vertex()) for tr in (0, 2)]
        line["allocation_vs_uniform"] = extra(allocation_vs_uniform, q, torch)
        line["convergence"] = [extra(convergence, q, w, tr) for w in (qi.massless_box(), qi.double_box(), qi.nonplanar_vertex())
                               for tr in (0, 2)]
        line["cbc_vs_korobov"] = extra(cbc_vs_korobov, q, dev)
        line["per_sector_mode"] = extra(per_sector_mode, q, t, min(N, 999983), m, q.qmc_generating_vector(min(N, 999983), t.dim, device=dev), shifts, dev, torch)
        line["other_workloads"] = extra(other_workloads, q, torch, dev, args.config)
        line["kinematic_scan"] = extra(kinematic_scan, q, torch)
        line["pole_extraction"] = extra(pole_extraction_comparison, q, dev)
        line["strategy_comparison"] = extra(strategy_comparison, q, dev)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


EVAL_KERNEL_NOTE = ("qmc4_eval_kernel: one launch per run of sectors, overlapped on side streams; duration = CUDA events around "
                    "the whole set on the launching stream, flops = all launches of the step")


def _traffic_from_profiles():
    """DRAM bytes per launch of the evaluation kernel from the committed `ncu --set full` capture (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", "eval_kernel_traffic.json")
    try:
        with open(p) as f:
            return json.load(f).get("dram_bytes_per_launch")
    except Exception:
        return None


def other_workloads(q, torch, dev, skip_cfg):
    """Device-timed throughput of the other multi-sector configs (context; the headline is `value`)."""
    out = []
    for cfg in (2, 3, 4, 5):
        if cfg == skip_cfg:
            continue
        wl = workload(cfg)
        N = DEFAULT_N[cfg]
        t = q.qmc_prepare(wl, eps_order=wl.eps_order, lam=wl.lam)
        z = q.qmc_generating_vector(N, t.dim, device=dev)
        q.qmc_integrate_async(t, N, wl.m, seed=wl.seed, z=z, resident=0, device=dev)
        q.qmc_integrate_async(t, N, wl.m, seed=wl.seed, z=z, resident=2, device=dev)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 3
        a.record()
        for _ in range(reps):
            q.qmc_integrate_async(t, N, wl.m, seed=wl.seed, z=z, resident=2, device=dev)
        b.record()
        b.synchronize()
        ms = a.elapsed_time(b) / reps
        r = q.qmc_result_fetch(t, wl.m, device=dev)
        fp, fs, corners = q.qmc_flop_model(t)
        out.append({"workload": wl.name, "N": N, "m": wl.m, "n_sectors": t.n_sectors, "ms_per_step": ms,
                    "evals_per_sec": N * wl.m * t.n_sectors / (ms * 1e-3),
                    "corner_evals_per_sec": N * wl.m * corners / (ms * 1e-3),
                    "tflops": (fp + fs) * N * wl.m / (r.eval_kernel_ms * 1e-3) / 1e12,
                    "coeff_eps0": [float(r.coeff[-1 - wl.eps_order].real), float(r.coeff[-1 - wl.eps_order].imag)],
                    "err_eps0": [float(r.err[-1 - wl.eps_order].real), float(r.err[-1 - wl.eps_order].imag)]})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config (1-based); default 4 = two-loop planar double box, 293 sectors")
    ap.add_argument("--N", type=int, default=0, help="lattice size (prime); default: DEFAULT_N[config]")
    ap.add_argument("--impl", default="product", choices=["product", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip cpu_baseline, time-to-accuracy and other workloads")
    ap.add_argument("--waves", type=int, default=0, help="qmc_run.waves: blocks per resident block slot over a step (0 = library default 16)")
    ap.add_argument("--streams", type=int, default=0, help="qmc_run.streams: side streams of a step (0 = default 4, -1 = none: launches in order)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_product(args)


if __name__ == "__main__":
    main()
