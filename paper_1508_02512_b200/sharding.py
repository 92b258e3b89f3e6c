"""Multi-GPU plumbing of the path.  Two ways to shard, both without any exchange inside the evaluation:
(1) by SHIFT VECTORS (weak scaling, what bench.py --gpus N times): gather per-shift totals, Eqs. 19-20 over all of them;
(2) by contiguous LATTICE-INDEX ranges (SURVEY 8(e), strong scaling): index_block + one all_reduce(SUM), at the end.

Every (lattice point, shift, sector) evaluation is independent (Eq. 18), so rank r of W integrates rows
[r*m, (r+1)*m) of the ONE SplitMix64 stream of m*W shift vectors: a W-GPU run is the same estimator as a 1-GPU run with
m*W shifts.  The only exchange is an all_gather of the per-shift totals ([K][m] complex per rank).  torch.distributed
carries it (NCCL on GPUs, gloo in the CPU tests); the statistics run in the C library (qmc_statistics).
"""
from __future__ import annotations

import numpy as np

from .binding import qmc_shifts, qmc_statistics


def shift_block(seed: int, m: int, dim: int, rank: int, world: int) -> np.ndarray:
    """Rows [rank*m, (rank+1)*m) of the stream of m*world shift vectors keyed by `seed` (library generator)."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return qmc_shifts(seed, m * world, dim)[rank * m:(rank + 1) * m].copy()


def gather_shift_totals(local_totals, group=None):
    """all_gather of per-shift totals.  `local_totals`: torch tensor [K, m, 2] float64 (any device the backend of
    `group` supports) or numpy complex [K, m].  Returns numpy complex [K, m*world], ranks in order."""
    import torch
    import torch.distributed as dist
    if isinstance(local_totals, np.ndarray):
        local_totals = torch.from_numpy(np.ascontiguousarray(local_totals, dtype=np.complex128).view(np.float64)
                                        .reshape(local_totals.shape[0], local_totals.shape[1], 2))
    x = local_totals.contiguous()
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    if world == 1:
        g = x.unsqueeze(0)
    else:
        parts = [torch.empty_like(x) for _ in range(world)]
        dist.all_gather(parts, x, group=group)
        g = torch.stack(parts)
    a = g.cpu().numpy()                                      # [world, K, m, 2]
    T = np.concatenate([a[r] for r in range(a.shape[0])], axis=1)
    return T[..., 0] + 1j * T[..., 1]


def combine(local_totals, group=None):
    """Laurent coefficients and errors over the shifts of all ranks: (coeff[K], err[K], totals[K, m*world])."""
    T = gather_shift_totals(local_totals, group)
    coeff, err = qmc_statistics(T)
    return coeff, err, T


# ---- contiguous lattice-index ranges per rank (strong scaling: the total work is fixed) -------------------

def index_block(N: int, rank: int, world: int):
    """Lattice indices [begin, begin + count) of rank `rank` of `world`: contiguous, balanced to one index, covering
    0..N-1 exactly once.  Returns (index_begin, index_step, index_count) for qmc_run / qmc_integrate(index_range=...).
    The kernels always normalise by 1/N (Eq. 18), so the per-rank results ADD to the full-lattice result."""
    if not (0 <= rank < world) or world > N:
        raise ValueError("rank out of range or more ranks than lattice points")
    base, extra = divmod(N, world)
    begin = rank * base + min(rank, extra)
    return begin, 1, base + (1 if rank < extra else 0)


def reduce_index_blocks(local_totals, group=None):
    """Sum over ranks of the per-shift totals of their index blocks: one all_reduce(SUM) of [K][m][2] doubles (the only
    exchange of the path), then Eqs. 19-20.  `local_totals`: torch tensor [K, m, 2] float64 or numpy complex [K, m].
    Returns (coeff[K], err[K], totals[K, m]) -- the same on every rank."""
    import torch
    import torch.distributed as dist
    if isinstance(local_totals, np.ndarray):
        local_totals = torch.from_numpy(np.ascontiguousarray(local_totals, dtype=np.complex128).view(np.float64)
                                        .reshape(local_totals.shape[0], local_totals.shape[1], 2))
    x = local_totals.contiguous().clone()
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(x, op=dist.ReduceOp.SUM, group=group)
    a = x.cpu().numpy()
    T = a[..., 0] + 1j * a[..., 1]
    coeff, err = qmc_statistics(T)
    return coeff, err, T
