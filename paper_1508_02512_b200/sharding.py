"""Multi-GPU plumbing of the path: shard by SHIFT VECTORS, gather per-shift totals, Eqs. 19-20 over all of them.

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
