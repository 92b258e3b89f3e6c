"""world_size-2 gloo tests (CPU) of the multi-GPU plumbing: shift-vector sharding, gather order, statistics over all
shifts.  The evaluation itself needs a GPU; here each rank fabricates its per-shift totals as a deterministic function
of its OWN shift block, so a wrong block, a wrong gather order or a wrong combination changes the result."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import qmc_inputs as qi
from paper_1508_02512_b200 import sharding
import paper_1508_02512_b200 as q

K, M, DIM, SEED = 3, 4, 5, 17


def fake_totals(block):          # [m, dim] -> [K, m] complex, injective enough in the shift values
    k = np.arange(1, K + 1)[:, None]
    return (block.sum(axis=1)[None, :] ** k) + 1j * (block[:, 0][None, :] * k)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        block = sharding.shift_block(SEED, M, DIM, rank, world)
        coeff, err, T = sharding.combine(fake_totals(block))
        torch.save({"block": block, "coeff": coeff, "err": err, "T": T}, os.path.join(out, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_shift_sharding_gather_and_statistics_world2(tmp_path):
    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    res = [torch.load(os.path.join(str(tmp_path), f"r{r}.pt"), weights_only=False) for r in range(world)]
    full = qi.splitmix64_shifts(SEED, M * world, DIM)            # the ONE stream, from the independent generator
    for r in range(world):
        assert np.array_equal(res[r]["block"], full[r * M:(r + 1) * M])
    T_want = fake_totals(full)                                   # what a single rank with m*world shifts would hold
    for r in range(world):
        assert np.array_equal(res[r]["T"], T_want)               # gather order = rank order, bit-exact
        mean = T_want.mean(axis=1)
        err_re = T_want.real.std(axis=1, ddof=1) / np.sqrt(M * world)
        err_im = T_want.imag.std(axis=1, ddof=1) / np.sqrt(M * world)
        assert np.allclose(res[r]["coeff"], mean, rtol=1e-14)
        assert np.allclose(res[r]["err"].real, err_re, rtol=1e-12) and np.allclose(res[r]["err"].imag, err_im, rtol=1e-12)
    assert np.array_equal(res[0]["coeff"], res[1]["coeff"])      # every rank holds the same answer


def test_single_process_path_and_argument_checks():
    b = sharding.shift_block(SEED, M, DIM, 0, 1)
    assert np.array_equal(b, qi.splitmix64_shifts(SEED, M, DIM))
    coeff, err, T = sharding.combine(fake_totals(b))             # no process group: world = 1
    assert T.shape == (K, M) and np.allclose(coeff, fake_totals(b).mean(axis=1))
    try:
        sharding.shift_block(SEED, M, DIM, 2, 2)
        assert False
    except ValueError:
        pass
    c2, e2 = q.qmc_statistics(T)
    assert np.array_equal(c2, coeff) and np.array_equal(e2, err)


# ---- contiguous lattice-index ranges, one all_reduce(SUM) ---------------------------------------------------

def fake_index_totals(N, begin, count):
    """Per-shift totals a rank would hold for its index block: (1/N) sum over its indices of a function of (index, shift,
    order) -- additive over blocks like the kernels' sums (Eq. 18)."""
    i = np.arange(begin, begin + count, dtype=np.float64)[None, None, :]
    k = np.arange(1, K + 1, dtype=np.float64)[:, None, None]
    kap = np.arange(M, dtype=np.float64)[None, :, None]
    return (np.cos(0.001 * i * k + kap) + 1j * np.sin(0.002 * i + k * kap)).sum(axis=2) / N


def _index_worker(rank, world, port, out, N):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        b, step, c = sharding.index_block(N, rank, world)
        coeff, err, T = sharding.reduce_index_blocks(fake_index_totals(N, b, c))
        torch.save({"block": (b, step, c), "coeff": coeff, "err": err, "T": T}, os.path.join(out, f"i{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_index_range_sharding_allreduce_world2(tmp_path):
    world, N = 2, 10007
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_index_worker, args=(world, port, str(tmp_path), N), nprocs=world, join=True)
    res = [torch.load(os.path.join(str(tmp_path), f"i{r}.pt"), weights_only=False) for r in range(world)]
    # the blocks tile 0..N-1 exactly once, contiguous, balanced to one index
    assert res[0]["block"] == (0, 1, 5004) and res[1]["block"] == (5004, 1, 5003)
    want = fake_index_totals(N, 0, N)                              # what one rank over the whole lattice would hold
    for r in range(world):
        assert np.allclose(res[r]["T"], want, rtol=1e-12, atol=1e-15)   # the two half-sums add to the single-rank totals
        c, e = q.qmc_statistics(res[r]["T"])
        assert np.array_equal(c, res[r]["coeff"]) and np.array_equal(e, res[r]["err"])
    assert np.array_equal(res[0]["T"], res[1]["T"])                # every rank holds the same answer


def test_index_blocks_tile_the_lattice():
    for N, world in ((10007, 1), (10007, 3), (99991, 8), (16, 16)):
        blocks = [sharding.index_block(N, r, world) for r in range(world)]
        assert blocks[0][0] == 0 and sum(b[2] for b in blocks) == N
        for a, b in zip(blocks, blocks[1:]):
            assert a[0] + a[2] == b[0] and 0 <= a[2] - b[2] <= 1
    try:
        sharding.index_block(4, 0, 5)
        assert False
    except ValueError:
        pass
