"""N>1 host logic on CPU: world_size-2 gloo run of the batch sharding used by bench.py --gpus N.
The per-rank 'outputs' here are a stand-in function of the external index (the integrators need a GPU); what is
tested is the partition (disjoint, covering, balanced) and the all-gather epilogue."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2412_13043_b200.shard import gather_blocks, shard_bounds


def test_shard_bounds_partition():
    for n in (0, 1, 5, 64, 129, 8192):
        for w in (1, 2, 3, 8):
            b = [shard_bounds(n, w, r) for r in range(w)]
            assert b[0][0] == 0 and b[-1][1] == n
            assert all(b[r][1] == b[r + 1][0] for r in range(w - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard_bounds(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_ext, n_field, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lo, hi = shard_bounds(n_ext, world, rank)
        e = torch.arange(lo, hi, dtype=torch.float64)[:, None]
        f = torch.arange(n_field, dtype=torch.float64)[None, :]
        local = torch.sin(0.37 * e) + 1e-3 * f * e           # stand-in for out[e][f] of this rank's block
        full = gather_blocks(local, n_ext, dist)
        t = torch.tensor([float(hi - lo)])                   # bench.py's max-over-ranks of the step time
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        q.put((rank, lo, hi, full.numpy(), float(t.item())))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_ext", [64, 7])
def test_two_rank_gloo_gather_matches_unsharded(n_ext):
    world, n_field = 2, 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_ext, n_field, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    e = np.arange(n_ext, dtype=np.float64)[:, None]
    f = np.arange(n_field, dtype=np.float64)[None, :]
    ref = np.sin(0.37 * e) + 1e-3 * f * e
    covered = np.zeros(n_ext, dtype=int)
    for rank, lo, hi, full, tmax in got:
        assert np.array_equal(full, ref)
        covered[lo:hi] += 1
        assert tmax == float(max(h - l for _, l, h, _, _ in got))
    assert np.all(covered == 1)
