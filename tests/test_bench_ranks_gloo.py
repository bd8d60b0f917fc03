"""bench.py's own multi-rank logic (not a stand-in): the functions its main() calls to read the launcher's environment,
cut this rank's share of the global batch, take the MAX of the step time over ranks and form the whole-job rate, driven at
world_size 2 on gloo / CPU; and the launcher behind `python bench.py --gpus N`, which must refuse to run fewer ranks than
asked."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

import bench
from paper_2412_13043_b200 import inputs
from paper_2412_13043_b200.shard import shard_bounds

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    r, w, local = bench.rank_env(world)
    dist.init_process_group("gloo", rank=r, world_size=w)
    try:
        c = bench.rank_workload(inputs, shard_bounds, w, r)
        ms_local = 1.5 + 0.5 * r                                   # rank 1 is the slow one
        ms = bench.max_over_ranks(ms_local, dist, "cpu")
        q.put((r, w, local, c["pext_global_range"], c["pext"].copy(), ms, bench.whole_job_rate(w, 1000, ms)))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_bench_shard_and_max_reduce():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=120) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    full = inputs.config4(n_p=64 * world)["pext"]                 # the global batch: 64 momenta per rank
    assert full.size == 128
    for r, (rank, w, local, (lo, hi), pext, ms, rate) in enumerate(got):
        assert (rank, w, local) == (r, world, r)
        assert (lo, hi) == (64 * r, 64 * (r + 1))                   # contiguous, disjoint, covering
        assert np.array_equal(pext, full[lo:hi])
        assert ms == 2.0                                            # the MAX over ranks, on every rank
        assert rate == world * 1000 / 2.0e-3                        # whole-job units per second
    # one process, no launcher: rank 0 of 1, the unsharded BASELINE.json config
    assert bench.max_over_ranks(1.25, None, "cpu") == 1.25
    c1 = bench.rank_workload(inputs, shard_bounds, 1, 0)
    assert np.array_equal(c1["pext"], inputs.config4()["pext"])


def test_rank_env_rejects_a_world_that_differs_from_gpus(monkeypatch):
    monkeypatch.setenv("RANK", "0")
    monkeypatch.setenv("WORLD_SIZE", "1")
    assert bench.rank_env(1) == (0, 1, 0)
    with pytest.raises(SystemExit):
        bench.rank_env(2)                                           # --gpus 2 but one rank: never silently run one GPU
    monkeypatch.setenv("RANK", "3")
    with pytest.raises(SystemExit):
        bench.rank_env(1)


def test_bench_gpus_n_refuses_to_run_with_fewer_devices():
    # this container has no GPU: `python bench.py --gpus 2` must fail loudly, not print a one-GPU line
    import torch
    if torch.cuda.device_count() >= 2:
        pytest.skip("two GPUs visible: the launcher would run")
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0
    assert "--gpus 2" in r.stderr and "visible" in r.stderr
    assert not r.stdout.strip()
