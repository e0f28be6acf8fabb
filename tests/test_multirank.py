"""N > 1 path of bench.py on CPU: 2 processes, gloo.  The composition shards by independent problems (one
seeded pair per rank, no data-path collective); only the timing/throughput reduction crosses ranks."""
from __future__ import annotations

import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank: int, world: int, port: int, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        t_ms, arcs = 100.0 + 50.0 * rank, 1000.0 * (rank + 1)
        (tmax,), (asum, lsum) = bench.reduce_over_ranks(dist, world, [t_ms], [arcs, 7], "cpu")
        q.put((rank, tmax, asum, lsum, bench.rank_seeds("tiny", rank)))
    finally:
        dist.destroy_process_group()


def test_two_rank_reduction_and_seed_sharding():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, tmax, asum, lsum, seeds in out:
        assert tmax == 150.0 and asum == 3000.0 and lsum == 14.0       # max of times, sum of units
        assert seeds == (102 + 1000 * rank, 103 + 1000 * rank)          # distinct problems per rank
    # whole-job value = units of all ranks / max time
    assert out[0][2] / (out[0][1] * 1e-3) == pytest.approx(20000.0)


def test_single_rank_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(None, 1, [3.5], [2, 9], "cpu") == ([3.5], [2.0, 9.0])
