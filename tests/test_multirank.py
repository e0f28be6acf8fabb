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


# ---------------------------------------------------------------------------------------------------------------------
# One composition sharded by ownership of the pair keys (paper_1805_06383_b200/sharded.py): the exchange
# logic on CPU tensors over gloo.  The per-rank expansion, which is the CUDA library's job on a GPU, is done here by the
# oracle's one-pair expander, so that what is tested is exactly the part that crosses ranks: key -> owner, the all-to-all,
# find-or-create at the owner, global ids back, the owned frontier, the joint end of the search.
def _sharded_worker(rank: int, world: int, port: int, q, config: str, scale: float, max_levels: int):
    import numpy as np
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1805_06383_b200 import workloads
    from paper_1805_06383_b200.sharded import KeyExchange
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m1, m2 = workloads.make_config(config, scale=scale)
        q2_bits = max(1, int(m2.n_states - 1).bit_length())
        x = oracle.PairExpander(m1, m2)
        ex = KeyExchange(rank, world, "cpu")
        start_key = (int(m1.start) << q2_bits) | int(m2.start)
        pairs = []                                                # this rank's states, local id order
        if ex.owns(start_key):
            ex.insert_start(start_key)
            pairs.append((int(m1.start), int(m2.start)))
        arcs = []                                                 # (local src, global tgt, a, b, w)
        f_lo, level = 0, 0
        while True:
            if max_levels and level == max_levels:
                break
            f_hi = len(pairs)
            keys, meta = [], []
            for sid in range(f_lo, f_hi):
                r1, r2, a, b, w = x.expand(*pairs[sid], merge=True)
                keys.append((r1.astype(np.int64) << q2_bits) | r2.astype(np.int64))
                meta.append((np.full(len(w), sid), a, b, w))
            k = torch.from_numpy(np.concatenate(keys)) if keys else torch.empty(0, dtype=torch.int64)
            # three exchanges per level, like the library (classes F, G, U): two of them empty here
            created = False
            for call in range(3):
                gids, new_keys = ex.resolve(k if call == 2 else torch.empty(0, dtype=torch.int64))
                created = created or new_keys.numel() > 0
                for nk in new_keys.tolist():
                    pairs.append((nk >> q2_bits, nk & ((1 << q2_bits) - 1)))
            if meta:
                src = np.concatenate([m[0] for m in meta])
                arcs.append((src, gids.numpy(), np.concatenate([m[1] for m in meta]), np.concatenate([m[2] for m in meta]),
                             np.concatenate([m[3] for m in meta])))
            f_lo = f_hi
            level += 1
            if not ex.any_rank(created):
                break
        assert ex.n_local == len(pairs)
        cat = lambda i, dt: np.concatenate([a[i] for a in arcs]).astype(dt) if arcs else np.empty(0, dt)
        q.put((rank, np.array(pairs, np.int64).reshape(-1, 2), cat(0, np.int64), cat(1, np.int64), cat(2, np.int64),
               cat(3, np.int64), cat(4, np.float64), level, ex.exchanged_keys))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,config,scale,max_levels", [(2, "tiny", 1.0, 0), (3, "tiny", 1.0, 0), (2, "medium", 0.004, 0),
                                                           (2, "tiny", 1.0, 5)])
def test_sharded_composition_equals_the_oracle(world, config, scale, max_levels):
    import numpy as np
    import torch.multiprocessing as mp
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1805_06383_b200 import workloads
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + (os.getpid() * 7 + world * 13 + max_levels) % 2000
    procs = [ctx.Process(target=_sharded_worker, args=(r, world, port, q, config, scale, max_levels)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    m1, m2 = workloads.make_config(config, scale=scale)
    ref = oracle.compose(m1, m2, merge=True, max_levels=max_levels)
    nq2 = m2.n_states
    # global id -> pair key: local state i of rank r is global i * world + r
    key_of = {}
    for rank, pairs, *_ in out:
        for i, (a, b) in enumerate(pairs.tolist()):
            key_of[i * world + rank] = a * nq2 + b
    assert len(set(key_of.values())) == len(key_of) == ref.n_states                 # every state owned exactly once
    assert sorted(key_of.values()) == sorted(ref.state_keys().tolist())
    assert all(len(t[1]) > 0 for t in out)                                          # the work really was split
    got = []
    for rank, pairs, src, tgt, a, b, w, level, moved in out:
        assert level == out[0][7]                                                   # all ranks stop at the same level
        ks = np.array([key_of[int(s) * world + rank] for s in src], np.int64)
        kt = np.array([key_of[int(t)] for t in tgt], np.int64)
        got.append(np.stack([ks, kt, a, b], 1))
    got = np.concatenate(got)
    gw = np.concatenate([t[6] for t in out])
    o = np.lexsort((got[:, 3], got[:, 2], got[:, 1], got[:, 0]))
    rk = ref.state_keys()
    rt = np.stack([rk[ref.src], rk[ref.tgt], ref.ilabel.astype(np.int64), ref.olabel.astype(np.int64)], 1)
    ro = np.lexsort((rt[:, 3], rt[:, 2], rt[:, 1], rt[:, 0]))
    assert got.shape == rt.shape and (got[o] == rt[ro]).all()
    np.testing.assert_allclose(gw[o], ref.weight[ro], rtol=1e-12)
    assert sum(t[8] for t in out) > 0                                               # keys did cross ranks
