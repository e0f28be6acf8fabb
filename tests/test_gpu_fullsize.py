"""Full-size parity (`-m gpu`): BASELINE.json's configs at their stated sizes, in the launch configuration
bench.py times.  The oracle cannot hold 1e9 arcs, so each config is checked three ways:

  1. exact element-by-element parity with the oracle on the FULL-SIZE inputs under a smaller budget the oracle
     finishes in seconds (rule T makes that a well-defined prefix of the same search);
  2. at the bench budget: sampled sources — every outgoing arc of a sampled expanded state must equal the
     oracle's one-pair expansion (definition) of that (q1,q2), structure exact, weights rtol 1e-5;
  3. at the bench budget: properties that hold at any size (unique states, arcs sorted by source, every state but
     the start has an incoming arc, unexpanded states have no arcs, counters consistent, accept set exact).
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1805_06383_b200 import workloads
from test_gpu_parity import check_parity

pytestmark = pytest.mark.gpu
RTOL = 1e-5


@pytest.fixture(scope="module")
def fstc():
    import torch
    assert torch.cuda.is_available()
    from paper_1805_06383_b200 import fstc as mod
    mod.lib()
    return mod


def _properties_and_samples(fstc, m1, m2, res, n_samples=300, seed=0):
    import torch
    nq2 = m2.n_states
    ns, na = res.n_states, res.n_arcs
    pair = res.pair.long()
    key = pair[:, 0] * nq2 + pair[:, 1]
    # --- unique states, state 0 = start pair, ids in range
    assert pair[0].tolist() == [m1.start, m2.start]
    sk = torch.sort(key).values
    assert bool((sk[1:] != sk[:-1]).all())
    del sk
    assert int(pair[:, 0].min()) >= 0 and int(pair[:, 0].max()) < m1.n_states
    assert int(pair[:, 1].min()) >= 0 and int(pair[:, 1].max()) < m2.n_states
    # --- arcs sorted by source, targets in range, every non-start state has an incoming arc
    indeg = torch.zeros(ns, dtype=torch.int32, device="cuda")
    outdeg = torch.zeros(ns, dtype=torch.int64, device="cuda")
    step = 1 << 27
    prev_last = -1
    for lo in range(0, na, step):
        s = res.src[lo:lo + step]
        t = res.tgt[lo:lo + step]
        assert int(s[0]) >= prev_last and bool((s[1:] >= s[:-1]).all())
        prev_last = int(s[-1])
        assert int(t.min()) >= 0 and int(t.max()) < ns
        indeg.index_put_((t.long(),), torch.ones_like(t), accumulate=True)
        outdeg += torch.bincount(s.long(), minlength=ns)
    assert bool((indeg[1:] > 0).all())
    expanded = res.expanded.bool()
    assert int(expanded.sum()) == res.n_expanded
    assert bool((outdeg[~expanded] == 0).all())                       # unexpanded states carry no arcs
    assert int(outdeg.sum()) == na
    # --- accept set: exactly the states with q1 in F1 and q2 in F2, ascending
    f1 = torch.zeros(m1.n_states, dtype=torch.bool, device="cuda"); f1[torch.from_numpy(m1.accept).long().cuda()] = True
    f2 = torch.zeros(m2.n_states, dtype=torch.bool, device="cuda"); f2[torch.from_numpy(m2.accept).long().cuda()] = True
    want = torch.nonzero(f1[pair[:, 0]] & f2[pair[:, 1]]).flatten()
    assert want.numel() == res.n_accept and bool((want == res.accept.long()).all())
    # --- sampled sources against the oracle's one-pair expansion
    x = oracle.PairExpander(m1, m2)
    rng = np.random.default_rng(seed)
    exp_ids = torch.nonzero(expanded).flatten()
    pick = exp_ids[torch.from_numpy(rng.integers(0, exp_ids.numel(), n_samples)).cuda()]
    pick = torch.unique(torch.cat([pick, exp_ids[:3], exp_ids[-3:]]))
    lo = torch.searchsorted(res.src, pick.int())
    hi = torch.searchsorted(res.src, pick.int(), right=True)
    raw_sum = 0
    for sid, a, b in zip(pick.tolist(), lo.tolist(), hi.tolist()):
        q1, q2 = pair[sid].tolist()
        r1, r2, sa, sb, w = x.expand(q1, q2, merge=True)
        raw_sum += x.raw_count(q1, q2)
        assert int(outdeg[sid]) == b - a == len(w), (sid, q1, q2)
        tp = pair[res.tgt[a:b].long()].cpu().numpy()
        got = np.stack([tp[:, 0], tp[:, 1], res.ilabel[a:b].cpu().numpy(), res.olabel[a:b].cpu().numpy()], 1).astype(np.int64)
        gw = res.weight[a:b].cpu().numpy()
        o = np.lexsort((got[:, 3], got[:, 2], got[:, 1], got[:, 0]))
        ref = np.stack([r1, r2, sa, sb], 1).astype(np.int64)
        assert (got[o] == ref).all(), (sid, q1, q2)
        np.testing.assert_allclose(gw[o], w, rtol=RTOL, atol=0)
    assert raw_sum > 0
    x.close()


def test_large_full_size_inputs_small_budget_exact(fstc):
    m1, m2 = workloads.make_config("large")
    check_parity(fstc, m1, m2, max_raw_arcs=3_000_000)


def test_large_bench_budget_properties_and_samples(fstc):
    m1, m2 = workloads.make_config("large")
    budget = workloads.CONFIGS["large"]["max_raw_arcs"]
    res = fstc.fstc_compose(fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2), max_raw_arcs=budget)
    assert res.truncated == 1 and res.n_raw_arcs <= budget and res.n_raw_arcs > 0.99 * budget
    assert res.n_arcs == res.n_raw_arcs                                 # no source of this config can merge
    st = res.stats
    assert sum(st["level_raw"]) == res.n_raw_arcs and 1 + sum(st["level_new_states"]) == res.n_states
    # complete levels agree with the oracle run under the small budget (same search prefix)
    ref = oracle.compose(m1, m2, max_raw_arcs=3_000_000, keep_arcs=False)
    full_levels = ref.n_levels - 1
    assert st["level_raw"][:full_levels] == [int(v) for v in ref.level_raw[:full_levels]]
    assert st["level_frontier"][:ref.n_levels] == [int(v) for v in ref.level_size]
    _properties_and_samples(fstc, m1, m2, res)


def test_medium_full_size_inputs_small_budget_exact(fstc):
    m1, m2 = workloads.make_config("medium")
    check_parity(fstc, m1, m2, max_raw_arcs=5_000_000)


def test_medium_complete_properties_and_samples(fstc):
    """The heaviest COMPLETE composition.  Expected totals: tests/golden/medium_totals.json, written by
    tests/golden/make_medium_totals.py (the CPU oracle on the same seeded inputs, ~4 min on one core)."""
    import json
    import os
    want = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "medium_totals.json")))
    m1, m2 = workloads.make_config("medium")
    res = fstc.fstc_compose(fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2))
    assert (res.n_states, res.n_arcs, res.n_raw_arcs, res.n_levels, res.truncated) == \
           (want["n_states"], want["n_arcs"], want["n_raw_arcs"], want["n_levels"], want["truncated"])
    assert res.stats["level_raw"] == want["level_raw"]
    assert res.stats["level_frontier"] == want["level_size"]
    assert res.n_expanded == res.n_states == want["n_expanded"]
    _properties_and_samples(fstc, m1, m2, res)


def test_skewed_full_size_inputs_small_budget_exact(fstc):
    m1, m2 = workloads.make_config("skewed")
    res, ref = check_parity(fstc, m1, m2, max_raw_arcs=3_000_000)
    assert ref.n_arcs < ref.n_raw_arcs                                  # merges happen


def test_skewed_bench_budget_properties_and_samples(fstc):
    m1, m2 = workloads.make_config("skewed")
    budget = workloads.CONFIGS["skewed"]["max_raw_arcs"]
    res = fstc.fstc_compose(fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2), max_raw_arcs=budget)
    assert res.truncated == 1 and res.n_raw_arcs <= budget and res.n_arcs < res.n_raw_arcs
    assert res.stats["n_raw_sorted"] + res.stats["n_raw_grouped"] > 0.5 * res.n_raw_arcs
    _properties_and_samples(fstc, m1, m2, res, n_samples=60)


def test_nlp_full_size_exact(fstc):
    m1, m2 = workloads.make_config("nlp")
    res, ref = check_parity(fstc, m1, m2)
    assert ref.n_levels == 51


@pytest.mark.parametrize("margin", ["0.02", "0.3", "40"])
def test_cut_level_key_limit_is_exact_whatever_the_guess(fstc, margin):
    """A level that rule T will cut is counted only below a guessed key limit (1.5 x the predicted cut).  The guess must
    not matter: far too low (the level is recounted with a 4x wider limit, several times), too low, far too high."""
    import os
    m1, m2 = workloads.make_config("large", scale=0.1)
    os.environ["FSTC_KEY_LIMIT_MARGIN"] = margin
    try:
        res, ref = check_parity(fstc, m1, m2, max_raw_arcs=2_000_000)
    finally:
        del os.environ["FSTC_KEY_LIMIT_MARGIN"]
    assert res.truncated == 1 and ref.level_size[-1] > 100_000       # the cut level is big enough to be compacted
