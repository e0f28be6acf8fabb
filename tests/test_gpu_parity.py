"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on the same
seeded inputs.  Structure bit-exact after canonical sorting by pair key / arc key; weights within
rtol 1e-5 of the oracle's fp64 sums (BASELINE.json north_star).  `-m gpu`."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1805_06383_b200 import workloads
from helpers import canon_arc_table, fst_from_arcs, messy_random_fst

pytestmark = pytest.mark.gpu

RTOL = 1e-5   # fp32 products and fp32 sums vs exact fp64 (north_star); positive weights, no cancellation


@pytest.fixture(scope="module")
def fstc():
    import torch
    assert torch.cuda.is_available()
    from paper_1805_06383_b200 import fstc as mod
    mod.lib()                          # fails loudly if the CUDA library is missing
    return mod


def gpu_tables(res, n_q2):
    pair = res.pair.cpu().numpy().astype(np.int64)
    q1, q2 = pair[:, 0], pair[:, 1]
    tab, w = canon_arc_table(q1, q2, res.src.cpu().numpy(), res.tgt.cpu().numpy(), res.ilabel.cpu().numpy(),
                             res.olabel.cpu().numpy(), res.weight.cpu().numpy(), n_q2)
    keys = q1 * n_q2 + q2
    return keys, tab, w


def check_parity(fstc, m1, m2, *, merge_mode=0, max_raw_arcs=0, max_levels=0, device_inputs=True, resolve_mode=0, small_path=1,
                 result=None):
    """small_path: 1 (default here) = the level-synchronous path of compose.cu, so that small test inputs still exercise
    it; tests/test_gpu_small.py passes 2 (one-block path only) and 0 (auto).  `result`: compare this result instead of
    composing (batch tests)."""
    ref = oracle.compose(m1, m2, merge=True, max_raw_arcs=max_raw_arcs, max_levels=max_levels)
    a = fstc.DeviceFst.from_host(m1) if device_inputs else m1
    b = fstc.DeviceFst.from_host(m2) if device_inputs else m2
    res = result if result is not None else fstc.fstc_compose(
        a, b, merge_mode=merge_mode, max_raw_arcs=max_raw_arcs, max_levels=max_levels, resolve_mode=resolve_mode,
        small_path=small_path)
    nq2 = m2.n_states
    keys, tab, w = gpu_tables(res, nq2)
    # --- states
    assert res.n_states == ref.n_states
    assert (res.pair[0].cpu().numpy() == [m1.start, m2.start]).all()          # state 0 = (s1, s2)
    rkeys = ref.state_keys()
    assert len(np.unique(keys)) == len(keys)
    order, rorder = np.argsort(keys), np.argsort(rkeys)
    assert (keys[order] == rkeys[rorder]).all()
    assert (res.expanded.cpu().numpy()[order] == ref.expanded[rorder]).all()
    # --- accept set (ascending ids, compared as keys)
    acc = res.accept.cpu().numpy()
    assert (np.diff(acc) > 0).all()
    assert (np.sort(keys[acc]) == np.sort(rkeys[ref.accept])).all()
    # --- counters
    assert (res.n_raw_arcs, res.n_levels, res.truncated, res.n_expanded) == \
           (ref.n_raw_arcs, ref.n_levels, ref.truncated, ref.n_expanded)
    st = res.stats
    assert st["level_raw"][:ref.n_levels] == [int(x) for x in ref.level_raw]
    assert st["level_frontier"][:ref.n_levels] == [int(x) for x in ref.level_size]
    # --- arcs
    src = res.src.cpu().numpy()
    assert (np.diff(src) >= 0).all()                                           # sorted by source id
    rtab, rw = canon_arc_table(ref.q1, ref.q2, ref.src, ref.tgt, ref.ilabel, ref.olabel, ref.weight, nq2)
    if merge_mode == fstc.MERGE_OFF:
        assert res.n_arcs == ref.n_raw_arcs == len(src)
        # host-merge the raw GPU arcs (fp64) and compare with the oracle's merged arcs
        if len(tab):
            head = np.ones(len(tab), bool)
            head[1:] = (tab[1:] != tab[:-1]).any(axis=1)
            seg = np.cumsum(head) - 1
            mw = np.zeros(int(seg[-1]) + 1)
            np.add.at(mw, seg, w.astype(np.float64))
            tab, w = tab[head], mw
    else:
        assert res.n_arcs == ref.n_arcs == len(src)
        if len(tab) > 1:
            assert (tab[1:] != tab[:-1]).any(axis=1).all()                     # no duplicate (src,tgt,a,b)
    assert tab.shape == rtab.shape
    assert (tab == rtab).all()
    np.testing.assert_allclose(w, rw, rtol=RTOL, atol=0)
    if merge_mode == fstc.MERGE_SORT_ALL and res.n_arcs:
        t = np.stack([src, res.tgt.cpu().numpy(), res.ilabel.cpu().numpy(), res.olabel.cpu().numpy()], 1).astype(np.int64)
        o = np.lexsort((t[:, 3], t[:, 2], t[:, 1], t[:, 0]))
        assert (o == np.arange(len(o))).all()                                  # fully sorted by (src,tgt,a,b)
    return res, ref


SMALL = [  # (seed, |Q1|, |Σ|, |Γ|, arcs1, |Q2|, |Δ|, arcs2)
    (1, 4, 3, 2, 14, 3, 4, 12),
    (2, 6, 2, 3, 30, 5, 2, 25),
    (3, 7, 5, 4, 20, 6, 3, 18),
    (4, 1, 3, 3, 9, 1, 2, 7),
    (5, 8, 2, 2, 60, 7, 2, 50),
    (6, 5, 4, 6, 6, 5, 4, 6),
    (7, 40, 3, 5, 400, 30, 3, 300),     # several emit tiles, many merges
    (8, 300, 50, 7, 3000, 200, 40, 2500),
]


@pytest.mark.parametrize("case", SMALL)
@pytest.mark.parametrize("merge_mode", [0, 1, 2])
def test_small_random_machines(fstc, case, merge_mode):
    seed, n1, sig, gam, a1, n2, dlt, a2 = case
    m1 = messy_random_fst(seed, n1, sig, gam, a1)
    m2 = messy_random_fst(seed + 100, n2, gam, dlt, a2)
    check_parity(fstc, m1, m2, merge_mode=merge_mode)


@pytest.mark.parametrize("merge_mode", [0, 1, 2])
def test_config_tiny(fstc, merge_mode):
    m1, m2 = workloads.make_config("tiny")
    res, ref = check_parity(fstc, m1, m2, merge_mode=merge_mode)
    assert ref.n_states >= 100


def test_host_inputs_are_staged_by_the_library(fstc):
    m1, m2 = workloads.make_config("tiny")
    check_parity(fstc, m1, m2, device_inputs=False)


@pytest.mark.parametrize("budget", [1, 5, 17, 100, 777, 2000, 3739, 3740, 10 ** 6])
def test_budget_rule_T(fstc, budget):
    m1, m2 = workloads.make_config("tiny")
    check_parity(fstc, m1, m2, max_raw_arcs=budget)


@pytest.mark.parametrize("max_levels", [1, 2, 5, 16, 17, 40])
def test_max_levels(fstc, max_levels):
    m1, m2 = workloads.make_config("tiny")
    check_parity(fstc, m1, m2, max_levels=max_levels)


def test_budget_on_small_messy_machines(fstc):
    for case in SMALL[:3] + SMALL[6:7]:
        seed, n1, sig, gam, a1, n2, dlt, a2 = case
        m1 = messy_random_fst(seed, n1, sig, gam, a1)
        m2 = messy_random_fst(seed + 100, n2, gam, dlt, a2)
        for budget in (1, 3, 7, 12, 20, 35, 60, 500):
            for mm in (0, 1):
                check_parity(fstc, m1, m2, max_raw_arcs=budget, merge_mode=mm)


@pytest.mark.parametrize("merge_mode", [0, 1])
def test_config_medium_scaled(fstc, merge_mode):
    """Medium config at 1/20 scale: ~250k states, several frontier tiles, ragged tails."""
    m1, m2 = workloads.make_config("medium", scale=0.05)
    res, ref = check_parity(fstc, m1, m2, merge_mode=merge_mode)
    assert ref.n_states > 10_000


def test_config_skewed_scaled_with_budget(fstc):
    """Skewed / high-merge config at 1/20 scale under a budget: nearly every source goes through sort + reduce,
    one match spans many emit tiles."""
    m1, m2 = workloads.make_config("skewed", scale=0.05)
    res, ref = check_parity(fstc, m1, m2, max_raw_arcs=2_000_000)
    assert res.stats["n_raw_sorted"] + res.stats["n_raw_grouped"] > 0 and ref.n_arcs < ref.n_raw_arcs


def test_config_nlp_scaled(fstc):
    m1, m2 = workloads.make_config("nlp", scale=0.1)
    res, ref = check_parity(fstc, m1, m2)
    assert ref.n_levels > 20


def test_config_large_scaled_with_budget(fstc):
    m1, m2 = workloads.make_config("large", scale=0.02)
    check_parity(fstc, m1, m2, max_raw_arcs=3_000_000)


def test_degenerate_and_error_cases(fstc):
    # start pair with no matching arcs
    m1 = fst_from_arcs(2, 2, 3, [(0, 0, 0, 1, 1.0)], accept=[0])
    m2 = fst_from_arcs(2, 3, 2, [(0, 1, 0, 1, 1.0)], accept=[0])
    res, _ = check_parity(fstc, m1, m2)
    assert (res.n_states, res.n_arcs) == (1, 0)
    # machines without arcs / without accept states
    e = fst_from_arcs(1, 1, 1, [])
    check_parity(fstc, e, e)
    # zero weights, self loops, arcs to visited targets, parallel duplicates
    m1 = fst_from_arcs(2, 1, 1, [(0, 0, 0, 1, 0.0), (1, 0, 0, 1, 2.0), (1, 0, 0, 0, 3.0), (1, 0, 0, 0, 3.0)])
    m2 = fst_from_arcs(1, 1, 1, [(0, 0, 0, 0, 0.5)] * 3)
    for mm in (0, 1, 2):
        check_parity(fstc, m1, m2, merge_mode=mm)
    # errors: inner alphabets differ; id out of range
    with pytest.raises(fstc.FstcError) as ei:
        fstc.fstc_compose(fst_from_arcs(1, 1, 2, []), fst_from_arcs(1, 3, 1, []))
    assert ei.value.code == -1
    bad = fst_from_arcs(2, 2, 2, [(0, 0, 0, 1, 1.0)])
    bad.tgt = bad.tgt.copy(); bad.tgt[0] = 5
    with pytest.raises(fstc.FstcError) as ei:
        fstc.fstc_compose(bad, bad)
    assert ei.value.code == -2


def test_packed_layout_matches_a_host_sort(fstc):
    """Host-logic check of the packer: arcs sorted by (src, inner, outer, tgt), segment index, flags, accept bits."""
    for side in (1, 2):
        m = messy_random_fst(21, 37, 5, 6, 500, n_accept=4)
        p = fstc.fstc_pack(fstc.DeviceFst.from_host(m), side).to_host()
        inner = m.olabel if side == 1 else m.ilabel
        outer = m.ilabel if side == 1 else m.olabel
        o = np.lexsort((m.tgt, outer, inner, m.src))
        want = np.stack([m.tgt[o], outer[o], m.weight[o].view(np.uint32), inner[o]], 1).astype(np.uint32)
        got = p["arcs"].copy()
        # weights of exact duplicate arcs may come in either order: compare the rest exactly, weights as multisets
        assert (got[:, [0, 1, 3]] == want[:, [0, 1, 3]]).all()
        gk = np.lexsort((got[:, 2], got[:, 3], got[:, 1], got[:, 0]))
        assert (got[:, 2] == want[:, 2]).all() or \
            sorted(map(tuple, got.tolist())) == sorted(map(tuple, want.tolist()))
        s_src, s_in = m.src[o], inner[o]
        head = np.ones(len(o), bool)
        head[1:] = (s_src[1:] != s_src[:-1]) | (s_in[1:] != s_in[:-1])
        assert p["n_segments"] == int(head.sum())
        assert (p["segs"][:-1, 0] == s_in[head]).all() and (p["segs"][:-1, 1] == np.nonzero(head)[0]).all()
        assert tuple(p["segs"][-1]) == (0xFFFFFFFF, m.n_arcs)
        assert (p["seg_ptr"] == np.searchsorted(s_src[head], np.arange(m.n_states + 1))).all()
        D = np.zeros(m.n_states, bool); X = np.zeros(m.n_states, bool)
        seen_ot, seen_iot = set(), set()
        for s, i, ot, t in zip(m.src, inner, outer, m.tgt):
            if (s, ot, t) in seen_ot: D[s] = True
            if (s, i, ot, t) in seen_iot: X[s] = True
            seen_ot.add((s, ot, t)); seen_iot.add((s, i, ot, t))
        assert ((p["flags"] & 1).astype(bool) == D).all() and ((p["flags"] & 2).astype(bool) == X).all()
        bits = np.zeros_like(p["accept_bits"])
        for a in m.accept:
            bits[a >> 5] |= np.uint32(1 << (a & 31))
        assert (p["accept_bits"] == bits).all()


def test_result_to_host_roundtrip(fstc):
    m1, m2 = workloads.make_config("tiny")
    res = fstc.fstc_compose(m1, m2)
    h = res.to_host()
    for k in ("pair", "src", "ilabel", "olabel", "tgt", "weight", "accept", "expanded"):
        assert (h[k].numpy() == getattr(res, k).cpu().numpy()).all(), k


def test_merge_by_construction_and_sort_merge_agree(fstc):
    """Class G (group products, no sort) and class F (radix sort + segmented sum) are two ways to the same merged arcs:
    both against the oracle, on an input where nearly every source can hold duplicates.  (The packed operand's grouped
    copy and its inner-symbol masks are not exported: they are checked end to end, through these results.)"""
    import os
    m1, m2 = workloads.make_config("skewed", scale=0.05)
    res_g, ref = check_parity(fstc, m1, m2, max_raw_arcs=2_000_000)
    assert res_g.stats["n_raw_grouped"] > 0
    os.environ["FSTC_NO_GROUP_MERGE"] = "1"
    try:
        res_f, _ = check_parity(fstc, m1, m2, max_raw_arcs=2_000_000)
    finally:
        del os.environ["FSTC_NO_GROUP_MERGE"]
    assert res_f.stats["n_raw_grouped"] == 0 and res_f.stats["n_raw_sorted"] > 0
    assert (res_f.n_arcs, res_f.n_states) == (res_g.n_arcs, res_g.n_states)
    # small machines with parallel duplicate arcs and zero weights (messy_random_fst): both classes, all merge modes
    for case in SMALL[4:8]:
        seed, n1, sig, gam, a1, n2, dlt, a2 = case
        a = messy_random_fst(seed, n1, sig, gam, a1)
        b = messy_random_fst(seed + 100, n2, gam, dlt, a2)
        check_parity(fstc, a, b)


@pytest.mark.parametrize("small_path", [1, 2])
@pytest.mark.parametrize("no_group", [False, True])
def test_long_runs_of_parallel_arcs_stay_within_tolerance(fstc, small_path, no_group, monkeypatch):
    """3 000 parallel duplicates of one arc on each side, weights spread over three decades: the merged arc is a sum of 9e6
    products (class G: 3 000 x 3 000 by group sums; class F and the small path: sums of up to 3 000 x 3 000 / merged terms).
    A plain sequential fp32 sum of that many terms can leave rtol 1e-5; the merges use compensated sums /
    trees.  Both merge classes and the one-block path against the oracle's fp64 sums."""
    if no_group:
        monkeypatch.setenv("FSTC_NO_GROUP_MERGE", "1")
    rng = np.random.default_rng(12)
    n = 3000 if small_path == 1 else 80                      # the one-block path caps a duplicate-prone source at 8192 raw arcs
    w1 = 10.0 ** rng.uniform(-3, 0, n)
    w2 = 10.0 ** rng.uniform(-3, 0, n)
    arcs1 = [(0, 1, 2, 1, float(w)) for w in w1] + [(1, 0, 1, 0, 0.5), (0, 2, 0, 1, 0.25)]
    arcs2 = [(0, 2, 3, 1, float(w)) for w in w2] + [(1, 1, 0, 0, 0.125), (0, 0, 1, 1, 2.0)]
    m1 = fst_from_arcs(2, 3, 3, arcs1, accept=[1])
    m2 = fst_from_arcs(2, 3, 4, arcs2, accept=[0])
    res, ref = check_parity(fstc, m1, m2, small_path=small_path)
    assert ref.n_raw_arcs > n * n and ref.n_arcs < 20
    assert res.stats["small_path"] == (1 if small_path == 2 else 0)
