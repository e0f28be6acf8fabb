"""Parity of the SMALL path (csrc/small.cu: the whole search of one problem inside one thread block, a batch of problems
in one launch) with the CPU oracle: the same element-by-element comparison as test_gpu_parity.py, with
`small_path=SMALL_ONLY` so that nothing falls back to the level-synchronous path, plus the automatic hand-over of a
problem that outgrows a block, and fstc_compose_batch on many seeded lattices against one packed language model
(PAPER.md:251-259).  `-m gpu`."""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from paper_1805_06383_b200 import workloads
from helpers import fst_from_arcs, messy_random_fst
from test_gpu_parity import SMALL, check_parity, fstc  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu

ONLY, AUTO, OFF = 2, 0, 1


@pytest.mark.parametrize("case", SMALL)
@pytest.mark.parametrize("merge_mode", [0, 1])
def test_small_random_machines_one_block(fstc, case, merge_mode):
    seed, n1, sig, gam, a1, n2, dlt, a2 = case
    m1 = messy_random_fst(seed, n1, sig, gam, a1)
    m2 = messy_random_fst(seed + 100, n2, gam, dlt, a2)
    if n1 * n2 <= 8192:
        res, _ = check_parity(fstc, m1, m2, merge_mode=merge_mode, small_path=ONLY)
        assert res.stats["small_path"] == 1 and res.stats["n_kernel_launches"] == 1
    else:   # up to 60 000 states and levels of more than 4096 pairs: handed over to the level-synchronous path
        res, ref = check_parity(fstc, m1, m2, merge_mode=merge_mode, small_path=AUTO)
        assert res.stats["small_path"] == 0 and ref.n_states > 8192


@pytest.mark.parametrize("merge_mode", [0, 1])
def test_config_tiny_one_block(fstc, merge_mode):
    m1, m2 = workloads.make_config("tiny")
    res, ref = check_parity(fstc, m1, m2, merge_mode=merge_mode, small_path=ONLY)
    assert res.stats["small_path"] == 1 and ref.n_states > 1000


def test_config_nlp_one_block(fstc):
    """The full NLP-shaped config (BASELINE.json configs[2]): 51 levels of <= 8 pairs against 100-symbol lists of the
    bigram machine (q2's list is staged in one chunk of <= 128 entries)."""
    m1, m2 = workloads.make_config("nlp")
    res, ref = check_parity(fstc, m1, m2, small_path=ONLY)
    assert res.stats["small_path"] == 1 and ref.n_levels > 40


@pytest.mark.parametrize("budget", [1, 2, 17, 100, 777, 2500, 3739, 3740, 10**9])
def test_budget_rule_T_one_block(fstc, budget):
    m1, m2 = workloads.make_config("tiny")
    check_parity(fstc, m1, m2, max_raw_arcs=budget, small_path=ONLY)


@pytest.mark.parametrize("max_levels", [1, 3, 9, 40])
def test_max_levels_one_block(fstc, max_levels):
    m1, m2 = workloads.make_config("tiny")
    check_parity(fstc, m1, m2, max_levels=max_levels, small_path=ONLY)
    check_parity(fstc, m1, m2, max_levels=max_levels, max_raw_arcs=1500, small_path=ONLY)


def test_long_symbol_lists_are_staged_in_chunks(fstc):
    """States with 300 distinct inner symbols on both sides: q2's list does not fit one staged chunk (128 entries), q1's
    takes ten rounds of 32 lanes; sparse overlap so that rounds and chunks interleave."""
    rng = np.random.default_rng(77)
    gam = 1000
    def machine(n_states, n_sym, in_side):
        arcs = []
        for q in range(n_states):
            for c in rng.choice(gam, size=n_sym, replace=False):
                outer = int(rng.integers(0, 5))
                t = int(rng.integers(0, n_states))
                arcs.append((q, outer, int(c), t, float(1 - rng.random())) if in_side == 1 else (q, int(c), outer, t, float(1 - rng.random())))
        return arcs
    m1 = fst_from_arcs(6, 5, gam, machine(6, 300, 1), accept=[1, 2])
    m2 = fst_from_arcs(5, gam, 5, machine(5, 300, 2), accept=[0, 3])
    res, ref = check_parity(fstc, m1, m2, small_path=ONLY)
    assert ref.n_raw_arcs > 1000
    check_parity(fstc, m1, m2, merge_mode=1, small_path=ONLY)


def test_degenerate_one_block(fstc):
    m1 = fst_from_arcs(2, 2, 3, [(0, 0, 0, 1, 1.0)], accept=[0])
    m2 = fst_from_arcs(2, 3, 2, [(0, 1, 0, 1, 1.0)], accept=[0])
    res, _ = check_parity(fstc, m1, m2, small_path=ONLY)
    assert (res.n_states, res.n_arcs) == (1, 0)
    m1 = fst_from_arcs(2, 1, 1, [(0, 0, 0, 1, 0.0), (1, 0, 0, 1, 2.0), (1, 0, 0, 0, 3.0), (1, 0, 0, 0, 3.0)])
    m2 = fst_from_arcs(1, 1, 1, [(0, 0, 0, 0, 0.5)] * 3)
    for mm in (0, 1):
        check_parity(fstc, m1, m2, merge_mode=mm, small_path=ONLY)
    empty = fst_from_arcs(1, 1, 2, [])
    check_parity(fstc, empty, fst_from_arcs(1, 2, 1, []), small_path=ONLY)


def test_a_problem_that_outgrows_the_block_is_handed_over(fstc):
    m1, m2 = workloads.make_config("medium", scale=0.05)
    a, b = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    with pytest.raises(fstc.FstcError) as e:
        fstc.fstc_compose(a, b, small_path=ONLY)
    assert e.value.code == fstc.ERR_CAPACITY
    res, ref = check_parity(fstc, m1, m2, small_path=AUTO)
    assert res.stats["small_path"] == 0 and ref.n_states > 10_000
    with pytest.raises(fstc.FstcError):
        fstc.fstc_compose(a, b, small_path=ONLY, merge_mode=fstc.MERGE_SORT_ALL)


def test_capacity_hints_widen_the_block(fstc):
    """skewed at 1/20 scale under a budget: more arcs than the default capacities; the hints make it fit one block."""
    m1, m2 = workloads.make_config("skewed", scale=0.05)
    ref = oracle.compose(m1, m2, merge=True, max_raw_arcs=150_000)
    a, b = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    res = fstc.fstc_compose(a, b, max_raw_arcs=150_000, small_path=AUTO, arc_capacity_hint=400_000, state_capacity_hint=100_000)
    check_parity(fstc, m1, m2, max_raw_arcs=150_000, result=res)
    assert ref.n_arcs < ref.n_raw_arcs                       # merges happened


def test_batch_of_lattices_against_one_language_model(fstc):
    """96 seeded 12 x 6 lattices against one bigram machine of 2 000 words, one call: every result equals the oracle's."""
    vocab = 2000
    lm = workloads._nlp_bigram(9000, vocab, 60, 1.1)
    lats = [workloads._nlp_lattice(9100 + k, 8 + k % 9, 3 + k % 5, vocab, 1.1) for k in range(96)]
    p2 = fstc.fstc_pack(fstc.DeviceFst.from_host(lm), 2)
    p1s = [fstc.fstc_pack(fstc.DeviceFst.from_host(m), 1) for m in lats]
    results = fstc.fstc_compose_batch(p1s, p2)
    assert len(results) == 96 and all(r.stats["small_path"] == 1 for r in results)
    n_nontrivial = 0
    for m, r in zip(lats, results):
        _, ref = check_parity(fstc, m, lm, result=r)
        n_nontrivial += ref.n_arcs > 20
    assert n_nontrivial > 48
    # results of a batch share one block: freeing them in any order, then composing again, works
    for r in results[::2]:
        r.free()
    again = fstc.fstc_compose_batch(p1s[:3], p2, max_levels=4)
    for m, r in zip(lats[:3], again):
        check_parity(fstc, m, lm, max_levels=4, result=r)


@pytest.mark.parametrize("n", [300, 640])
def test_big_batches_take_narrower_blocks(fstc, n):
    """From 2 x and 4 x (number of SMs) problems on, a batch runs in blocks of 256 and 128 threads (several problems
    resident per SM): same results.  Lattices with merges (parallel arcs) and `tiny`-like random machines among them, so
    that the narrower blocks run every step (cut, merge, several matches per pair), each against the oracle."""
    import torch
    assert n >= (4 if n > 600 else 2) * torch.cuda.get_device_properties(0).multi_processor_count
    vocab = 500
    lm = workloads._nlp_bigram(9500, vocab, 40, 1.1)
    lats = []
    for k in range(n):
        m = workloads._nlp_lattice(9600 + k, 4 + k % 7, 2 + k % 4, vocab, 1.1)
        if k % 3 == 0:                                     # parallel duplicate arcs: duplicate-prone sources, merged in the block
            m = workloads._with_parallel_arcs(m, k, 0.5)
        lats.append(m)
    p2 = fstc.fstc_pack(fstc.DeviceFst.from_host(lm), 2)
    p1s = [fstc.fstc_pack(fstc.DeviceFst.from_host(m), 1) for m in lats]
    for opts in ({}, {"max_raw_arcs": 40}):
        results = fstc.fstc_compose_batch(p1s, p2, **opts)
        assert all(r.stats["small_path"] == 1 and r.stats["n_kernel_launches"] == 1 for r in results)
        merged = 0
        for m, r in zip(lats, results):
            _, ref = check_parity(fstc, m, lm, result=r, **opts)
            merged += ref.n_arcs < ref.n_raw_arcs
        assert merged > n // 10


def test_batch_hands_over_what_does_not_fit(fstc):
    m1, m2 = workloads.make_config("medium", scale=0.03)
    t1, _ = workloads.make_config("tiny")
    # two small left operands over M2's input alphabet, and the big one
    rng = np.random.default_rng(5)
    gam = m2.n_isyms
    small = [fst_from_arcs(3, 4, gam, [(0, 1, int(rng.integers(0, 20)), 1, 0.5), (1, 2, int(rng.integers(0, 20)), 2, 0.25),
                                       (0, 3, int(rng.integers(0, 20)), 2, 1.0)], accept=[2]) for _ in range(2)]
    ops = [small[0], m1, small[1]]
    p2 = fstc.fstc_pack(fstc.DeviceFst.from_host(m2), 2)
    p1s = [fstc.fstc_pack(fstc.DeviceFst.from_host(m), 1) for m in ops]
    results = fstc.fstc_compose_batch(p1s, p2)
    assert [r.stats["small_path"] for r in results] == [1, 0, 1]
    for m, r in zip(ops, results):
        check_parity(fstc, m, m2, result=r)
    with pytest.raises(fstc.FstcError):
        fstc.fstc_compose_batch(p1s, p2, small_path=ONLY)
