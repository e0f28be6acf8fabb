"""Pins for the CPU oracle (oracle/fst_compose_oracle.cpp) against things that are NOT the oracle:
brute force over the full product, closed forms, textbook special cases and the paper's printed
example.  All CPU (`-m "not gpu"`).  Citations are PAPER.md lines.
"""
from __future__ import annotations

import os
from collections import defaultdict

import numpy as np
import pytest

import oracle
from oracle import brute_force
from paper_1805_06383_b200 import workloads
from helpers import canon_arcs, canon_states, fst_from_arcs, messy_random_fst

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _oracle_canon(res):
    return canon_arcs(res.q1, res.q2, res.src, res.tgt, res.ilabel, res.olabel, res.weight)


def _assert_arcs_equal(got, want, rtol=1e-12):
    assert set(got) == set(want)
    for k, w in want.items():
        assert got[k] == pytest.approx(w, rel=rtol, abs=0.0), k


CASES = [  # (seed, |Q1|, |Σ|, |Γ|, arcs1, |Q2|, |Δ|, arcs2)
    (1, 4, 3, 2, 14, 3, 4, 12),
    (2, 6, 2, 3, 30, 5, 2, 25),        # tiny outer alphabets: many merges
    (3, 7, 5, 4, 20, 6, 3, 18),
    (4, 1, 3, 3, 9, 1, 2, 7),          # single states
    (5, 8, 2, 2, 60, 7, 2, 50),        # dense: lots of parallel duplicates
    (6, 5, 4, 6, 6, 5, 4, 6),          # sparse: search dies early
]


@pytest.mark.parametrize("case", CASES)
@pytest.mark.parametrize("force_map", [False, True])
def test_matches_brute_force_full_product_then_trim(case, force_map):
    """Definition PAPER.md:47-65 over ALL of Q1×Q2, trimmed to the accessible part (:77)."""
    seed, n1, sig, gam, a1, n2, dlt, a2 = case
    m1 = messy_random_fst(seed, n1, sig, gam, a1)
    m2 = messy_random_fst(seed + 100, n2, gam, dlt, a2)
    level, arcs, accept, raw = brute_force.compose(m1, m2)
    res = oracle.compose(m1, m2, force_map=force_map)
    assert (res.q1[0], res.q2[0]) == (m1.start, m2.start)
    pairs = canon_states(res.q1, res.q2)
    assert len(set(pairs)) == len(pairs)
    assert pairs == sorted(level)
    got_level = {(int(a), int(b)): int(l) for a, b, l in zip(res.q1, res.q2, res.level)}
    assert got_level == level
    _assert_arcs_equal(_oracle_canon(res), arcs)
    assert res.n_arcs == len(arcs) == len(res.src)            # merged: one arc per key
    assert {(int(res.q1[i]), int(res.q2[i])) for i in res.accept} == accept
    assert res.n_raw_arcs == sum(raw.values())
    assert res.truncated == 0 and res.n_expanded == res.n_states and res.expanded.all()
    by_level = defaultdict(int)
    for p, l in level.items():
        by_level[l] += raw[p]
    assert [int(x) for x in res.level_raw] == [by_level[l] for l in range(res.n_levels)]
    # |F_l|, the frontier sizes (the GPU tests use them as the expected `level_frontier`): counted from the brute force's levels
    assert [int(x) for x in res.level_size] == [sum(1 for l in level.values() if l == i) for i in range(res.n_levels)]


@pytest.mark.parametrize("case", CASES[:4])
def test_unmerged_mode_is_the_raw_multiset(case):
    """PAPER.md:289 'without performing any reductions': every (e1,e2) match is its own arc."""
    seed, n1, sig, gam, a1, n2, dlt, a2 = case
    m1 = messy_random_fst(seed, n1, sig, gam, a1)
    m2 = messy_random_fst(seed + 100, n2, gam, dlt, a2)
    _, arcs, _, raw = brute_force.compose(m1, m2)
    res = oracle.compose(m1, m2, merge=False)
    assert res.n_arcs == res.n_raw_arcs == sum(raw.values()) == len(res.src)
    _assert_arcs_equal(_oracle_canon(res), arcs)               # host-merged raw == merged definition


def test_closed_form_total_outweight_per_state():
    """Σ_{arcs leaving (q1,q2)} w = Σ_c W1(q1,c)·W2(q2,c), W(q,c) = Σ weights of q's arcs on inner c."""
    m1, m2 = workloads.make_config("tiny")
    res = oracle.compose(m1, m2)
    assert res.n_states >= 100, "degenerate seed (DESIGN.md seed rule)"
    W1 = np.zeros((m1.n_states, m1.n_osyms))
    W2 = np.zeros((m2.n_states, m2.n_isyms))
    np.add.at(W1, (m1.src, m1.olabel), m1.weight.astype(np.float64))
    np.add.at(W2, (m2.src, m2.ilabel), m2.weight.astype(np.float64))
    want = (W1[res.q1] * W2[res.q2]).sum(axis=1)
    got = np.zeros(res.n_states)
    np.add.at(got, res.src, res.weight)
    np.testing.assert_allclose(got, want, rtol=1e-12, atol=0)
    # and the raw count closed form: raw(q1,q2) = Σ_c n1(q1,c)·n2(q2,c)
    N1 = np.zeros((m1.n_states, m1.n_osyms), np.int64)
    N2 = np.zeros((m2.n_states, m2.n_isyms), np.int64)
    np.add.at(N1, (m1.src, m1.olabel), 1)
    np.add.at(N2, (m2.src, m2.ilabel), 1)
    assert res.n_raw_arcs == int((N1[res.q1] * N2[res.q2]).sum())


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_single_state_machines_are_a_matrix_product(seed):
    """|Q1|=|Q2|=1: arc a:b has weight (A·B)[a,b], A[a,c], B[c,b] the summed symbol-weight matrices;
    it exists iff row a of A and column b of B share a structural nonzero."""
    rng = np.random.default_rng(seed)
    sig, gam, dlt = 5, 7, 4                                     # all different: a transposed operand fails
    n1, n2 = 17, 15
    m1 = fst_from_arcs(1, sig, gam, [(0, int(rng.integers(sig)), int(rng.integers(gam)), 0, float(rng.random() + 0.1))
                                     for _ in range(n1)], accept=[0])
    m2 = fst_from_arcs(1, gam, dlt, [(0, int(rng.integers(gam)), int(rng.integers(dlt)), 0, float(rng.random() + 0.1))
                                     for _ in range(n2)], accept=[0])
    A = np.zeros((sig, gam)); B = np.zeros((gam, dlt))
    np.add.at(A, (m1.ilabel, m1.olabel), m1.weight.astype(np.float64))
    np.add.at(B, (m2.ilabel, m2.olabel), m2.weight.astype(np.float64))
    C = np.matmul(A, B)
    S = np.matmul((A != 0).astype(np.int64), (B != 0).astype(np.int64)) > 0
    res = oracle.compose(m1, m2)
    assert res.n_states == 1 and list(res.accept) == [0]
    got = np.zeros((sig, dlt)); seen = np.zeros((sig, dlt), bool)
    for a, b, w, s, t in zip(res.ilabel, res.olabel, res.weight, res.src, res.tgt):
        assert s == 0 and t == 0 and not seen[a, b]
        seen[a, b] = True
        got[a, b] = w
    assert (seen == S).all()
    np.testing.assert_allclose(got, np.where(S, C, 0.0), rtol=1e-12)


def test_identity_right_operand_returns_accessible_m1_with_parallel_arcs_summed():
    m1 = messy_random_fst(11, 9, 4, 5, 40, n_accept=3)
    gam = m1.n_osyms
    ident = fst_from_arcs(1, gam, gam, [(0, c, c, 0, 1.0) for c in range(gam)], accept=[0])
    res = oracle.compose(m1, ident)
    # accessible part of M1 by a plain graph search
    succ = defaultdict(set)
    for s, t in zip(m1.src, m1.tgt):
        succ[int(s)].add(int(t))
    reach, todo = {m1.start}, [m1.start]
    while todo:
        q = todo.pop()
        for r in succ[q]:
            if r not in reach:
                reach.add(r); todo.append(r)
    want = defaultdict(float)
    for s, a, c, t, p in zip(m1.src, m1.ilabel, m1.olabel, m1.tgt, m1.weight):
        if int(s) in reach:
            want[((int(s), 0), int(a), int(c), (int(t), 0))] += float(p)
    assert canon_states(res.q1, res.q2) == sorted((q, 0) for q in reach)
    _assert_arcs_equal(_oracle_canon(res), dict(want))
    assert {int(res.q1[i]) for i in res.accept} == reach & set(int(x) for x in m1.accept)


def test_two_linear_chains_stop_at_first_mismatch():
    inner = [3, 1, 4, 1, 5, 2]
    other = [3, 1, 4, 0, 5, 2]                                  # differs at position 3
    m1 = fst_from_arcs(7, 9, 6, [(i, i + 1, inner[i], i + 1, 0.5 + 0.05 * i) for i in range(6)], accept=[6])
    m2 = fst_from_arcs(7, 6, 9, [(i, other[i], 8 - i, i + 1, 0.25 + 0.1 * i) for i in range(6)], accept=[6])
    res = oracle.compose(m1, m2)
    assert canon_states(res.q1, res.q2) == [(i, i) for i in range(4)]
    want = {((i, i), i + 1, 8 - i, (i + 1, i + 1)): float(np.float32(0.5 + 0.05 * i)) * float(np.float32(0.25 + 0.1 * i))
            for i in range(3)}
    _assert_arcs_equal(_oracle_canon(res), want)
    assert res.n_levels == 4 and len(res.accept) == 0
    assert [int(x) for x in res.level_raw] == [1, 1, 1, 0]


def test_lattice_times_bigram_total_weight_is_the_hmm_forward_recursion():
    """Config-3-shaped pair (acyclic lattice ∘ bigram): Σ over accepting paths of the result,
    by forward sums over its DAG, equals the forward recursion over (position, last word)."""
    m1, m2 = workloads.make_config("nlp", seeds=(7, 8), scale=0.01)   # vocab 300
    res = oracle.compose(m1, m2)
    assert res.n_levels > 10
    # forward over the composed DAG in level order (level == lattice position)
    alpha = np.zeros(res.n_states); alpha[0] = 1.0
    order = np.argsort(res.level[res.src], kind="stable")
    for i in order:
        alpha[res.tgt[i]] += alpha[res.src[i]] * res.weight[i]
    total = float(alpha[res.accept].sum())
    # direct recursion
    big = defaultdict(float)
    for u, w_in, w_out, t, p in zip(m2.src, m2.ilabel, m2.olabel, m2.tgt, m2.weight):
        assert w_in == w_out == t
        big[(int(u), int(w_in))] += float(p)
    n_pos = m1.n_states - 1
    lat = defaultdict(list)
    for s, a, c, t, p in zip(m1.src, m1.ilabel, m1.olabel, m1.tgt, m1.weight):
        assert a == c and t == s + 1
        lat[int(s)].append((int(c), float(p)))
    f = {int(m2.start): 1.0}
    for i in range(n_pos):
        g = defaultdict(float)
        for u, fu in f.items():
            for w, p in lat[i]:
                b = big.get((u, w))
                if b is not None:
                    g[w] += fu * p * b
        f = g
    want = sum(f.values())                                      # F1 = {last position}, F2 = all states
    assert want > 0
    assert total == pytest.approx(want, rel=1e-10)


BUDGETS = [1, 3, 7, 12, 20, 35, 60, 10_000]


@pytest.mark.parametrize("case", CASES[:3])
def test_budget_rule_T_against_brute_force(case):
    seed, n1, sig, gam, a1, n2, dlt, a2 = case
    m1 = messy_random_fst(seed, n1, sig, gam, a1)
    m2 = messy_random_fst(seed + 100, n2, gam, dlt, a2)
    for budget in BUDGETS:
        for max_levels in (0, 1, 2):
            states, expanded, arcs, trunc, n_raw = brute_force.compose_truncated(m1, m2, budget, max_levels)
            res = oracle.compose(m1, m2, max_raw_arcs=budget, max_levels=max_levels)
            assert canon_states(res.q1, res.q2) == sorted(states), (budget, max_levels)
            assert {(int(a), int(b)) for a, b, e in zip(res.q1, res.q2, res.expanded) if e} == expanded
            _assert_arcs_equal(_oracle_canon(res), arcs)
            assert res.truncated == trunc and res.n_raw_arcs == n_raw <= max(budget, 0) or budget == 0
            assert res.n_expanded == len(expanded)


def test_truncation_on_a_level_boundary_equals_the_level_restricted_full_result():
    m1, m2 = workloads.make_config("tiny")
    full = oracle.compose(m1, m2)
    cum = np.cumsum(full.level_raw)
    L = 5
    cut = oracle.compose(m1, m2, max_raw_arcs=int(cum[L - 1]))   # levels 0..L-1 fit exactly, level L does not
    assert cut.truncated == 1
    fc = _oracle_canon(full)
    lvl = {(int(a), int(b)): int(l) for a, b, l in zip(full.q1, full.q2, full.level)}
    want = {k: w for k, w in fc.items() if lvl[k[0]] < L}
    got = _oracle_canon(cut)
    extra = {k: w for k, w in got.items() if k not in want}       # a (possibly empty) prefix of level L
    assert all(lvl[k[0]] == L for k in extra)
    _assert_arcs_equal({k: w for k, w in got.items() if k in want}, want)
    assert cut.n_raw_arcs <= int(cum[L - 1]) + int(full.level_raw[L])


def test_paper_printed_example_structure():
    """three inner symbols, gata matches nothing, two composed arcs from (0,0)."""
    sec = defaultdict(list)
    cur = None
    for line in open(os.path.join(GOLDEN, "paper_fig1_start_pair.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        if line.startswith("["):
            name, _, rest = line[1:].partition("]")
            cur = name
            if rest.strip():
                sec[cur].append(rest.split())
        else:
            sec[cur].append(line.split())
    inner = {s: i for i, s in enumerate(sec["inner"][0])}
    sig, dlt = {}, {}
    arcs1 = [(int(s), sig.setdefault(a, len(sig)), inner[c], int(t), 0.5) for s, a, c, t in sec["m1_start_arcs"]]
    arcs2 = [(int(s), inner[c], dlt.setdefault(b, len(dlt)), int(t), 0.5) for s, c, b, t in sec["m2_start_arcs"]]
    m1 = fst_from_arcs(3, len(sig), len(inner), arcs1)
    m2 = fst_from_arcs(3, len(inner), len(dlt), arcs2)
    res = oracle.compose(m1, m2, max_levels=1)
    want = {((int(q1), int(q2)), sig[a], dlt[b], (int(r1), int(r2))) for q1, q2, a, b, r1, r2 in sec["composed_from_start"]}
    assert set(_oracle_canon(res)) == want
    assert res.n_raw_arcs == 2
    x = oracle.PairExpander(m1, m2)
    assert x.raw_count(0, 0) == 2                                # la:1·1 + gata:0 + una:1·1


def test_degenerate_inputs():
    # N15: start pair with no matching arcs -> one state, no arcs
    m1 = fst_from_arcs(2, 2, 3, [(0, 0, 0, 1, 1.0)], accept=[0])
    m2 = fst_from_arcs(2, 3, 2, [(0, 1, 0, 1, 1.0)], accept=[0])
    r = oracle.compose(m1, m2)
    assert (r.n_states, r.n_arcs, r.n_raw_arcs, r.n_levels, r.truncated) == (1, 0, 0, 1, 0)
    assert list(r.accept) == [0]
    # no arcs at all
    e1 = fst_from_arcs(1, 1, 1, [])
    r = oracle.compose(e1, e1)
    assert (r.n_states, r.n_arcs) == (1, 0) and len(r.accept) == 0
    # N8: zero weight still makes an arc and a state;  N7: self loop / arc to a visited target is emitted
    m1 = fst_from_arcs(2, 1, 1, [(0, 0, 0, 1, 0.0), (1, 0, 0, 1, 2.0), (1, 0, 0, 0, 3.0)])
    m2 = fst_from_arcs(1, 1, 1, [(0, 0, 0, 0, 0.5)])
    r = oracle.compose(m1, m2)
    assert canon_arcs(r.q1, r.q2, r.src, r.tgt, r.ilabel, r.olabel, r.weight) == {
        ((0, 0), 0, 0, (1, 0)): 0.0, ((1, 0), 0, 0, (1, 0)): 1.0, ((1, 0), 0, 0, (0, 0)): 1.5}
    # N9: parallel duplicate input arcs each contribute
    m1 = fst_from_arcs(1, 1, 1, [(0, 0, 0, 0, 0.25)] * 3)
    r = oracle.compose(m1, m2)
    assert r.n_raw_arcs == 3 and r.n_arcs == 1 and r.weight[0] == pytest.approx(0.375)
    with pytest.raises(ValueError):
        oracle.compose(fst_from_arcs(1, 1, 2, []), fst_from_arcs(1, 3, 1, []))   # N14


def test_tiny_config_invariants_and_pair_expander():
    m1, m2 = workloads.make_config("tiny")
    res = oracle.compose(m1, m2)
    raw = oracle.compose(m1, m2, merge=False)
    assert res.n_states == raw.n_states and res.n_raw_arcs == raw.n_raw_arcs == raw.n_arcs
    assert res.n_arcs <= res.n_raw_arcs
    keys = set(zip(res.src.tolist(), res.tgt.tolist(), res.ilabel.tolist(), res.olabel.tolist()))
    assert len(keys) == res.n_arcs                              # no duplicate (src,tgt,a,b)
    # every state but the start has an incoming arc from exactly one level below
    best = np.full(res.n_states, 1 << 30)
    np.minimum.at(best, res.tgt, res.level[res.src] + 1)
    assert (best[1:] == res.level[1:]).all() and res.level[0] == 0
    # total weight per source is unchanged by merging
    s_m = np.zeros(res.n_states); s_r = np.zeros(res.n_states)
    np.add.at(s_m, res.src, res.weight); np.add.at(s_r, raw.src, raw.weight)
    by_pair_m = dict(zip(zip(res.q1.tolist(), res.q2.tolist()), s_m))     # ids differ between the two runs
    by_pair_r = dict(zip(zip(raw.q1.tolist(), raw.q2.tolist()), s_r))
    assert by_pair_m.keys() == by_pair_r.keys()
    for k, v in by_pair_r.items():
        assert by_pair_m[k] == pytest.approx(v, rel=1e-12)
    # one pair at a time == the whole run
    x = oracle.PairExpander(m1, m2)
    whole = _oracle_canon(res)
    n = 0
    for i in range(0, res.n_states, 7):
        q1, q2 = int(res.q1[i]), int(res.q2[i])
        r1, r2, a, b, w = x.expand(q1, q2)
        assert x.raw_count(q1, q2) >= len(w)
        for j in range(len(w)):
            assert whole[((q1, q2), int(a[j]), int(b[j]), (int(r1[j]), int(r2[j])))] == pytest.approx(w[j], rel=1e-12)
        assert len(w) == sum(1 for k in whole if k[0] == (q1, q2))
        n += len(w)
    assert n > 0


@pytest.mark.parametrize("seed", [11, 12, 13, 14])
def test_merged_weights_are_a_contraction_over_the_inner_symbol(seed):
    """PAPER.md:53 read as tensors: with A[q1,a,c,r1] and B[q2,c,b,r2] the summed input weights (and their structural
    0/1 versions), the merged arc (q1q2, a, b, r1r2) exists iff the structural contraction over c is non-zero and weighs
    sum_c A·B.  Checked with numpy.einsum for every reached source: a dropped duplicate, a product summed in the wrong
    group or a transposed operand fails it.  (Also the identity behind the CUDA path's merge by construction.)"""
    n1, n2, sig, gam, dlt = 5, 4, 3, 4, 3
    m1 = messy_random_fst(seed, n1, sig, gam, 60, dup_frac=0.3)
    m2 = messy_random_fst(seed + 50, n2, gam, dlt, 50, dup_frac=0.3)
    A = np.zeros((n1, sig, gam, n1)); As = np.zeros_like(A)
    B = np.zeros((n2, gam, dlt, n2)); Bs = np.zeros_like(B)
    np.add.at(A, (m1.src, m1.ilabel, m1.olabel, m1.tgt), m1.weight.astype(np.float64))
    np.add.at(As, (m1.src, m1.ilabel, m1.olabel, m1.tgt), 1.0)
    np.add.at(B, (m2.src, m2.ilabel, m2.olabel, m2.tgt), m2.weight.astype(np.float64))
    np.add.at(Bs, (m2.src, m2.ilabel, m2.olabel, m2.tgt), 1.0)
    W = np.einsum("pacr,qcbs->pqabrs", A, B)            # [q1, q2, a, b, r1, r2]
    S = np.einsum("pacr,qcbs->pqabrs", As, Bs) > 0
    res = oracle.compose(m1, m2, merge=True)
    got = _oracle_canon(res)
    want = {}
    for q1, q2 in zip(res.q1, res.q2):                   # every reached (and here expanded) source pair
        for a, b, r1, r2 in zip(*np.nonzero(S[q1, q2])):
            want[((int(q1), int(q2)), int(a), int(b), (int(r1), int(r2)))] = float(W[q1, q2, a, b, r1, r2])
    _assert_arcs_equal(got, want, rtol=1e-12)
    assert len(got) < res.n_raw_arcs                     # the inputs are made so that merging really happens
