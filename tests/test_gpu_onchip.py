"""Class S, the merge ON CHIP (compose.cu `k_fchip`, SURVEY §8(f)1 / PAPER.md:321): sources that can hold duplicates and
have at most 512 raw arcs are composed, merged and summed in shared memory; only their merged arcs reach HBM.  Parity
with the oracle element by element like test_gpu_parity.py, on inputs that put raw arcs on every merge route at once
(S on chip, F through the HBM sort, G by construction), on every way to the target ids (dense table, hash table,
partitioned resolve), under a budget cut, in chunks, and with long runs of parallel arcs.  `-m gpu`."""
from __future__ import annotations

import numpy as np
import pytest

from paper_1805_06383_b200 import workloads
from helpers import fst_from_arcs, messy_random_fst
from test_gpu_parity import SMALL, check_parity, fstc  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu

TABLE, PARTITIONED, HASH = 1, 2, 3


def sparse_duplicate_machines(seed, n_states, n_sym, n_inner, arcs_per_state, dup_frac=0.3):
    """Machines whose sources are duplicate-prone but whose (outer, target) groups hardly ever share an inner symbol:
    many arcs per state over a wide inner alphabet, a part of them repeated as parallel arcs (flag X) — the group
    product of a pair is far above 8 x its raw arcs, so AUTO sends the pair to class F / S, not to class G."""
    rng = np.random.default_rng(seed)
    arcs = []
    for q in range(n_states):
        k = int(rng.integers(arcs_per_state // 2, arcs_per_state + 1))
        base = [(q, int(rng.integers(n_sym)), int(rng.integers(n_inner)), int(rng.integers(n_states)), float(rng.uniform(0.1, 1.0)))
                for _ in range(k)]
        dups = [base[int(i)][:4] + (float(rng.uniform(0.1, 1.0)),) for i in rng.integers(0, k, int(k * dup_frac))]
        arcs += base + dups
    return arcs


def make_pair(seed, n1=60, n2=50, n_inner=40, per_state=24):
    a1 = sparse_duplicate_machines(seed, n1, 5, n_inner, per_state)
    a2 = sparse_duplicate_machines(seed + 1, n2, 5, n_inner, per_state)
    m1 = fst_from_arcs(n1, 5, n_inner, [(s, a, c, t, w) for (s, a, c, t, w) in a1], accept=[n1 - 1])
    m2 = fst_from_arcs(n2, n_inner, 5, [(s, c, b, t, w) for (s, b, c, t, w) in a2], accept=[0, n2 - 1])
    return m1, m2


@pytest.mark.parametrize("resolve_mode", [0, TABLE, PARTITIONED, HASH])
@pytest.mark.parametrize("seed", [1, 2])
def test_sparse_duplicate_prone_sources_merge_on_chip(fstc, seed, resolve_mode, monkeypatch):
    m1, m2 = make_pair(seed)
    res, ref = check_parity(fstc, m1, m2, resolve_mode=resolve_mode)
    st = res.stats
    assert st["n_raw_onchip"] > 0.5 * ref.n_raw_arcs and ref.n_arcs < ref.n_raw_arcs
    assert st["n_raw_onchip"] <= st["n_raw_sorted"]
    monkeypatch.setenv("FSTC_NO_CHIP_MERGE", "1")             # the same sources through the HBM sort: the same machine
    res_f, _ = check_parity(fstc, m1, m2, resolve_mode=resolve_mode)
    assert res_f.stats["n_raw_onchip"] == 0 and res_f.stats["n_raw_sorted"] == st["n_raw_sorted"]
    assert (res_f.n_states, res_f.n_arcs) == (res.n_states, res.n_arcs)


@pytest.mark.parametrize("budget", [1, 500, 20_000, 150_000])
def test_on_chip_merge_under_a_budget_cut(fstc, budget):
    m1, m2 = make_pair(3)
    res, ref = check_parity(fstc, m1, m2, max_raw_arcs=budget)
    assert ref.truncated == 1 or budget >= ref.n_raw_arcs


@pytest.mark.parametrize("merge_mode", [0, 1, 2])
def test_every_merge_mode_on_the_same_input(fstc, merge_mode):
    m1, m2 = make_pair(4)
    res, _ = check_parity(fstc, m1, m2, merge_mode=merge_mode)
    assert (res.stats["n_raw_onchip"] > 0) == (merge_mode == 0)     # MERGE_OFF merges nothing; SORT_ALL keeps its total order


@pytest.mark.parametrize("case", SMALL)
def test_messy_machines_without_class_g(fstc, case, monkeypatch):
    """Zero weights, parallel duplicates, states without arcs (messy_random_fst), class G off: every duplicate-prone
    source of at most 512 raw arcs goes on chip, the heavier ones through the sort."""
    monkeypatch.setenv("FSTC_NO_GROUP_MERGE", "1")
    seed, n1, sig, gam, a1, n2, dlt, a2 = case
    m1 = messy_random_fst(seed, n1, sig, gam, a1)
    m2 = messy_random_fst(seed + 100, n2, gam, dlt, a2)
    for rm in (0, PARTITIONED):
        res, ref = check_parity(fstc, m1, m2, resolve_mode=rm)
        if ref.n_arcs < ref.n_raw_arcs:
            assert res.stats["n_raw_sorted"] > 0 and res.stats["n_raw_grouped"] == 0


@pytest.mark.parametrize("no_group", [False, True])
def test_all_merge_routes_in_one_run(fstc, no_group, monkeypatch):
    """The sparse machines plus a few HEAVY states (70 arcs on one inner symbol): a pair of heavy states has 4 900 raw arcs,
    above the cap of class S, and a dense group product: class G takes it, or the HBM sort when class G is off; the light
    pairs around it, some in the same level, merge on chip."""
    if no_group:
        monkeypatch.setenv("FSTC_NO_GROUP_MERGE", "1")
    n1, n2, n_inner = 60, 50, 40
    rng = np.random.default_rng(11)
    a1 = sparse_duplicate_machines(21, n1, 5, n_inner, 24)
    a2 = sparse_duplicate_machines(22, n2, 5, n_inner, 24)
    for q in (0, 7, 13):
        a1 += [(q, int(rng.integers(5)), 3, int(rng.choice([0, 7, 13, 20])), float(rng.uniform(0.1, 1.0))) for _ in range(70)]
        a2 += [(q, int(rng.integers(5)), 3, int(rng.choice([0, 7, 13, 21])), float(rng.uniform(0.1, 1.0))) for _ in range(70)]
    m1 = fst_from_arcs(n1, 5, n_inner, a1, accept=[n1 - 1])
    m2 = fst_from_arcs(n2, n_inner, 5, [(s, c, b, t, w) for (s, b, c, t, w) in a2], accept=[0])
    res, ref = check_parity(fstc, m1, m2)
    st = res.stats
    assert st["n_raw_onchip"] > 0 and ref.n_arcs < ref.n_raw_arcs
    if no_group:
        assert st["n_raw_grouped"] == 0 and st["n_raw_sorted"] >= st["n_raw_onchip"] + 4900
    else:
        assert st["n_raw_grouped"] >= 4900


def test_on_chip_merge_in_chunks(fstc, monkeypatch):
    monkeypatch.setenv("FSTC_CHUNK_ARCS", "5000")
    m1, m2 = make_pair(5)
    res, _ = check_parity(fstc, m1, m2)
    assert res.stats["n_chunks"] > 1 and res.stats["n_raw_onchip"] > 0


def test_long_runs_of_parallel_arcs_on_chip(fstc, monkeypatch):
    """22 x 22 = 484 products into ONE merged arc (a source just under the cap of class S), weights over three decades, next to
    sources of a handful of arcs: the fp64 slot sums keep rtol 1e-5 (check_parity) whatever the order of arrival."""
    monkeypatch.setenv("FSTC_NO_GROUP_MERGE", "1")
    rng = np.random.default_rng(7)
    n = 22
    w1, w2 = 10.0 ** rng.uniform(-3, 0, n), 10.0 ** rng.uniform(-3, 0, n)
    arcs1 = [(0, 1, 2, 1, float(w)) for w in w1] + [(1, 0, 1, 0, 0.5), (1, 0, 1, 0, 0.25), (0, 2, 0, 1, 0.25)]
    arcs2 = [(0, 2, 3, 1, float(w)) for w in w2] + [(1, 1, 0, 0, 0.125), (1, 1, 0, 0, 0.5), (0, 0, 1, 1, 2.0)]
    m1 = fst_from_arcs(2, 3, 3, arcs1, accept=[1])
    m2 = fst_from_arcs(2, 3, 4, arcs2, accept=[0])
    res, ref = check_parity(fstc, m1, m2)
    assert res.stats["n_raw_onchip"] >= n * n and ref.n_arcs < 20


def test_empty_and_single_arc_sources(fstc, monkeypatch):
    monkeypatch.setenv("FSTC_NO_GROUP_MERGE", "1")
    m1 = fst_from_arcs(3, 2, 2, [(0, 0, 0, 1, 0.5), (0, 0, 0, 1, 0.25), (1, 1, 1, 2, 1.0)], accept=[2])
    m2 = fst_from_arcs(3, 2, 2, [(0, 0, 1, 1, 2.0), (0, 0, 1, 1, 4.0), (1, 1, 0, 2, 1.0)], accept=[2])
    res, ref = check_parity(fstc, m1, m2)
    assert ref.n_raw_arcs == 5 and ref.n_arcs == 2 and res.stats["n_raw_onchip"] == 4      # (the single arc of (1,1) is class U)
