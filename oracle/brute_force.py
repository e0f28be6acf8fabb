"""ORACLE PIN — TEST INFRASTRUCTURE ONLY.

Brute force for tiny inputs, straight from the definition:
build δ over the FULL state set Q1×Q2 (every pair, reachable or not), then trim
to the pairs accessible from s1s2.  Pure-Python loops and dicts,
fp64 (Python floats); shares no code with fst_compose_oracle.cpp or the CUDA path.
"""
from __future__ import annotations

from collections import defaultdict
from typing import Dict, List, Set, Tuple

Pair = Tuple[int, int]
ArcKey = Tuple[Pair, int, int, Pair]        # (source pair, a, b, target pair)


def full_product(m1, m2) -> Tuple[Dict[ArcKey, float], Dict[Pair, int]]:
    """δ(q1q2,a,b,r1r2) = Σ_c δ1(q1,a,c,r1)·δ2(q2,c,b,r2) for ALL (q1,q2) ∈ Q1×Q2.

    Returns (delta, raw) where raw[(q1,q2)] counts the (e1,e2) matches of the pair.
    """
    out1: Dict[int, List[Tuple[int, int, int, float]]] = defaultdict(list)
    out2: Dict[int, List[Tuple[int, int, int, float]]] = defaultdict(list)
    for s, a, c, r, p in zip(m1.src, m1.ilabel, m1.olabel, m1.tgt, m1.weight):
        out1[int(s)].append((int(a), int(c), int(r), float(p)))
    for s, c, b, r, p in zip(m2.src, m2.ilabel, m2.olabel, m2.tgt, m2.weight):
        out2[int(s)].append((int(c), int(b), int(r), float(p)))
    delta: Dict[ArcKey, float] = defaultdict(float)
    raw: Dict[Pair, int] = defaultdict(int)
    for q1 in range(int(m1.n_states)):
        for q2 in range(int(m2.n_states)):
            for (a, c1, r1, p1) in out1.get(q1, ()):
                for (c2, b, r2, p2) in out2.get(q2, ()):
                    if c1 == c2:
                        delta[((q1, q2), a, b, (r1, r2))] += p1 * p2
                        raw[(q1, q2)] += 1
    return dict(delta), dict(raw)


def trim(m1, m2, delta: Dict[ArcKey, float]) -> Tuple[Dict[Pair, int], Dict[ArcKey, float]]:
    """Accessible part: BFS levels of every pair reachable from (s1,s2), and the arcs leaving them."""
    succ: Dict[Pair, Set[Pair]] = defaultdict(set)
    for (p, _a, _b, r) in delta:
        succ[p].add(r)
    start = (int(m1.start), int(m2.start))
    level = {start: 0}
    frontier = [start]
    while frontier:
        nxt = []
        for p in frontier:
            for r in succ.get(p, ()):
                if r not in level:
                    level[r] = level[p] + 1
                    nxt.append(r)
        frontier = nxt
    arcs = {k: w for k, w in delta.items() if k[0] in level}
    return level, arcs


def compose(m1, m2):
    """-> (level: {pair: BFS distance}, arcs: {(src pair, a, b, tgt pair): weight}, accept: set of pairs, raw)."""
    delta, raw = full_product(m1, m2)
    level, arcs = trim(m1, m2, delta)
    f1 = set(int(x) for x in m1.accept)
    f2 = set(int(x) for x in m2.accept)
    accept = {p for p in level if p[0] in f1 and p[1] in f2}
    return level, arcs, accept, {p: raw.get(p, 0) for p in level}


def compose_truncated(m1, m2, max_raw_arcs: int = 0, max_levels: int = 0):
    """Rule T replayed on the brute-force product.

    -> (states: set of pairs, expanded: set of pairs, arcs, truncated flag, n_raw)
    """
    delta, raw = full_product(m1, m2)
    by_src: Dict[Pair, List[ArcKey]] = defaultdict(list)
    for k in delta:
        by_src[k[0]].append(k)
    nq2 = int(m2.n_states)
    start = (int(m1.start), int(m2.start))
    states = {start}
    expanded: Set[Pair] = set()
    arcs: Dict[ArcKey, float] = {}
    frontier = [start]
    cum, lvl, truncated = 0, 0, 0
    while frontier:
        if max_levels > 0 and lvl == max_levels:
            truncated = 1
            break
        r_l = sum(raw.get(p, 0) for p in frontier)
        stop = False
        if max_raw_arcs == 0 or cum + r_l <= max_raw_arcs:
            todo = list(frontier)
        else:
            todo = []
            c = cum
            for p in sorted(frontier, key=lambda p: p[0] * nq2 + p[1]):
                if c + raw.get(p, 0) > max_raw_arcs:
                    break
                c += raw.get(p, 0)
                todo.append(p)
            truncated, stop = 1, True
        nxt = []
        for p in todo:
            expanded.add(p)
            cum += raw.get(p, 0)
            for k in by_src.get(p, ()):
                arcs[k] = delta[k]
                if k[3] not in states:
                    states.add(k[3])
                    nxt.append(k[3])
        if stop:
            break
        frontier = nxt
        lvl += 1
    return states, expanded, arcs, truncated, cum
