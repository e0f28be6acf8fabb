"""Shared test helpers: tiny hand-made transducers and canonical (pair-coordinate) forms.

No method arithmetic lives here beyond re-keying results for comparison.
"""
from __future__ import annotations

from typing import Dict, Iterable, Tuple

import numpy as np

from paper_1805_06383_b200.workloads import Fst


def fst_from_arcs(n_states: int, n_isyms: int, n_osyms: int, arcs: Iterable[Tuple[int, int, int, int, float]],
                  start: int = 0, accept: Iterable[int] = ()) -> Fst:
    arcs = list(arcs)
    cols = list(zip(*arcs)) if arcs else [(), (), (), (), ()]
    f = Fst(n_states, n_isyms, n_osyms, start,
            np.asarray(cols[0], np.int32), np.asarray(cols[1], np.int32), np.asarray(cols[2], np.int32),
            np.asarray(cols[3], np.int32), np.asarray(cols[4], np.float32),
            np.asarray(sorted(set(accept)), np.int32))
    f.check()
    return f


def messy_random_fst(seed: int, n_states: int, n_isyms: int, n_osyms: int, n_arcs: int, n_accept: int = 2,
                     start: int = 0, dup_frac: float = 0.15, zero_frac: float = 0.05) -> Fst:
    """Small random machine WITHOUT a spanning chain: unreachable states, arc-less states,
    self loops, parallel duplicate arcs (same src,in,out,tgt) and a few zero weights."""
    rng = np.random.default_rng(seed)
    src = rng.integers(0, n_states, n_arcs)
    tgt = rng.integers(0, n_states, n_arcs)
    il = rng.integers(0, n_isyms, n_arcs)
    ol = rng.integers(0, n_osyms, n_arcs)
    n_dup = int(n_arcs * dup_frac)
    if n_dup and n_arcs > 1:
        pick = rng.integers(0, n_arcs, n_dup)
        into = rng.integers(0, n_arcs, n_dup)
        src[into], tgt[into], il[into], ol[into] = src[pick], tgt[pick], il[pick], ol[pick]
    w = (1.0 - rng.random(n_arcs)).astype(np.float32)
    w[rng.random(n_arcs) < zero_frac] = 0.0
    acc = rng.choice(n_states, size=min(n_accept, n_states), replace=False)
    f = Fst(n_states, n_isyms, n_osyms, start, src.astype(np.int32), il.astype(np.int32), ol.astype(np.int32),
            tgt.astype(np.int32), w, np.sort(acc).astype(np.int32))
    f.check()
    return f


ArcDict = Dict[Tuple[Tuple[int, int], int, int, Tuple[int, int]], float]


def canon_arcs(q1, q2, src, tgt, a, b, w) -> ArcDict:
    """arcs -> {((q1,q2)_src, a, b, (q1,q2)_tgt): weight}; duplicate keys are summed (fp64)."""
    out: ArcDict = {}
    for s, t, x, y, p in zip(src, tgt, a, b, w):
        k = ((int(q1[s]), int(q2[s])), int(x), int(y), (int(q1[t]), int(q2[t])))
        out[k] = out.get(k, 0.0) + float(p)
    return out


def canon_states(q1, q2):
    return sorted(zip((int(x) for x in q1), (int(x) for x in q2)))


def canon_arc_table(q1, q2, src, tgt, a, b, w, n_q2: int):
    """Vectorised canonical form: rows (k_src, k_tgt, a, b) sorted lexicographically + weights in that order."""
    q1 = np.asarray(q1, np.int64); q2 = np.asarray(q2, np.int64)
    key = q1 * n_q2 + q2
    ks, kt = key[np.asarray(src, np.int64)], key[np.asarray(tgt, np.int64)]
    a = np.asarray(a, np.int64); b = np.asarray(b, np.int64)
    order = np.lexsort((b, a, kt, ks))
    table = np.stack([ks[order], kt[order], a[order], b[order]], axis=1)
    return table, np.asarray(w)[order]
