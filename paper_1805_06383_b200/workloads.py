"""Seeded synthetic transducers for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic: it only draws random
transducers (numpy, host) and returns plain arrays.  Both the CPU oracle
(`oracle/`) and the CUDA path consume the *same* arrays, so no cross-language
random generator is needed.  It imports neither of them.

The inputs stand in for the paper's Europarl-derived transducers
(§4.1, Table 1), which are not available; the
recipe is the one SURVEY.md §8(d) states and DESIGN.md repeats:

* Zipf:  p_c ∝ (c+1)^(-s) on the finite alphabet, inverse CDF, symbol id = rank.
* Spanning chain: arcs i -> i+1 (i = 0..|Q|-2) with random symbols, counted
  INSIDE the stated arc total; the remaining arcs have uniform src and tgt.
* Weights: 1 - U[0,1) cast to fp32, i.e. in (0, 1].
* M1: ilabel ∈ Σ uniform, olabel ∈ Γ Zipf.   M2: ilabel ∈ Γ Zipf, olabel ∈ Δ uniform.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, Tuple

import numpy as np

__all__ = ["Fst", "CONFIGS", "make_config", "make_lattices", "random_fst", "zipf_symbols"]


@dataclass
class Fst:
    """A weighted FST M = (Q, Σ, Γ, s, F, δ) as flat host arrays.

    States are 0..n_states-1, symbols 0..n-1 (no epsilon: 0 is an ordinary
    symbol).  Arcs are in arbitrary order; parallel duplicates are allowed.
    """

    n_states: int
    n_isyms: int
    n_osyms: int
    start: int
    src: np.ndarray      # int32 [n_arcs]
    ilabel: np.ndarray   # int32 [n_arcs]
    olabel: np.ndarray   # int32 [n_arcs]
    tgt: np.ndarray      # int32 [n_arcs]
    weight: np.ndarray   # float32 [n_arcs]
    accept: np.ndarray   # int32 [n_accept], distinct state ids
    meta: Dict[str, object] = field(default_factory=dict)

    @property
    def n_arcs(self) -> int:
        return int(self.src.shape[0])

    def check(self) -> None:
        n = self.n_arcs
        for a in (self.src, self.ilabel, self.olabel, self.tgt):
            assert a.dtype == np.int32 and a.shape == (n,)
        assert self.weight.dtype == np.float32 and self.weight.shape == (n,)
        assert self.accept.dtype == np.int32
        assert 0 <= self.start < self.n_states
        if n:
            assert self.src.min() >= 0 and self.src.max() < self.n_states
            assert self.tgt.min() >= 0 and self.tgt.max() < self.n_states
            assert self.ilabel.min() >= 0 and self.ilabel.max() < self.n_isyms
            assert self.olabel.min() >= 0 and self.olabel.max() < self.n_osyms


def _zipf_cdf(n: int, s: float) -> np.ndarray:
    p = np.arange(1, n + 1, dtype=np.float64) ** (-float(s))
    cdf = np.cumsum(p)
    cdf /= cdf[-1]
    return cdf


def zipf_symbols(rng: np.random.Generator, n_syms: int, s: float, size: int) -> np.ndarray:
    """`size` symbols with P(c) ∝ (c+1)^(-s), c in [0, n_syms); s = 0 is uniform."""
    if s == 0.0:
        return rng.integers(0, n_syms, size=size, dtype=np.int64).astype(np.int32)
    cdf = _zipf_cdf(n_syms, s)
    u = rng.random(size)
    c = np.searchsorted(cdf, u, side="right")
    return np.minimum(c, n_syms - 1).astype(np.int32)


def _weights(rng: np.random.Generator, n: int) -> np.ndarray:
    return (1.0 - rng.random(n)).astype(np.float32)  # (0, 1]


def random_fst(
    seed: int,
    n_states: int,
    n_isyms: int,
    n_osyms: int,
    n_arcs: int,
    *,
    inner_side: str,             # "out" for M1 (inner = olabel), "in" for M2 (inner = ilabel)
    inner_zipf: float = 0.0,
    n_accept: int = 1,
    chain: bool = True,
    src_weights: np.ndarray | None = None,
) -> Fst:
    """Uniform random transducer with an optional spanning chain from state 0.

    `src_weights` (length n_states, positive) makes the non-chain arcs' sources
    non-uniform (config 5's power-law out-degree).
    """
    assert inner_side in ("in", "out")
    rng = np.random.default_rng(seed)
    n_chain = n_states - 1 if chain else 0
    assert n_arcs >= n_chain
    n_rand = n_arcs - n_chain

    src = np.empty(n_arcs, np.int32)
    tgt = np.empty(n_arcs, np.int32)
    if n_chain:
        src[:n_chain] = np.arange(0, n_states - 1, dtype=np.int32)
        tgt[:n_chain] = np.arange(1, n_states, dtype=np.int32)
    if src_weights is None:
        src[n_chain:] = rng.integers(0, n_states, size=n_rand, dtype=np.int64)
    else:
        cdf = np.cumsum(np.asarray(src_weights, np.float64))
        cdf /= cdf[-1]
        src[n_chain:] = np.minimum(np.searchsorted(cdf, rng.random(n_rand), side="right"), n_states - 1)
    tgt[n_chain:] = rng.integers(0, n_states, size=n_rand, dtype=np.int64)

    if inner_side == "out":
        ilabel = rng.integers(0, n_isyms, size=n_arcs, dtype=np.int64).astype(np.int32)
        olabel = zipf_symbols(rng, n_osyms, inner_zipf, n_arcs)
    else:
        ilabel = zipf_symbols(rng, n_isyms, inner_zipf, n_arcs)
        olabel = rng.integers(0, n_osyms, size=n_arcs, dtype=np.int64).astype(np.int32)
    weight = _weights(rng, n_arcs)
    accept = np.sort(rng.choice(n_states, size=min(n_accept, n_states), replace=False)).astype(np.int32)
    fst = Fst(n_states, n_isyms, n_osyms, 0, src, ilabel, olabel, tgt, weight, accept)
    fst.check()
    return fst


def _powerlaw_degrees(rng: np.random.Generator, n: int, alpha: float, lo: float, hi: float) -> np.ndarray:
    """x iid with pdf ∝ x^(-alpha) on [lo, hi] (inverse CDF); SURVEY §8(d) reading of 'power-law α'."""
    u = rng.random(n)
    e = 1.0 - alpha
    return (lo ** e + u * (hi ** e - lo ** e)) ** (1.0 / e)


def _nlp_lattice(seed: int, n_pos: int, n_alt: int, vocab: int, s: float) -> Fst:
    """M1 of config 3: left-to-right lattice, n_alt DISTINCT Zipf words per position, in = out."""
    rng = np.random.default_rng(seed)
    cdf = _zipf_cdf(vocab, s)
    src, lab, w = [], [], []
    for i in range(n_pos):
        words: list[int] = []
        seen = set()
        while len(words) < n_alt:
            c = int(min(np.searchsorted(cdf, rng.random(), side="right"), vocab - 1))
            if c not in seen:
                seen.add(c)
                words.append(c)
        p = 1.0 - rng.random(n_alt)
        p = (p / p.sum()).astype(np.float32)        # normalised per state
        src += [i] * n_alt
        lab += words
        w += list(p)
    src_a = np.asarray(src, np.int32)
    lab_a = np.asarray(lab, np.int32)
    fst = Fst(n_pos + 1, vocab, vocab, 0, src_a, lab_a, lab_a.copy(), src_a + 1,
              np.asarray(w, np.float32), np.asarray([n_pos], np.int32))
    fst.check()
    return fst


def _nlp_bigram(seed: int, vocab: int, n_succ: int, s: float) -> Fst:
    """M2 of config 3: one state per word, n_succ DISTINCT Zipf successors per state, arc
    u -w:w-> w, weights normalised per state, start = 0, every state accepting.

    Successors are drawn by successive sampling: Zipf draws with replacement, keeping
    the first n_succ distinct symbols of each row (= sampling without replacement ∝ p).
    """
    rng = np.random.default_rng(seed)
    cdf = _zipf_cdf(vocab, s)
    succ = np.empty((vocab, n_succ), np.int32)
    todo = np.arange(vocab)
    n_draw = 4 * n_succ
    while todo.size:
        u = rng.random((todo.size, n_draw))
        d = np.minimum(np.searchsorted(cdf, u.reshape(-1), side="right"), vocab - 1).reshape(todo.size, n_draw)
        # first occurrence of each symbol per row: sort (symbol, position), mark heads, keep by position
        pos = np.argsort(d, axis=1, kind="stable")
        ds = np.take_along_axis(d, pos, axis=1)
        first = np.ones_like(ds, dtype=bool)
        first[:, 1:] = ds[:, 1:] != ds[:, :-1]
        keep = np.zeros_like(first)
        np.put_along_axis(keep, pos, first, axis=1)               # keep[r, j]: draw j is a first occurrence
        rank = np.cumsum(keep, axis=1)
        ok = rank[:, -1] >= n_succ
        sel = keep & (rank <= n_succ)
        rows_ok = np.nonzero(ok)[0]
        picked = d[rows_ok][sel[rows_ok]].reshape(rows_ok.size, n_succ)
        succ[todo[rows_ok]] = np.sort(picked, axis=1)
        todo = todo[~ok]
        n_draw *= 2
    w = 1.0 - rng.random((vocab, n_succ))
    w = (w / w.sum(axis=1, keepdims=True)).astype(np.float32)
    src = np.repeat(np.arange(vocab, dtype=np.int32), n_succ)
    lab = succ.reshape(-1)
    fst = Fst(vocab, vocab, vocab, 0, src, lab.copy(), lab.copy(), lab.copy(), w.reshape(-1),
              np.arange(vocab, dtype=np.int32))
    fst.check()
    return fst


# name -> (description, default seeds, default max_raw_arcs budget [0 = unlimited])
def _with_parallel_arcs(m: Fst, seed: int, frac: float) -> Fst:
    """m plus round(frac * arcs) copies of randomly chosen arcs (same source, labels, target; a new weight)."""
    rng = np.random.default_rng(seed + 20_000)
    pick = rng.integers(0, m.n_arcs, size=int(round(frac * m.n_arcs)))
    cat = lambda a: np.concatenate([a, a[pick]])          # noqa: E731
    out = Fst(m.n_states, m.n_isyms, m.n_osyms, m.start, cat(m.src), cat(m.ilabel), cat(m.olabel), cat(m.tgt),
              np.concatenate([m.weight, _weights(rng, len(pick))]), m.accept)
    out.check()
    return out


CONFIGS: Dict[str, Dict[str, object]] = {
    "tiny":   {"index": 0, "seeds": (102, 103), "max_raw_arcs": 0},
    "medium": {"index": 1, "seeds": (201, 202), "max_raw_arcs": 0},
    "nlp":    {"index": 2, "seeds": (301, 302), "max_raw_arcs": 0},
    "large":  {"index": 3, "seeds": (401, 402), "max_raw_arcs": 1_000_000_000},
    "skewed": {"index": 4, "seeds": (501, 502), "max_raw_arcs": 1_000_000_000},
    # not a BASELINE.json config: `medium` with parallel duplicate arcs, the workload of the merge on chip
    "dups":   {"index": 5, "seeds": (601, 602), "max_raw_arcs": 0},
}


def make_lattices(n: int, seed0: int = 301, scale: float = 1.0) -> list:
    """n seeded word lattices of config `nlp`'s shape (50 positions x 8 alternatives over the same vocabulary): the many
    left operands of ONE language model, the paper's translation use case."""
    vocab = max(200, int(round(30_000 * scale)))
    return [_nlp_lattice(seed0 + 1000 * (k + 1), 50, 8, vocab, 1.1) for k in range(n)]


def make_config(name: str, seeds: Tuple[int, int] | None = None, scale: float = 1.0) -> Tuple[Fst, Fst]:
    """Return (M1, M2) for one of BASELINE.json's configs.

    `scale` < 1 shrinks the random configs proportionally (states, alphabets and
    arcs) for parity tests the oracle finishes in seconds; 1.0 is the stated size.
    """
    if name not in CONFIGS:
        raise KeyError(f"unknown config {name!r}; have {sorted(CONFIGS)}")
    s1, s2 = seeds if seeds is not None else CONFIGS[name]["seeds"]  # type: ignore[misc]

    def sc(x: int, lo: int = 2) -> int:
        return max(lo, int(round(x * scale)))

    if name == "tiny":
        m1 = random_fst(s1, 50, 20, 16, 300, inner_side="out", n_accept=5)
        m2 = random_fst(s2, 40, 16, 20, 250, inner_side="in", n_accept=5)
    elif name == "medium":
        q, sig, gam, arcs = sc(10_000), sc(1_000), sc(1_000), sc(200_000)
        m1 = random_fst(s1, q, sig, gam, arcs, inner_side="out", inner_zipf=1.0, n_accept=max(1, q // 100))
        m2 = random_fst(s2, q, gam, sig, arcs, inner_side="in", inner_zipf=1.0, n_accept=max(1, q // 100))
    elif name == "nlp":
        vocab = sc(30_000, 200)
        m1 = _nlp_lattice(s1, 50, 8, vocab, 1.1)
        m2 = _nlp_bigram(s2, vocab, min(100, vocab // 2), 1.1)
    elif name == "large":
        q, sig, gam, arcs = sc(100_000), sc(20_000), sc(5_000), sc(5_000_000)
        m1 = random_fst(s1, q, sig, gam, arcs, inner_side="out", inner_zipf=1.1, n_accept=max(1, q // 100))
        m2 = random_fst(s2, q, gam, sig, arcs, inner_side="in", inner_zipf=1.1, n_accept=max(1, q // 100))
    elif name == "dups":
        # every state can hold duplicates (10 % of the arcs are repeated with a new weight: same source, labels and
        # target), while two states seldom share an inner symbol: many small sources whose raw arcs must be merged
        q, sig, gam, arcs = sc(10_000), sc(1_000), sc(1_000), sc(200_000)
        m1 = _with_parallel_arcs(random_fst(s1, q, sig, gam, arcs, inner_side="out", inner_zipf=1.0, n_accept=max(1, q // 100)), s1, 0.1)
        m2 = _with_parallel_arcs(random_fst(s2, q, gam, sig, arcs, inner_side="in", inner_zipf=1.0, n_accept=max(1, q // 100)), s2, 0.1)
    else:  # skewed
        q, arcs = sc(2_000), sc(1_000_000)
        r1 = np.random.default_rng(s1 + 10_000)
        r2 = np.random.default_rng(s2 + 10_000)
        x1 = _powerlaw_degrees(r1, q, 1.8, 1.0, 1e6)
        x2 = _powerlaw_degrees(r2, q, 1.8, 1.0, 1e6)
        m1 = random_fst(s1, q, 10, 50, arcs, inner_side="out", inner_zipf=1.5,
                        n_accept=max(1, q // 100), src_weights=x1)
        m2 = random_fst(s2, q, 50, 10, arcs, inner_side="in", inner_zipf=1.5,
                        n_accept=max(1, q // 100), src_weights=x2)
    for m, s in ((m1, s1), (m2, s2)):
        m.meta.update({"config": name, "seed": s, "scale": scale})
    return m1, m2
