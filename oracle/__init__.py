"""ORACLE — TEST INFRASTRUCTURE ONLY (see fst_compose_oracle.cpp for what it computes and why).

ctypes front end of the plain serial C++ composer.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_1805_06383_b200 (inputs are
passed in as plain numpy arrays / any object with the Fst field names).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import List

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fst_compose_oracle.cpp")
_LIB = os.path.join(_HERE, "libfst_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C++ oracle with g++ -O2 (rebuilds when the source is newer)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


class _InFst(ctypes.Structure):
    _fields_ = [
        ("n_states", ctypes.c_int32), ("n_isyms", ctypes.c_int32), ("n_osyms", ctypes.c_int32),
        ("start", ctypes.c_int32), ("n_arcs", ctypes.c_int64),
        ("src", ctypes.c_void_p), ("ilabel", ctypes.c_void_p), ("olabel", ctypes.c_void_p),
        ("tgt", ctypes.c_void_p), ("weight", ctypes.c_void_p),
        ("n_accept", ctypes.c_int32), ("accept", ctypes.c_void_p),
    ]


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P, I, L = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64
        lib.fsto_compose.restype = P
        lib.fsto_compose.argtypes = [P, P, I, L, I, I, I]
        lib.fsto_info.argtypes = [P, P]
        lib.fsto_seconds.restype = ctypes.c_double
        lib.fsto_seconds.argtypes = [P]
        lib.fsto_get_states.argtypes = [P, P, P, P, P]
        lib.fsto_get_arcs.argtypes = [P, P, P, P, P, P]
        lib.fsto_get_accept.argtypes = [P, P]
        lib.fsto_get_levels.argtypes = [P, P, P]
        lib.fsto_free.argtypes = [P]
        lib.fsto_prepare.restype = P
        lib.fsto_prepare.argtypes = [P, P]
        lib.fsto_raw_count.restype = L
        lib.fsto_raw_count.argtypes = [P, ctypes.c_int32, ctypes.c_int32]
        lib.fsto_expand_pair.restype = L
        lib.fsto_expand_pair.argtypes = [P, ctypes.c_int32, ctypes.c_int32, I]
        lib.fsto_pair_arcs.argtypes = [P, P, P, P, P, P]
        lib.fsto_prepared_free.argtypes = [P]
        _lib = lib
    return _lib


def _marshal(fst):
    """-> (_InFst, keepalive list).  `fst` is any object with the Fst field names."""
    keep = []

    def arr(x, dt):
        a = np.ascontiguousarray(np.asarray(x), dtype=dt)
        keep.append(a)
        return a.ctypes.data

    s = _InFst()
    s.n_states, s.n_isyms, s.n_osyms, s.start = int(fst.n_states), int(fst.n_isyms), int(fst.n_osyms), int(fst.start)
    s.n_arcs = int(np.asarray(fst.src).shape[0])
    s.src, s.ilabel = arr(fst.src, np.int32), arr(fst.ilabel, np.int32)
    s.olabel, s.tgt = arr(fst.olabel, np.int32), arr(fst.tgt, np.int32)
    s.weight = arr(fst.weight, np.float32)
    s.n_accept = int(np.asarray(fst.accept).shape[0])
    s.accept = arr(fst.accept, np.int32)
    if int(fst.n_osyms) < 0 or int(fst.n_isyms) < 0:
        raise ValueError("negative alphabet size")
    return s, keep


@dataclass
class OracleResult:
    """M1∘M2 as the oracle built it.  State i is the pair (q1[i], q2[i]); state 0 = (s1,s2).

    Ids are the oracle's own (creation order); compare in pair coordinates.
    Weights are fp64 sums of exact fp64 products.
    """
    q1: np.ndarray
    q2: np.ndarray
    level: np.ndarray
    expanded: np.ndarray
    src: np.ndarray
    tgt: np.ndarray
    ilabel: np.ndarray
    olabel: np.ndarray
    weight: np.ndarray
    accept: np.ndarray
    level_raw: np.ndarray
    level_size: np.ndarray
    n_states: int
    n_arcs: int
    n_raw_arcs: int
    n_levels: int
    truncated: int
    n_expanded: int
    seconds: float
    n_q2: int

    def state_keys(self) -> np.ndarray:
        return self.q1.astype(np.int64) * self.n_q2 + self.q2.astype(np.int64)


def compose(m1, m2, *, merge: bool = True, max_raw_arcs: int = 0, max_levels: int = 0,
            keep_arcs: bool = True, force_map: bool = False) -> OracleResult:
    """Serial composition by Algorithm 1 + merge (:65) + budget rule T."""
    if int(m1.n_osyms) != int(m2.n_isyms):
        raise ValueError("inner alphabets differ (PAPER.md:45)")
    lib = _load()
    s1, k1 = _marshal(m1)
    s2, k2 = _marshal(m2)
    h = lib.fsto_compose(ctypes.addressof(s1), ctypes.addressof(s2), int(merge), int(max_raw_arcs),
                         int(max_levels), int(keep_arcs), int(force_map))
    try:
        info = np.zeros(8, np.int64)
        lib.fsto_info(h, info.ctypes.data)
        ns, na, nraw, nacc, nlev, trunc, nexp, kept = (int(x) for x in info)
        q1 = np.empty(ns, np.int32); q2 = np.empty(ns, np.int32)
        level = np.empty(ns, np.int32); expanded = np.empty(ns, np.uint8)
        lib.fsto_get_states(h, q1.ctypes.data, q2.ctypes.data, level.ctypes.data, expanded.ctypes.data)
        src = np.empty(kept, np.int64); tgt = np.empty(kept, np.int64)
        a = np.empty(kept, np.int32); b = np.empty(kept, np.int32); w = np.empty(kept, np.float64)
        lib.fsto_get_arcs(h, src.ctypes.data, tgt.ctypes.data, a.ctypes.data, b.ctypes.data, w.ctypes.data)
        acc = np.empty(nacc, np.int64)
        lib.fsto_get_accept(h, acc.ctypes.data)
        lraw = np.empty(nlev, np.int64); lsize = np.empty(nlev, np.int64)
        lib.fsto_get_levels(h, lraw.ctypes.data, lsize.ctypes.data)
        secs = float(lib.fsto_seconds(h))
    finally:
        lib.fsto_free(h)
    del k1, k2
    return OracleResult(q1, q2, level, expanded, src, tgt, a, b, w, acc, lraw, lsize, ns, na, nraw, nlev,
                        trunc, nexp, secs, int(m2.n_states))


class PairExpander:
    """Expand single state pairs by the definition (sampled checks at full size)."""

    def __init__(self, m1, m2):
        self._lib = _load()
        s1, self._k1 = _marshal(m1)
        s2, self._k2 = _marshal(m2)
        self._h = self._lib.fsto_prepare(ctypes.addressof(s1), ctypes.addressof(s2))

    def raw_count(self, q1: int, q2: int) -> int:
        return int(self._lib.fsto_raw_count(self._h, int(q1), int(q2)))

    def expand(self, q1: int, q2: int, merge: bool = True):
        """-> (r1, r2, a, b, w) arrays of the pair's outgoing arcs, sorted by (r1,r2,a,b) when merged."""
        n = int(self._lib.fsto_expand_pair(self._h, int(q1), int(q2), int(merge)))
        r1 = np.empty(n, np.int32); r2 = np.empty(n, np.int32)
        a = np.empty(n, np.int32); b = np.empty(n, np.int32); w = np.empty(n, np.float64)
        self._lib.fsto_pair_arcs(self._h, r1.ctypes.data, r2.ctypes.data, a.ctypes.data, b.ctypes.data,
                                 w.ctypes.data)
        return r1, r2, a, b, w

    def close(self):
        if self._h:
            self._lib.fsto_prepared_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
