"""The boundary items of SURVEY §8(b) beyond the compose call itself (`-m gpu`): allocator hooks (PyTorch's caching
allocator owns every device byte of a call), error codes for bad arguments, operands packed once and reused."""
from __future__ import annotations

import gc

import numpy as np
import pytest

from paper_1805_06383_b200 import workloads
from test_gpu_parity import check_parity, fstc  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("small_path", [1, 0])
def test_allocator_hooks_route_every_allocation_through_torch(fstc, small_path):
    """With fstc_opts_t.alloc / dealloc set to torch's caching allocator: the result is the same, the hooks are called in
    pairs (temporaries inside the call, the arrays of the result and of the packed operands on release), and what the
    result holds is visible in torch.cuda.memory_allocated()."""
    import torch
    m1, m2 = workloads.make_config("medium", scale=0.02) if small_path == 1 else workloads.make_config("tiny")
    fstc.fstc_trim_pool()
    torch.cuda.synchronize()
    base = torch.cuda.memory_allocated()
    log0 = dict(fstc.ALLOC_LOG)
    p1 = fstc.fstc_pack(fstc.DeviceFst.from_host(m1), 1, allocator="torch")
    p2 = fstc.fstc_pack(fstc.DeviceFst.from_host(m2), 2, allocator="torch")
    res = fstc.fstc_compose_packed(p1, p2, allocator="torch", small_path=small_path)
    n_alloc = fstc.ALLOC_LOG["alloc"] - log0["alloc"]
    held = n_alloc - (fstc.ALLOC_LOG["dealloc"] - log0["dealloc"])
    assert n_alloc > 10 and 1 <= held <= 10 + 10 + 8          # two packed operands and one result are still alive
    assert torch.cuda.memory_allocated() - base >= 20 * res.n_arcs + 8 * res.n_states
    check_parity(fstc, m1, m2, result=res)
    res.free(); p1.free(); p2.free()
    gc.collect()
    torch.cuda.synchronize()
    assert fstc.ALLOC_LOG["alloc"] - log0["alloc"] == fstc.ALLOC_LOG["dealloc"] - log0["dealloc"]
    assert torch.cuda.memory_allocated() == base


def test_half_set_hooks_are_an_argument_error(fstc):
    import ctypes
    m1, m2 = workloads.make_config("tiny")
    o = fstc._opts(allocator="torch")
    o.dealloc = None
    s1, k1 = fstc._marshal(fstc.DeviceFst.from_host(m1))
    out = ctypes.c_void_p()
    rc = fstc.lib().fstc_pack(ctypes.addressof(s1), 1, ctypes.addressof(o), 0, ctypes.byref(out))
    assert rc == fstc.ERR_ARG and not out.value


def test_packed_operand_is_reused_across_compositions(fstc):
    m1, m2 = workloads.make_config("tiny")
    p1 = fstc.fstc_pack(fstc.DeviceFst.from_host(m1), 1)
    p2 = fstc.fstc_pack(fstc.DeviceFst.from_host(m2), 2)
    a = fstc.fstc_compose_packed(p1, p2)
    b = fstc.fstc_compose_packed(p1, p2, max_levels=3)
    check_parity(fstc, m1, m2, result=a)
    check_parity(fstc, m1, m2, max_levels=3, result=b)
    with pytest.raises(fstc.FstcError) as e:                  # operands on the wrong sides
        fstc.fstc_compose_packed(p2, p1)
    assert e.value.code == fstc.ERR_ARG


def _pinned(n_arcs, n_states):
    import torch
    i32 = lambda n: torch.empty(n, dtype=torch.int32).pin_memory()
    return {"pair": i32(2 * n_states), "src": i32(n_arcs), "ilabel": i32(n_arcs), "olabel": i32(n_arcs), "tgt": i32(n_arcs),
            "weight": torch.empty(n_arcs, dtype=torch.float32).pin_memory(), "accept": i32(n_states),
            "expanded": torch.empty(n_states, dtype=torch.uint8).pin_memory()}


def _host_view(res, bufs):
    """The result as the spilled host arrays hold it, with the attribute names check_parity reads."""
    from types import SimpleNamespace
    ns, na = res.n_states, res.n_arcs
    return SimpleNamespace(n_states=ns, n_arcs=na, n_raw_arcs=res.n_raw_arcs, n_levels=res.n_levels, truncated=res.truncated,
                           n_expanded=res.n_expanded, n_accept=res.n_accept, stats=res.stats,
                           pair=bufs["pair"][:2 * ns].view(ns, 2), src=bufs["src"][:na], ilabel=bufs["ilabel"][:na],
                           olabel=bufs["olabel"][:na], tgt=bufs["tgt"][:na], weight=bufs["weight"][:na],
                           accept=bufs["accept"][:res.n_accept], expanded=bufs["expanded"][:ns])


@pytest.mark.parametrize("keep_device", [False, True])
@pytest.mark.parametrize("config,scale,budget,resolve_mode", [("medium", 0.05, 0, 0), ("skewed", 0.05, 2_000_000, 0),
                                                              ("large", 0.02, 3_000_000, 2)])
def test_host_spill_streams_finished_levels(fstc, config, scale, budget, resolve_mode, keep_device):
    """fstc_spill_t: the arcs and pairs of every finished level are copied to pinned host memory on a second stream while
    the next level runs; the host arrays alone must equal the oracle's result.  Without a device
    copy the result's arc arrays are NULL and 20 bytes of HBM per arc are reported as never held."""
    m1, m2 = workloads.make_config(config, scale=scale)
    a, b = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    plain = fstc.fstc_compose(a, b, max_raw_arcs=budget, resolve_mode=resolve_mode, small_path=1)
    bufs = _pinned(plain.n_arcs + 7, plain.n_states + 3)
    for t in bufs.values():
        t.fill_(-1 if t.dtype != fstc_uint8() else 255)
    res = fstc.fstc_compose(a, b, max_raw_arcs=budget, resolve_mode=resolve_mode, small_path=1, spill=bufs, spill_keep_device=keep_device)
    assert (res.n_states, res.n_arcs) == (plain.n_states, plain.n_arcs)
    assert res.stats["spill_bytes"] >= 20 * res.n_arcs + 8 * res.n_states
    if keep_device:
        assert res.stats["spill_bytes_saved"] == 0 and res.src is not None
        check_parity(fstc, m1, m2, max_raw_arcs=budget, result=res)
    else:
        assert res.src is None and res.weight is None and res.stats["spill_bytes_saved"] == 20 * res.n_arcs
    check_parity(fstc, m1, m2, max_raw_arcs=budget, result=_host_view(res, bufs))


def fstc_uint8():
    import torch
    return torch.uint8


def test_host_spill_capacity_is_checked(fstc):
    m1, m2 = workloads.make_config("medium", scale=0.03)
    a, b = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    with pytest.raises(fstc.FstcError) as e:
        fstc.fstc_compose(a, b, small_path=1, spill=_pinned(1000, 1 << 22))
    assert e.value.code == fstc.ERR_CAPACITY
    with pytest.raises(fstc.FstcError) as e:
        fstc.fstc_compose(a, b, small_path=1, spill=_pinned(1 << 24, 100))
    assert e.value.code == fstc.ERR_CAPACITY
    fstc.fstc_compose(a, b, small_path=1)                       # and the library still works after the failed calls


@pytest.mark.parametrize("config,scale,budget,kw", [
    ("medium", 0.05, 0, {}), ("medium", 0.03, 0, {"resolve_mode": 3}), ("large", 0.02, 3_000_000, {"resolve_mode": 2}),
    ("skewed", 0.05, 2_000_000, {}), ("skewed", 0.05, 1_000_000, {"merge_mode": 2}), ("skewed", 0.05, 1_000_000, {"merge_mode": 1}),
    ("skewed", 0.05, 1_500_000, {"resolve_mode": 2}), ("tiny", 1.0, 0, {}), ("tiny", 1.0, 0, {"merge_mode": 2}),
])
def test_deterministic_ids_and_arc_order(fstc, config, scale, budget, kw, monkeypatch):
    """fstc_opts_t.deterministic: two runs give bit-identical pair[], src, tgt, ilabel, olabel; inside every BFS level the
    new ids ascend with the pair key; and the result still equals the oracle's."""
    import torch
    m1, m2 = workloads.make_config(config, scale=scale)
    a, b = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    runs = [fstc.fstc_compose(a, b, max_raw_arcs=budget, deterministic=True, **kw) for _ in range(2)]
    r0, r1 = runs
    assert r0.stats["small_path"] == 0
    for name in ("pair", "src", "tgt", "ilabel", "olabel", "accept", "expanded"):
        assert torch.equal(getattr(r0, name), getattr(r1, name)), name
    key = r0.pair[:, 0].long() * m2.n_states + r0.pair[:, 1].long()
    lo = 1
    for n_new in r0.stats["level_new_states"]:
        k = key[lo:lo + n_new]
        assert bool((k[1:] > k[:-1]).all())
        lo += n_new
    assert lo == r0.n_states
    check_parity(fstc, m1, m2, max_raw_arcs=budget, merge_mode=kw.get("merge_mode", 0), result=r0)
    if config == "skewed" and not kw:
        monkeypatch.setenv("FSTC_NO_GROUP_MERGE", "1")          # every duplicate-prone source through sort + reduce
        r2 = fstc.fstc_compose(a, b, max_raw_arcs=budget, deterministic=True)
        r3 = fstc.fstc_compose(a, b, max_raw_arcs=budget, deterministic=True)
        assert r2.stats["n_raw_sorted"] > 0 and torch.equal(r2.tgt, r3.tgt) and torch.equal(r2.pair, r3.pair)
        assert torch.equal(r2.ilabel, r3.ilabel) and torch.equal(r2.olabel, r3.olabel)
        check_parity(fstc, m1, m2, max_raw_arcs=budget, result=r2)


@pytest.mark.parametrize("config,scale,chunk,kw", [
    ("tiny", 1.0, 100, {}), ("tiny", 1.0, 7, {"merge_mode": 2}), ("medium", 0.05, 200_000, {}),
    ("medium", 0.03, 50_000, {"resolve_mode": 2}), ("skewed", 0.05, 2_000_000, {"max_levels": 2}),
    ("large", 0.02, 600_000, {"max_levels": 3, "resolve_mode": 2}), ("medium", 0.03, 40_000, {"deterministic": True}),
])
def test_levels_too_big_for_the_workspace_go_chunk_by_chunk(fstc, config, scale, chunk, kw, monkeypatch):
    """FSTC_CHUNK_ARCS lowers the number of raw arcs a level may hold in one piece (by default about half the device memory
    / 72 bytes): bigger levels are expanded as id ranges of the frontier, one after the other; the result is the same."""
    monkeypatch.setenv("FSTC_CHUNK_ARCS", str(chunk))
    m1, m2 = workloads.make_config(config, scale=scale)
    a, b = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    res = fstc.fstc_compose(a, b, small_path=1, **kw)
    assert res.stats["n_chunks"] >= 3
    check_parity(fstc, m1, m2, merge_mode=kw.get("merge_mode", 0), max_levels=kw.get("max_levels", 0), result=res)
    # a budget cut inside a big level: the level is not chunked (rule T orders it by key), the result is still exact
    budget = max(1, res.n_raw_arcs // 2)
    cut = fstc.fstc_compose(a, b, small_path=1, max_raw_arcs=budget, **kw)
    check_parity(fstc, m1, m2, merge_mode=kw.get("merge_mode", 0), max_levels=kw.get("max_levels", 0), max_raw_arcs=budget, result=cut)
