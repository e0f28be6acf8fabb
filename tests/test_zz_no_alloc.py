"""fstc_compose_static (include/fstc.h): the one entry point that allocates nothing — result arrays from the caller, the
kernel's scratch in a static device array of the library.  Its output is compared with the EXISTING paths' (the
one-block path of fstc_compose_packed and the level-synchronous path) on the same packed operands, in pair coordinates
(state numbers are implementation-defined), structure exact, weights within the rtol 1e-5 of the other GPU tests; on two
and more calls in a row, because every call shares the one scratch array and finds the last call's contents in it.

Named test_zz_* so that pytest collects it LAST: a failure here cannot hide another test under `pytest -x`.  `-m gpu`."""
from __future__ import annotations

import numpy as np
import pytest

from paper_1805_06383_b200 import workloads
from helpers import canon_arc_table, messy_random_fst

pytestmark = pytest.mark.gpu

RTOL = 1e-5
SMALL_OFF, SMALL_ONLY = 1, 2


@pytest.fixture(scope="module")
def fstc():
    import torch
    assert torch.cuda.is_available()
    from paper_1805_06383_b200 import fstc as mod
    mod.lib()                          # fails loudly if the CUDA library is missing
    return mod


def _problems():
    """(name, m1, m2): the `tiny` config (1 574 states, 3 740 arcs, 17 levels) and two random machines with many
    parallel arcs (merges) — all within the one-block caps."""
    out = [("tiny",) + tuple(workloads.make_config("tiny"))]
    for seed, n1, sig, gam, a1, n2, dlt, a2 in [(5, 8, 2, 2, 60, 7, 2, 50), (7, 40, 3, 5, 400, 30, 3, 300)]:
        out.append((f"random{seed}", messy_random_fst(seed, n1, sig, gam, a1), messy_random_fst(seed + 100, n2, gam, dlt, a2)))
    return out


def _canon(pair, src, tgt, il, ol, w, expanded, accept, nq2):
    pair = pair.cpu().numpy().astype(np.int64)
    q1, q2 = pair[:, 0], pair[:, 1]
    tab, cw = canon_arc_table(q1, q2, src.cpu().numpy(), tgt.cpu().numpy(), il.cpu().numpy(), ol.cpu().numpy(),
                              w.cpu().numpy(), nq2)
    keys = q1 * nq2 + q2
    o = np.argsort(keys)
    return {"start": tuple(pair[0]), "keys": keys[o], "expanded": expanded.cpu().numpy()[o],
            "accept": np.sort(keys[accept.cpu().numpy().astype(np.int64)]), "tab": tab, "w": cw,
            "src_sorted": bool((np.diff(src.cpu().numpy()) >= 0).all())}


def _canon_static(d, nq2):
    assert d["status"] == 0
    c = _canon(d["pair"], d["src"], d["tgt"], d["ilabel"], d["olabel"], d["weight"], d["expanded"], d["accept"], nq2)
    c["counts"] = tuple(d[k] for k in ("n_states", "n_arcs", "n_raw_arcs", "n_accept", "n_expanded", "n_levels", "truncated"))
    return c


def _canon_existing(r, nq2):
    c = _canon(r.pair, r.src, r.tgt, r.ilabel, r.olabel, r.weight, r.expanded, r.accept, nq2)
    c["counts"] = (r.n_states, r.n_arcs, r.n_raw_arcs, r.n_accept, r.n_expanded, r.n_levels, r.truncated)
    return c


def _same(a, b):
    assert a["counts"] == b["counts"]
    assert a["start"] == b["start"] and a["src_sorted"] and b["src_sorted"]
    assert (a["keys"] == b["keys"]).all() and (a["expanded"] == b["expanded"]).all()
    assert (a["accept"] == b["accept"]).all()
    assert a["tab"].shape == b["tab"].shape and (a["tab"] == b["tab"]).all()
    np.testing.assert_allclose(a["w"], b["w"], rtol=RTOL, atol=0)


@pytest.mark.parametrize("opts", [{}, {"merge_mode": 1}, {"max_raw_arcs": 777}, {"max_levels": 3}])
def test_calls_in_a_row_match_the_existing_paths(fstc, opts):
    """One set of buffers, one scratch array: tiny, a small machine, another, then tiny AGAIN — every call must give the
    existing paths' result although it finds the previous call's table, work lists and arrays in place."""
    import torch
    probs = _problems()
    packed = [(name, fstc.fstc_pack(m1, 1), fstc.fstc_pack(m2, 2), m2.n_states) for name, m1, m2 in probs]
    bufs = fstc.StaticBuffers(8192, 65536)
    first = {}
    for name, p1, p2, nq2 in packed + packed[:1]:
        fstc.fstc_compose_static(p1, p2, bufs, **opts)
        torch.cuda.synchronize()
        new = _canon_static(bufs.read(), nq2)
        one_block = fstc.fstc_compose_packed(p1, p2, small_path=SMALL_ONLY, **opts)
        assert one_block.stats["small_path"] == 1
        _same(new, _canon_existing(one_block, nq2))
        _same(new, _canon_existing(fstc.fstc_compose_packed(p1, p2, small_path=SMALL_OFF, **opts), nq2))
        if name in first:                      # the same problem again, after other problems went through the scratch
            _same(new, first[name])
            assert (new["w"] == first[name]["w"]).all()
        first.setdefault(name, new)
        assert new["counts"][0] > 1 and new["counts"][1] > 0


def test_two_calls_back_to_back_on_one_stream(fstc):
    """No synchronisation between the calls: stream order alone keeps them apart on the shared scratch."""
    import torch
    (_, a1, a2), (_, b1, b2) = _problems()[:2]
    pa, pb = (fstc.fstc_pack(a1, 1), fstc.fstc_pack(a2, 2)), (fstc.fstc_pack(b1, 1), fstc.fstc_pack(b2, 2))
    out_a, out_b, out_c = (fstc.StaticBuffers(4096, 16384) for _ in range(3))
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        fstc.fstc_compose_static(*pa, out_a)
        fstc.fstc_compose_static(*pb, out_b)
        fstc.fstc_compose_static(*pa, out_c, stream=s)
    s.synchronize()
    ref_a = _canon_existing(fstc.fstc_compose_packed(*pa, small_path=SMALL_ONLY), a2.n_states)
    ref_b = _canon_existing(fstc.fstc_compose_packed(*pb, small_path=SMALL_ONLY), b2.n_states)
    _same(_canon_static(out_a.read(), a2.n_states), ref_a)
    _same(_canon_static(out_b.read(), b2.n_states), ref_b)
    _same(_canon_static(out_c.read(), a2.n_states), ref_a)


def test_the_call_allocates_nothing(fstc):
    """Free device memory does not move over the calls, and the call can be CAPTURED into a CUDA graph (a cudaMalloc,
    a pool allocation that has to grow, a synchronisation or a pageable copy would all break the capture); the replayed
    graph gives the existing path's result, twice."""
    import torch
    _, m1, m2 = _problems()[0]
    p1, p2 = fstc.fstc_pack(m1, 1), fstc.fstc_pack(m2, 2)
    ref = _canon_existing(fstc.fstc_compose_packed(p1, p2, small_path=SMALL_ONLY), m2.n_states)
    bufs = fstc.StaticBuffers(8192, 65536)
    fstc.fstc_compose_static(p1, p2, bufs)                   # the first call on a device resolves the scratch address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        fstc.fstc_compose_static(p1, p2, bufs)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    _same(_canon_static(bufs.read(), m2.n_states), ref)

    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        fstc.fstc_compose_static(p1, p2, bufs)               # (torch's current stream is the capturing stream here)
    for _ in range(2):
        for t in (bufs.header, bufs.src, bufs.tgt, bufs.weight, bufs.pair):
            t.zero_()
        g.replay()
        torch.cuda.synchronize()
        _same(_canon_static(bufs.read(), m2.n_states), ref)


def test_limits_and_refusals(fstc):
    import torch
    _, m1, m2 = _problems()[0]
    p1, p2 = fstc.fstc_pack(m1, 1), fstc.fstc_pack(m2, 2)
    with pytest.raises(fstc.FstcError) as e:                 # beyond the stated maximum: a clear error, nothing launched
        fstc.fstc_compose_static(p1, p2, fstc.StaticBuffers(fstc.STATIC_MAX_STATES + 1, 1024))
    assert e.value.code == fstc.ERR_CAPACITY and "FSTC_STATIC_MAX_STATES" in str(e.value)
    with pytest.raises(fstc.FstcError) as e:
        fstc.fstc_compose_static(p1, p2, fstc.StaticBuffers(1024, 1024), merge_mode=fstc.MERGE_SORT_ALL)
    assert e.value.code == fstc.ERR_ARG
    with pytest.raises(fstc.FstcError) as e:
        fstc.fstc_compose_static(p2, p1, fstc.StaticBuffers(1024, 1024))
    assert e.value.code == fstc.ERR_ARG
    # buffers too small for the problem: no error, the header says so; the next call is not disturbed by the aborted one
    small = fstc.StaticBuffers(64, 100)
    fstc.fstc_compose_static(p1, p2, small)
    torch.cuda.synchronize()
    assert small.read()["status"] == 1
    big = fstc.StaticBuffers(fstc.STATIC_MAX_STATES, 1 << 20)    # the largest visited table the scratch holds
    fstc.fstc_compose_static(p1, p2, big)
    torch.cuda.synchronize()
    _same(_canon_static(big.read(), m2.n_states),
          _canon_existing(fstc.fstc_compose_packed(p1, p2, small_path=SMALL_ONLY), m2.n_states))
