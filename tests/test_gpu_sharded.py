"""FSTC_RESOLVE_EXTERNAL on one GPU (`-m gpu`): the library expands the pairs, every batch of target keys goes through
the caller's callback (paper_1805_06383_b200/sharded.py: KeyExchange over a process group of ONE rank here, so the
all-to-all is the identity) and comes back as global ids.  The shard of the only rank must be the whole composition.  The
multi-rank exchange itself is covered on CPU tensors over gloo in tests/test_multirank.py."""
from __future__ import annotations

import pytest

from paper_1805_06383_b200 import workloads
from test_gpu_parity import check_parity, fstc  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("config,scale,kw", [("tiny", 1.0, {}), ("tiny", 1.0, {"merge_mode": 1}), ("tiny", 1.0, {"merge_mode": 2}),
                                             ("tiny", 1.0, {"max_levels": 6}), ("medium", 0.03, {}), ("skewed", 0.02, {"max_levels": 3}),
                                             ("nlp", 0.1, {})])
def test_single_rank_shard_is_the_whole_composition(fstc, config, scale, kw):
    from paper_1805_06383_b200.sharded import KeyExchange, fstc_compose_sharded
    m1, m2 = workloads.make_config(config, scale=scale)
    p1 = fstc.fstc_pack(fstc.DeviceFst.from_host(m1), 1)
    p2 = fstc.fstc_pack(fstc.DeviceFst.from_host(m2), 2)
    ex = KeyExchange(0, 1, "cuda")
    res = fstc_compose_sharded(p1, p2, ex, n_q2=m2.n_states, start=(m1.start, m2.start), **kw)
    assert res.stats["n_resolve"] >= res.n_levels - 1 and ex.n_local == res.n_states
    check_parity(fstc, m1, m2, merge_mode=kw.get("merge_mode", 0), max_levels=kw.get("max_levels", 0), result=res)


def test_external_resolve_argument_errors(fstc):
    m1, m2 = workloads.make_config("tiny")
    a, b = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    with pytest.raises(fstc.FstcError) as e:                      # no callback
        fstc.fstc_compose(a, b, resolve_mode=fstc.RESOLVE_EXTERNAL, small_path=1)
    assert e.value.code == fstc.ERR_ARG
