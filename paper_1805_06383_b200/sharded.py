"""One composition sharded over several GPUs by OWNERSHIP of the state pairs ("owner computes").

Every rank holds both packed operands and expands only the pairs it owns; the target keys of its composed arcs are
routed to their owners with one all-to-all per exchange, the owners find or create the states and send a GLOBAL state
id back for every key.  Arcs stay with the owner of their source, and merging needs no communication because identical
arcs share a source.  The expansion itself is the C library's level-synchronous path with
`FSTC_RESOLVE_EXTERNAL`: it hands every batch of target keys to `KeyExchange.resolve` through `fstc_opts_t.resolve_cb`.

`KeyExchange` holds no method arithmetic beyond the key -> owner hash and the id bookkeeping; it works on CPU tensors
(gloo) as well as CUDA tensors (nccl), which is how the exchange logic is tested without hardware
(tests/test_multirank.py).  Global id of local state i of rank r: i * world + r.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Tuple

import torch
import torch.distributed as dist


def owner_of(keys: torch.Tensor, world: int) -> torch.Tensor:
    """Owner rank of every pair key: a multiplicative hash of the key, so that neighbouring keys spread over the ranks."""
    if world == 1:
        return torch.zeros_like(keys)
    h = keys * -7046029254386353131            # 0x9E3779B97F4A7C15 as int64; the product wraps modulo 2^64
    h = (h >> 33) & 0x7FFFFFFF
    return h % world


class KeyExchange:
    """The visited set of the states this rank owns, and the exchange that resolves target keys to global ids."""

    def __init__(self, rank: int, world: int, device, group=None):
        self.rank, self.world, self.device, self.group = rank, world, torch.device(device), group
        self.keys = torch.empty(0, dtype=torch.int64, device=self.device)    # owned keys, ascending
        self.lids = torch.empty(0, dtype=torch.int64, device=self.device)    # their local ids
        self.n_local = 0
        self.exchanged_keys = 0

    # ---- collectives (gloo has no all-to-all: point-to-point there)
    def _all_to_all(self, send: list) -> list:
        if self.world == 1:
            return [send[0]]
        counts = torch.tensor([t.numel() for t in send], dtype=torch.int64, device=self.device)
        rcounts = torch.empty_like(counts)
        if dist.get_backend(self.group) == "nccl":
            dist.all_to_all_single(rcounts, counts, group=self.group)
            recv = [torch.empty(int(n), dtype=send[0].dtype, device=self.device) for n in rcounts.tolist()]
            dist.all_to_all(recv, [t.contiguous() for t in send], group=self.group)
            return recv
        all_counts = [torch.empty_like(counts) for _ in range(self.world)]
        dist.all_gather(all_counts, counts, group=self.group)
        recv = [torch.empty(int(all_counts[p][self.rank]), dtype=send[0].dtype, device=self.device) for p in range(self.world)]
        recv[self.rank] = send[self.rank]
        reqs = []
        for p in range(self.world):
            if p == self.rank:
                continue
            reqs.append(dist.isend(send[p].contiguous(), p, group=self.group))
            reqs.append(dist.irecv(recv[p], p, group=self.group))
        for r in reqs:
            r.wait()
        return recv

    def any_rank(self, flag: bool) -> bool:
        if self.world == 1:
            return bool(flag)
        t = torch.tensor([int(flag)], dtype=torch.int64, device=self.device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group)
        return bool(int(t.item()))

    # ---- ownership
    def owns(self, key: int) -> bool:
        return int(owner_of(torch.tensor([key], dtype=torch.int64), self.world)[0]) == self.rank

    def insert_start(self, key: int) -> None:
        """The start pair is local state 0 of its owner."""
        assert self.n_local == 0 and self.owns(key)
        self.keys = torch.tensor([key], dtype=torch.int64, device=self.device)
        self.lids = torch.zeros(1, dtype=torch.int64, device=self.device)
        self.n_local = 1

    def resolve(self, keys: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor]:
        """keys: int64 target keys of this rank's arcs.  -> (global id of every key, the keys this rank now owns in
        addition, in local-id order).  A collective: every rank calls it the same number of times."""
        w = self.world
        own = owner_of(keys, w)
        order = torch.argsort(own, stable=True)
        counts = torch.bincount(own, minlength=w).tolist()
        recv = self._all_to_all(list(torch.split(keys[order], counts)))
        self.exchanged_keys += int(keys.numel()) - counts[self.rank]
        got = torch.cat(recv) if len(recv) > 1 else recv[0]
        # owner side: one entry per distinct key, found in the visited set or created
        uniq, inv = torch.unique(got, return_inverse=True)
        pos = torch.searchsorted(self.keys, uniq)
        found = torch.zeros(uniq.numel(), dtype=torch.bool, device=self.device)
        if self.keys.numel():
            inb = pos < self.keys.numel()
            found[inb] = self.keys[pos[inb]] == uniq[inb]
        lid = torch.empty(uniq.numel(), dtype=torch.int64, device=self.device)
        lid[found] = self.lids[pos[found]]
        new_keys = uniq[~found]
        n_new = int(new_keys.numel())
        lid[~found] = self.n_local + torch.arange(n_new, dtype=torch.int64, device=self.device)
        if n_new:
            allk = torch.cat([self.keys, new_keys])
            alll = torch.cat([self.lids, lid[~found]])
            o = torch.argsort(allk)
            self.keys, self.lids = allk[o], alll[o]
            self.n_local += n_new
        reply = (lid * w + self.rank)[inv]
        back = self._all_to_all(list(torch.split(reply, [int(t.numel()) for t in recv])))
        out = torch.empty_like(keys)
        out[order] = torch.cat(back) if len(back) > 1 else back[0]
        return out, new_keys


class _DevArray:
    """A device pointer as a CUDA array for torch.as_tensor."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (int(ptr), False), "version": 2}


_RESOLVE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_void_p,
                               ctypes.c_int64, ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(ctypes.c_int64),
                               ctypes.POINTER(ctypes.c_int32))


def fstc_compose_sharded(p1, p2, exchange: KeyExchange, *, n_q2: int, start: Tuple[int, int], stream=None, **opts):
    """This rank's shard of M1∘M2: `p1`, `p2` the operands packed on this rank's GPU, `exchange` a KeyExchange over the
    process group.  The result holds the states this rank owns (local ids) and their arcs (src local, tgt global)."""
    from . import fstc
    q2_bits = max(1, int(n_q2 - 1).bit_length())
    start_key = (int(start[0]) << q2_bits) | int(start[1])
    owns_start = exchange.owns(start_key)
    if owns_start:
        exchange.insert_start(start_key)
    state = {"new": None, "created": False, "error": None}

    def cb(_ctx, level, call, qb, keys_ptr, n_keys, ids_ptr, new_pairs, n_new, more):
        try:
            assert qb == q2_bits
            n = int(n_keys)
            keys = (torch.as_tensor(_DevArray(keys_ptr, n, "<i8"), device=exchange.device) if n
                    else torch.empty(0, dtype=torch.int64, device=exchange.device))
            gids, new_keys = exchange.resolve(keys)
            if n:
                torch.as_tensor(_DevArray(ids_ptr, n, "<i4"), device=exchange.device).copy_(gids.to(torch.int32))
            pairs = torch.stack([new_keys >> q2_bits, new_keys & ((1 << q2_bits) - 1)], 1).to(torch.int32).contiguous()
            state["new"] = pairs                                    # alive until the next call
            state["created"] = state["created"] or pairs.shape[0] > 0
            new_pairs[0] = pairs.data_ptr() if pairs.shape[0] else None
            n_new[0] = pairs.shape[0]
            if call == 2:
                more[0] = int(exchange.any_rank(state["created"]))
                state["created"] = False
            torch.cuda.synchronize(exchange.device)
            return 0
        except Exception as e:                                       # noqa: BLE001 — reported through the return code
            state["error"] = e
            return 1

    fn = _RESOLVE_FN(cb)
    o = fstc._opts(resolve_mode=fstc.RESOLVE_EXTERNAL, small_path=fstc.SMALL_OFF, **opts)
    o.resolve_cb = ctypes.cast(fn, ctypes.c_void_p)
    o.owns_start = int(owns_start)
    st = fstc._Stats()
    out = ctypes.POINTER(fstc._Result)()
    rc = fstc.lib().fstc_compose_packed(p1.ptr, p2.ptr, ctypes.addressof(o), fstc._stream_ptr(stream), ctypes.byref(out),
                                        ctypes.addressof(st))
    if rc != 0 and state["error"] is not None:
        raise state["error"]
    fstc._check(rc)
    return fstc.ComposeResult(out, st)
