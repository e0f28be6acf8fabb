"""Thin Python binding of libfstc.so (include/fstc.h): argument marshalling only.

Every step of the composition runs in the library's CUDA kernels.  PyTorch is used for
device memory (inputs as CUDA tensors, outputs wrapped zero-copy as CUDA tensors) and for
the current stream.  There is NO CPU fallback: if libfstc.so is missing, importing any
compute entry point raises.
"""
from __future__ import annotations

import ctypes
import os
import struct
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FSTC_LIB") or os.path.join(_HERE, "libfstc.so")   # FSTC_LIB: an experiment build

FSTC_MEM_DEVICE, FSTC_MEM_HOST = 0, 1
MERGE_AUTO, MERGE_OFF, MERGE_SORT_ALL = 0, 1, 2
RESOLVE_AUTO, RESOLVE_TABLE, RESOLVE_PARTITIONED, RESOLVE_HASH, RESOLVE_EXTERNAL = 0, 1, 2, 3, 4
SMALL_AUTO, SMALL_OFF, SMALL_ONLY = 0, 1, 2
ERR_ARG, ERR_INPUT, ERR_OOM, ERR_CAPACITY, ERR_CUDA, ERR_INTERNAL, ERR_CALLBACK = -1, -2, -3, -4, -5, -6, -7
MAX_LEVEL_STATS = 64
STAGES = ("count", "scan", "match", "emit", "sort", "reduce", "table", "assemble", "rs_scatter", "rs_dedupe", "rs_gather")

EXPORTS = (
    "fstc_pack", "fstc_packed_free", "fstc_packed_info", "fstc_packed_to_host", "fstc_compose_packed",
    "fstc_compose", "fstc_compose_batch", "fstc_compose_static", "fstc_result_to_host", "fstc_result_free", "fstc_trim_pool", "fstc_strerror",
    "fstc_last_error", "fstc_version",
)


class FstcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"fstc error {code}: {msg}")
        self.code = code


class _Fst(ctypes.Structure):
    _fields_ = [
        ("n_states", ctypes.c_int32), ("n_isyms", ctypes.c_int32), ("n_osyms", ctypes.c_int32),
        ("start", ctypes.c_int32), ("n_arcs", ctypes.c_int64),
        ("src", ctypes.c_void_p), ("ilabel", ctypes.c_void_p), ("olabel", ctypes.c_void_p),
        ("tgt", ctypes.c_void_p), ("weight", ctypes.c_void_p),
        ("n_accept", ctypes.c_int32), ("accept", ctypes.c_void_p), ("mem", ctypes.c_int32),
    ]


class _Opts(ctypes.Structure):
    _fields_ = [
        ("merge_mode", ctypes.c_int32), ("max_levels", ctypes.c_int32), ("max_raw_arcs", ctypes.c_int64),
        ("arc_capacity_hint", ctypes.c_int64), ("state_capacity_hint", ctypes.c_int64),
        ("profile", ctypes.c_int32), ("resolve_mode", ctypes.c_int32),
        ("small_path", ctypes.c_int32), ("deterministic", ctypes.c_int32),
        ("alloc", ctypes.c_void_p), ("dealloc", ctypes.c_void_p), ("alloc_ctx", ctypes.c_void_p),
        ("spill", ctypes.c_void_p),
        ("resolve_cb", ctypes.c_void_p), ("resolve_ctx", ctypes.c_void_p), ("owns_start", ctypes.c_int32),
        ("reserved_", ctypes.c_int32),
    ]


class _Spill(ctypes.Structure):
    _fields_ = [("host", ctypes.c_void_p), ("arc_capacity", ctypes.c_int64), ("state_capacity", ctypes.c_int64),
                ("keep_device", ctypes.c_int32), ("reserved_", ctypes.c_int32)]


class _Stats(ctypes.Structure):
    _fields_ = [
        ("n_states", ctypes.c_int64), ("n_arcs", ctypes.c_int64), ("n_raw_arcs", ctypes.c_int64),
        ("n_expanded", ctypes.c_int64), ("n_levels", ctypes.c_int32), ("truncated", ctypes.c_int32),
        ("n_seg_visited", ctypes.c_int64), ("n_matches", ctypes.c_int64), ("n_match_arcs", ctypes.c_int64),
        ("n_raw_sorted", ctypes.c_int64), ("n_raw_grouped", ctypes.c_int64), ("n_raw_onchip", ctypes.c_int64),
        ("table_capacity", ctypes.c_int64),
        ("n_rehash", ctypes.c_int32), ("n_grow", ctypes.c_int32),
        ("n_emit_launches", ctypes.c_int32), ("n_kernel_launches", ctypes.c_int32),
        ("n_resolve", ctypes.c_int32), ("small_path", ctypes.c_int32), ("n_resolved_arcs", ctypes.c_int64),
        ("rs_scatter_recs", ctypes.c_int64), ("rs_scatter_dest_recs", ctypes.c_int64), ("rs_dedupe_arcs", ctypes.c_int64),
        ("rs_dedupe_states", ctypes.c_int64), ("rs_dedupe_new", ctypes.c_int64), ("rs_gather_recs", ctypes.c_int64),
        ("rs_scatter_launches", ctypes.c_int32), ("rs_dedupe_launches", ctypes.c_int32),
        ("rs_gather_launches", ctypes.c_int32), ("n_chunks", ctypes.c_int32),
        ("spill_bytes", ctypes.c_int64), ("spill_bytes_saved", ctypes.c_int64),
        ("ms", ctypes.c_double * len(STAGES)), ("ms_total", ctypes.c_double),
        ("level_frontier", ctypes.c_int64 * MAX_LEVEL_STATS), ("level_raw", ctypes.c_int64 * MAX_LEVEL_STATS),
        ("level_new_states", ctypes.c_int64 * MAX_LEVEL_STATS),
    ]


class _Result(ctypes.Structure):
    _fields_ = [
        ("n_states", ctypes.c_int64), ("n_arcs", ctypes.c_int64), ("n_raw_arcs", ctypes.c_int64),
        ("n_accept", ctypes.c_int64), ("n_expanded", ctypes.c_int64),
        ("n_levels", ctypes.c_int32), ("truncated", ctypes.c_int32),
        ("pair", ctypes.c_void_p), ("src", ctypes.c_void_p), ("ilabel", ctypes.c_void_p),
        ("olabel", ctypes.c_void_p), ("tgt", ctypes.c_void_p), ("weight", ctypes.c_void_p),
        ("accept", ctypes.c_void_p), ("expanded", ctypes.c_void_p), ("impl", ctypes.c_void_p),
    ]


class _HostResult(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in
                ("pair", "src", "ilabel", "olabel", "tgt", "weight", "accept", "expanded")]


_lib = None


def lib():
    """The loaded C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1805_06383_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        P, I = ctypes.c_void_p, ctypes.c_int
        L.fstc_pack.argtypes = [P, I, P, P, ctypes.POINTER(P)]
        L.fstc_packed_free.argtypes = [P]
        L.fstc_packed_free.restype = None
        L.fstc_packed_info.argtypes = [P, P]
        L.fstc_packed_to_host.argtypes = [P, P, P, P, P, P, P]
        L.fstc_compose_packed.argtypes = [P, P, P, P, ctypes.POINTER(ctypes.POINTER(_Result)), P]
        L.fstc_compose.argtypes = [P, P, P, P, ctypes.POINTER(ctypes.POINTER(_Result)), P]
        L.fstc_compose_batch.argtypes = [P, ctypes.c_int32, P, P, P, P, P]
        L.fstc_compose_static.argtypes = [P, P, P, P, P]
        L.fstc_result_to_host.argtypes = [P, P, P]
        L.fstc_result_free.argtypes = [P]
        L.fstc_result_free.restype = None
        L.fstc_trim_pool.argtypes = []
        L.fstc_strerror.argtypes = [I]
        L.fstc_strerror.restype = ctypes.c_char_p
        L.fstc_last_error.restype = ctypes.c_char_p
        L.fstc_version.restype = I
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        L = lib()
        msg = L.fstc_last_error().decode() or L.fstc_strerror(rc).decode()
        raise FstcError(rc, msg)


def _stream_ptr(stream=None) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


# ------------------------------------------------------------------------------------------------ inputs
@dataclass
class DeviceFst:
    """A transducer whose arrays are CUDA tensors (int32 / float32, contiguous)."""
    n_states: int
    n_isyms: int
    n_osyms: int
    start: int
    src: "object"
    ilabel: "object"
    olabel: "object"
    tgt: "object"
    weight: "object"
    accept: "object"

    @staticmethod
    def from_host(f, device="cuda") -> "DeviceFst":
        import torch
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)   # noqa: E731
        return DeviceFst(int(f.n_states), int(f.n_isyms), int(f.n_osyms), int(f.start), t(f.src), t(f.ilabel),
                         t(f.olabel), t(f.tgt), t(f.weight), t(f.accept))


def _marshal(f):
    """-> (_Fst, keepalive).  Accepts DeviceFst (CUDA tensors) or any object with numpy arrays (host)."""
    keep = []
    s = _Fst()
    s.n_states, s.n_isyms, s.n_osyms, s.start = int(f.n_states), int(f.n_isyms), int(f.n_osyms), int(f.start)
    is_dev = hasattr(f.src, "data_ptr")
    names = (("src", np.int32), ("ilabel", np.int32), ("olabel", np.int32), ("tgt", np.int32),
             ("weight", np.float32), ("accept", np.int32))
    if is_dev:
        import torch
        want = {np.int32: torch.int32, np.float32: torch.float32}
        for n, dt in names:
            t = getattr(f, n)
            if not t.is_cuda and not t.is_pinned():
                raise ValueError(f"{n}: expected a CUDA (or pinned host) tensor")
            if t.dtype != want[dt] or not t.is_contiguous():
                raise ValueError(f"{n}: expected contiguous {want[dt]}")
            keep.append(t)
            setattr(s, n, t.data_ptr())
        s.mem = FSTC_MEM_DEVICE if f.src.is_cuda else FSTC_MEM_HOST
        s.n_arcs, s.n_accept = int(f.src.numel()), int(f.accept.numel())
    else:
        for n, dt in names:
            a = np.ascontiguousarray(np.asarray(getattr(f, n)), dtype=dt)
            keep.append(a)
            setattr(s, n, a.ctypes.data)
        s.mem = FSTC_MEM_HOST
        s.n_arcs, s.n_accept = int(keep[0].shape[0]), int(keep[5].shape[0])
    return s, keep


# ------------------------------------------------------------------------------------------------ outputs
class _DevView:
    """Zero-copy __cuda_array_interface__ view of library-owned device memory."""

    def __init__(self, ptr: int, shape, typestr: str, owner):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 3, "strides": None}
        self._owner = owner


def _tensor(ptr, shape, typestr, owner):
    import torch
    n = int(np.prod(shape))
    dt = {"<i4": torch.int32, "<f4": torch.float32, "|u1": torch.uint8}[typestr]
    if n > 0 and not ptr:
        return None                 # the array is not on the device (host spill without a device copy)
    if n == 0:
        return torch.empty(tuple(shape), dtype=dt, device="cuda")
    return torch.as_tensor(_DevView(ptr, shape, typestr, owner), device="cuda")


class _ResultHandle:
    def __init__(self, ptr):
        self.ptr = ptr

    def __del__(self):
        if self.ptr:
            try:
                lib().fstc_result_free(self.ptr)
            except Exception:
                pass
            self.ptr = None


class ComposeResult:
    """M1∘M2 on the device.  State i is the pair (pair[i,0], pair[i,1]) = (q1,q2); state 0 = (s1,s2).
    Arcs are sorted by source id; tensors are views of library memory kept alive by this object.  The views and the stats
    dict are made on first use: a batch of thousands of results costs the C call, not thousands of wrappers."""

    _ORDER = ("pair", "src", "ilabel", "olabel", "tgt", "weight", "accept", "expanded")
    _FIELDS = {"pair": ("n_states", 2, "<i4"), "src": ("n_arcs", 0, "<i4"), "ilabel": ("n_arcs", 0, "<i4"),
               "olabel": ("n_arcs", 0, "<i4"), "tgt": ("n_arcs", 0, "<i4"), "weight": ("n_arcs", 0, "<f4"),
               "accept": ("n_accept", 0, "<i4"), "expanded": ("n_states", 0, "|u1")}

    _HEAD = struct.Struct("5q2i8P")                   # fstc_result_t up to `impl`, read in one go

    def __init__(self, rptr, stats):
        """rptr: a POINTER(_Result) or the address of a fstc_result_t.  stats: None, a _Stats, or (array of _Stats, index)."""
        addr = rptr if isinstance(rptr, int) else ctypes.cast(rptr, ctypes.c_void_p).value
        self._h = _ResultHandle(addr)
        v = self._HEAD.unpack(ctypes.string_at(addr, self._HEAD.size))
        (self.n_states, self.n_arcs, self.n_raw_arcs, self.n_accept, self.n_expanded, self.n_levels, self.truncated) = v[:7]
        self._ptrs = v[7:]
        self._views = {}
        self._stats = stats

    def __getattr__(self, name):                      # only reached for names that are not set yet: the lazy views
        if name in ComposeResult._FIELDS and "_views" in self.__dict__:
            v = self._views
            if name not in v:
                if self._h is None:
                    return None
                length, inner, typestr = self._FIELDS[name]
                n = getattr(self, length)
                v[name] = _tensor(self._ptrs[self._ORDER.index(name)], (n, inner) if inner else (n,), typestr, self._h)
            return v[name]
        if name == "stats" and "_stats" in self.__dict__:
            st = self._stats
            if isinstance(st, tuple):
                st = st[0][st[1]]
            if st is not None and not isinstance(st, dict):
                st = self._stats = stats_dict(st)
            return st
        raise AttributeError(name)

    def free(self):
        """Releases the result now (fstc_result_free); the tensors of this object must no longer be used."""
        self._views = {k: None for k in self._FIELDS}
        h, self._h = self._h, None
        if h is not None and h.ptr:
            lib().fstc_result_free(h.ptr)
            h.ptr = None

    def to_host(self, out: Optional[dict] = None, stream=None) -> dict:
        """Copies every array to host memory through fstc_result_to_host.  `out` may hold preallocated
        (pinned) torch CPU tensors named like the fields, each at least as long as needed."""
        import torch
        spec = {"pair": ((self.n_states, 2), torch.int32), "src": ((self.n_arcs,), torch.int32),
                "ilabel": ((self.n_arcs,), torch.int32), "olabel": ((self.n_arcs,), torch.int32),
                "tgt": ((self.n_arcs,), torch.int32), "weight": ((self.n_arcs,), torch.float32),
                "accept": ((self.n_accept,), torch.int32), "expanded": ((self.n_states,), torch.uint8)}
        hr = _HostResult()
        res = {}
        for name, (shape, dt) in spec.items():
            n = int(np.prod(shape))
            if out is not None and name in out:
                buf = out[name]
                assert buf.dtype == dt and buf.numel() >= n and buf.is_contiguous()
            else:
                buf = torch.empty(n, dtype=dt)
            setattr(hr, name, buf.data_ptr() if n else None)
            res[name] = buf.view(-1)[:n].view(*shape)
        _check(lib().fstc_result_to_host(self._h.ptr, _stream_ptr(stream), ctypes.addressof(hr)))
        return res


def stats_dict(s: _Stats) -> dict:
    nl = min(int(s.n_levels), MAX_LEVEL_STATS)
    return {
        "n_states": int(s.n_states), "n_arcs": int(s.n_arcs), "n_raw_arcs": int(s.n_raw_arcs),
        "n_expanded": int(s.n_expanded), "n_levels": int(s.n_levels), "truncated": int(s.truncated),
        "n_seg_visited": int(s.n_seg_visited), "n_matches": int(s.n_matches), "n_match_arcs": int(s.n_match_arcs),
        "n_raw_sorted": int(s.n_raw_sorted), "n_raw_grouped": int(s.n_raw_grouped), "n_raw_onchip": int(s.n_raw_onchip),
        "table_capacity": int(s.table_capacity),
        "n_rehash": int(s.n_rehash), "n_grow": int(s.n_grow), "n_emit_launches": int(s.n_emit_launches),
        "n_kernel_launches": int(s.n_kernel_launches),
        "n_resolve": int(s.n_resolve), "n_resolved_arcs": int(s.n_resolved_arcs), "small_path": int(s.small_path),
        "n_chunks": int(s.n_chunks), "spill_bytes": int(s.spill_bytes), "spill_bytes_saved": int(s.spill_bytes_saved),
        **{k: int(getattr(s, k)) for k in ("rs_scatter_recs", "rs_scatter_dest_recs", "rs_dedupe_arcs", "rs_dedupe_states",
                                           "rs_dedupe_new", "rs_gather_recs", "rs_scatter_launches", "rs_dedupe_launches",
                                           "rs_gather_launches")},
        "ms": {k: float(s.ms[i]) for i, k in enumerate(STAGES)}, "ms_total": float(s.ms_total),
        "level_frontier": [int(s.level_frontier[i]) for i in range(nl)],
        "level_raw": [int(s.level_raw[i]) for i in range(nl)],
        "level_new_states": [int(s.level_new_states[i]) for i in range(nl)],
    }


def _opts(merge_mode=MERGE_AUTO, max_raw_arcs=0, max_levels=0, arc_capacity_hint=0, state_capacity_hint=0,
          profile=False, resolve_mode=0, small_path=0, deterministic=False, allocator=None, spill=None,
          spill_keep_device=False) -> _Opts:
    """allocator: None (the library's pool) or "torch": every device allocation of the call goes through PyTorch's caching
    allocator (fstc_opts_t.alloc / dealloc)."""
    o = _Opts()
    o.deterministic = int(bool(deterministic))
    if spill is not None:
        # spill: dict of PINNED torch CPU tensors named like the result's fields (pair [S,2] int32, src/ilabel/olabel/tgt
        # int32 [A], weight float32 [A], accept int32 [S], expanded uint8 [S]); they receive the result while it is built
        hr = _HostResult()
        for name in ("pair", "src", "ilabel", "olabel", "tgt", "weight", "accept", "expanded"):
            t = spill.get(name)
            if t is not None:
                assert t.is_contiguous() and t.device.type == "cpu"
                setattr(hr, name, t.data_ptr())
        sp = _Spill()
        sp.host = ctypes.addressof(hr)
        sp.arc_capacity = min(int(spill[k].numel()) for k in ("src", "ilabel", "olabel", "tgt", "weight"))
        sp.state_capacity = int(spill["pair"].numel()) // 2
        for k in ("accept", "expanded"):
            if spill.get(k) is not None:
                sp.state_capacity = min(sp.state_capacity, int(spill[k].numel()))
        sp.keep_device = int(bool(spill_keep_device))
        o.spill = ctypes.addressof(sp)
        o._keep = (hr, sp, spill)
    if allocator == "torch":
        a, d = _torch_allocator()
        o.alloc, o.dealloc = ctypes.cast(a, ctypes.c_void_p), ctypes.cast(d, ctypes.c_void_p)
    elif allocator is not None:
        raise ValueError("allocator must be None or 'torch'")
    o.resolve_mode = int(resolve_mode)
    o.small_path = int(small_path)
    o.merge_mode, o.max_levels, o.max_raw_arcs = int(merge_mode), int(max_levels), int(max_raw_arcs)
    o.arc_capacity_hint, o.state_capacity_hint, o.profile = int(arc_capacity_hint), int(state_capacity_hint), int(bool(profile))
    return o


_ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p)
_DEALLOC_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p)
_torch_hooks = None
ALLOC_LOG = {"alloc": 0, "dealloc": 0, "bytes": 0}      # calls that went through the torch hooks (tests)


def _torch_allocator():
    """ctypes callbacks over torch.cuda.caching_allocator_alloc / _delete (kept alive for the life of the process)."""
    global _torch_hooks
    if _torch_hooks is None:
        import torch

        def alloc(nbytes, stream, _ctx):
            try:
                p = torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
            except Exception:
                return None
            ALLOC_LOG["alloc"] += 1
            ALLOC_LOG["bytes"] += int(nbytes)
            return p

        def dealloc(ptr, _stream, _ctx):
            ALLOC_LOG["dealloc"] += 1
            torch.cuda.caching_allocator_delete(int(ptr))

        _torch_hooks = (_ALLOC_FN(alloc), _DEALLOC_FN(dealloc))
    return _torch_hooks


class Packed:
    """fstc_packed_t handle (device-resident, reusable)."""

    def __init__(self, ptr):
        self.ptr = ptr

    def info(self) -> dict:
        a = (ctypes.c_int64 * 7)()
        _check(lib().fstc_packed_info(self.ptr, ctypes.addressof(a)))
        return dict(zip(("n_states", "n_arcs", "n_segments", "n_inner", "n_outer", "side", "n_kernel_launches"), (int(x) for x in a)))

    def to_host(self, stream=None) -> dict:
        i = self.info()
        arcs = np.empty((i["n_arcs"], 4), np.uint32)
        segs = np.empty((i["n_segments"] + 1, 2), np.uint32)
        seg_ptr = np.empty(i["n_states"] + 1, np.uint32)
        flags = np.empty(i["n_states"], np.uint8)
        acc = np.empty((i["n_states"] + 31) // 32, np.uint32)
        _check(lib().fstc_packed_to_host(self.ptr, _stream_ptr(stream), arcs.ctypes.data, segs.ctypes.data,
                                         seg_ptr.ctypes.data, flags.ctypes.data, acc.ctypes.data))
        return {"arcs": arcs, "segs": segs, "seg_ptr": seg_ptr, "flags": flags, "accept_bits": acc, **i}

    def free(self):
        if self.ptr:
            lib().fstc_packed_free(self.ptr)
            self.ptr = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def fstc_pack(m, side: int, stream=None, allocator=None) -> Packed:
    s, keep = _marshal(m)
    out = ctypes.c_void_p()
    o = _opts(allocator=allocator)
    _check(lib().fstc_pack(ctypes.addressof(s), int(side), ctypes.addressof(o), _stream_ptr(stream), ctypes.byref(out)))
    del keep
    return Packed(out)


def fstc_compose_packed(p1: Packed, p2: Packed, *, stream=None, with_stats=True, **opts) -> ComposeResult:
    o = _opts(**opts)
    st = _Stats() if with_stats else None
    out = ctypes.POINTER(_Result)()
    _check(lib().fstc_compose_packed(p1.ptr, p2.ptr, ctypes.addressof(o), _stream_ptr(stream), ctypes.byref(out),
                                     ctypes.addressof(st) if st is not None else None))
    return ComposeResult(out, st)


def fstc_compose_batch(p1s, p2: Packed, *, stream=None, with_stats=True, **opts) -> list:
    """M1[k]∘M2 for every packed left operand of `p1s` against one packed right operand, in one call (the paper's
    use case of many lattices against one language model)."""
    n = len(p1s)
    o = _opts(**opts)
    ptrs = (ctypes.c_void_p * n)(*[p.ptr for p in p1s])
    outs = (ctypes.POINTER(_Result) * n)()
    sts = (_Stats * n)() if with_stats else None
    _check(lib().fstc_compose_batch(ctypes.addressof(ptrs), n, p2.ptr, ctypes.addressof(o), _stream_ptr(stream),
                                    ctypes.addressof(outs), ctypes.addressof(sts) if sts is not None else None))
    addrs = struct.unpack(f"{n}P", ctypes.string_at(ctypes.addressof(outs), 8 * n)) if n else ()
    return [ComposeResult(a, (sts, k) if sts is not None else None) for k, a in enumerate(addrs)]


# ------------------------------------------------------------------------------------------------ no allocation
STATIC_MAX_STATES = 65536
STATIC_SCRATCH_BYTES = 8 << 20


class _StaticHeader(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int64) for n in ("n_states", "n_arcs", "n_raw_arcs", "n_accept", "n_expanded",
                                              "n_seg_visited", "n_match_arcs", "n_matches")] + \
               [(n, ctypes.c_int32) for n in ("n_levels", "truncated", "status", "reserved_")]


class _StaticOut(ctypes.Structure):
    _fields_ = [("state_capacity", ctypes.c_int64), ("arc_capacity", ctypes.c_int64)] + \
               [(n, ctypes.c_void_p) for n in ("pair", "src", "ilabel", "olabel", "tgt", "weight", "accept", "expanded", "header")]


class StaticBuffers:
    """The caller's side of fstc_compose_static: result arrays and the 80-byte header as CUDA tensors, made ONCE (by
    PyTorch) and reused by any number of calls; the call itself allocates nothing."""

    def __init__(self, state_capacity: int, arc_capacity: int, device="cuda"):
        import torch
        S, A = int(state_capacity), int(arc_capacity)
        self.state_capacity, self.arc_capacity = S, A
        n_s, n_a = max(S, 1), max(A, 1)
        self.pair = torch.empty((n_s, 2), dtype=torch.int32, device=device)
        self.src, self.ilabel, self.olabel, self.tgt = (torch.empty(n_a, dtype=torch.int32, device=device) for _ in range(4))
        self.weight = torch.empty(n_a, dtype=torch.float32, device=device)
        self.accept = torch.empty(n_s, dtype=torch.int32, device=device)
        self.expanded = torch.empty(n_s, dtype=torch.uint8, device=device)
        self.header = torch.zeros(10, dtype=torch.int64, device=device)
        o = _StaticOut()
        o.state_capacity, o.arc_capacity = S, A
        for n in ("pair", "src", "ilabel", "olabel", "tgt", "weight", "accept", "expanded", "header"):
            setattr(o, n, getattr(self, n).data_ptr())
        self._out = o

    def read(self) -> dict:
        """After the stream's work is done: the header as a dict, and (status 0) the arrays cut to their lengths."""
        h = _StaticHeader.from_buffer_copy(self.header.cpu().numpy().tobytes())
        d = {n: int(getattr(h, n)) for n, _ in _StaticHeader._fields_ if n != "reserved_"}
        if d["status"] == 0:
            ns, na = d["n_states"], d["n_arcs"]
            d.update(pair=self.pair[:ns], src=self.src[:na], ilabel=self.ilabel[:na], olabel=self.olabel[:na], tgt=self.tgt[:na],
                     weight=self.weight[:na], accept=self.accept[:d["n_accept"]], expanded=self.expanded[:ns])
        return d


def fstc_compose_static(p1: Packed, p2: Packed, out: StaticBuffers, *, merge_mode=MERGE_AUTO, max_levels=0, max_raw_arcs=0,
                        stream=None) -> None:
    """M1∘M2 of one small problem into the caller's buffers with NO device allocation (include/fstc.h): only enqueues
    on the stream; `out.read()` after a synchronisation gives the result (status 1: it did not fit)."""
    o = _opts(merge_mode=merge_mode, max_levels=max_levels, max_raw_arcs=max_raw_arcs)
    _check(lib().fstc_compose_static(p1.ptr, p2.ptr, ctypes.addressof(o), _stream_ptr(stream), ctypes.addressof(out._out)))


def fstc_compose(m1, m2, *, stream=None, with_stats=True, **opts) -> ComposeResult:
    """fst_compose(M1, M2) -> M1∘M2.  m1/m2: DeviceFst (CUDA tensors) or host arrays."""
    s1, k1 = _marshal(m1)
    s2, k2 = _marshal(m2)
    o = _opts(**opts)
    st = _Stats() if with_stats else None
    out = ctypes.POINTER(_Result)()
    _check(lib().fstc_compose(ctypes.addressof(s1), ctypes.addressof(s2), ctypes.addressof(o), _stream_ptr(stream),
                              ctypes.byref(out), ctypes.addressof(st) if st is not None else None))
    del k1, k2
    return ComposeResult(out, st)


def fstc_trim_pool():
    _check(lib().fstc_trim_pool())
