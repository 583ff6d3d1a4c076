"""Thin Python binding of the C ABI in include/arc.h (same names, argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs in the CUDA kernels of
libarc_b200.so.  There is no CPU fallback: if the library is not built (or cannot be loaded) every entry
point raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

from . import build as _build

POLICY_ARC, POLICY_LRU, POLICY_DBL = 0, 1, 2
PIN_REQUEST, PIN_STEP, PIN_HELD = 0, 1, 2
MISS, HIT_T1, HIT_T2, GHOST_B1, GHOST_B2 = 0, 1, 2, 3, 4
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_REQUEST_TOO_LARGE, ERR_OOM, ERR_CUDA = 0, -1, -2, -3, -4, -5

STAT_FIELDS = ["steps", "requests", "tokens_seen", "tokens_hashed", "accesses", "hit_t1", "hit_t2", "ghost_b1",
               "ghost_b2", "miss", "evict_t1", "evict_t2", "drop_b1", "drop_b2", "fresh_ids_used",
               "prefix_hit_tokens", "t1", "t2", "b1", "b2", "p", "capacity_blocks"]

# every symbol include/arc.h declares (checked by the CPU test-suite against the built library)
EXPORTS = ["arc_create", "arc_reserve", "arc_step", "arc_step_host", "arc_stats", "arc_reset", "arc_destroy",
           "arc_last_error", "arc_hash_blocks", "arc_set_profiling", "arc_last_kernel_times", "arc_launch_count",
           "arc_set_machine", "arc_debug_list", "arc_debug_counters", "arc_debug_set_key_mask", "arc_debug_probe", "arc_set_pin_scope",
           "arc_release", "arc_hold_units", "arc_step_resume", "arc_debug_gather_sectors", "arc_hash_blocks_device", "arc_step_host_async",
           "arc_step_host_wait", "arc_route_requests", "arc_debug_latency_hist", "arc_hash_blocks_static"]


class ArcError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"arc error {code}: {text}")
        self.code = code


class _StepResult(C.Structure):
    _fields_ = [("n_access", C.c_uint64), ("prefix_len", C.c_void_p), ("blk_off", C.c_void_p), ("cls", C.c_void_p),
                ("block_id", C.c_void_p), ("evicted_id", C.c_void_p), ("p_after", C.c_void_p), ("alloc_ids", C.c_void_p),
                ("evict_ids", C.c_void_p), ("counts", C.c_void_p), ("chain_state", C.c_void_p)]


class _HostResult(C.Structure):
    _fields_ = [("n_access", C.c_uint64), ("n_alloc", C.c_uint32), ("n_evict", C.c_uint32),
                ("prefix_len", C.POINTER(C.c_int32)), ("alloc_ids", C.POINTER(C.c_int32)), ("evict_ids", C.POINTER(C.c_int32)),
                ("h2d_bytes", C.c_uint64), ("d2h_bytes", C.c_uint64)]


class _Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in STAT_FIELDS] + [("block_size", C.c_uint32), ("policy", C.c_int32)]


class _KernelTimes(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("hash_ms", "probe_ms", "machine_ms", "finalize_ms", "maint_ms", "total_ms")]


_lib = None


def load_library(path: Optional[Path] = None):
    """dlopen libarc_b200.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = Path(path) if path else _build.build()
    if not p.exists():
        raise RuntimeError(f"{p} is missing: the CUDA extension is not built (python -m paper_2606_21238_b200.build); "
                           "there is no CPU fallback")
    L = C.CDLL(str(p))
    vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
    L.arc_create.argtypes = [u64, u32, C.c_int, C.POINTER(vp)]
    L.arc_reserve.argtypes = [vp, u32, u64]
    L.arc_step.argtypes = [vp, vp, vp, u32, vp, C.POINTER(_StepResult)]
    L.arc_step_resume.argtypes = [vp, vp, vp, vp, u32, vp, C.POINTER(_StepResult)]
    L.arc_step_host.argtypes = [vp, vp, vp, u32, vp, C.POINTER(_HostResult)]
    L.arc_step_host_async.argtypes = [vp, vp, vp, u32, vp, C.POINTER(u32)]
    L.arc_step_host_wait.argtypes = [vp, u32, C.POINTER(_HostResult)]
    L.arc_stats.argtypes = [vp, C.POINTER(_Stats)]
    L.arc_reset.argtypes = [vp]
    L.arc_destroy.argtypes = [vp]
    L.arc_destroy.restype = None
    L.arc_last_error.argtypes = [vp]
    L.arc_last_error.restype = C.c_char_p
    L.arc_hash_blocks.argtypes = [vp, vp, u32, u32, vp, vp]
    L.arc_hash_blocks_static.argtypes = [vp, vp, u32, u32, vp, vp]
    L.arc_hash_blocks_device.argtypes = [vp, vp, u32, C.c_int64, C.c_int64, u32, vp, vp, vp]
    L.arc_route_requests.argtypes = [vp, vp, u32, u32, u32, vp, vp]
    L.arc_set_profiling.argtypes = [vp, C.c_int]
    L.arc_last_kernel_times.argtypes = [vp, C.POINTER(_KernelTimes)]
    L.arc_launch_count.argtypes = [vp]
    L.arc_launch_count.restype = u64
    L.arc_set_machine.argtypes = [vp, C.c_int]
    L.arc_debug_counters.argtypes = [vp, vp, u32]
    L.arc_debug_set_key_mask.argtypes = [vp, u64]
    L.arc_debug_probe.argtypes = [vp, vp, u64, vp, vp]
    L.arc_set_pin_scope.argtypes = [vp, C.c_int]
    L.arc_release.argtypes = [vp, vp, u64, vp]
    L.arc_hold_units.argtypes = [vp]
    L.arc_hold_units.restype = u64
    L.arc_debug_list.argtypes = [vp, C.c_int, vp, vp, u64, C.POINTER(u64)]
    L.arc_debug_latency_hist.argtypes = [vp, vp]
    L.arc_debug_gather_sectors.argtypes = [vp, u64, vp, u64, vp, vp]
    if path is None:
        _lib = L
    return L


def _torch():
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_21238_b200.arc needs a CUDA device (no CPU fallback)")
    return torch


class _DevView:
    """Zero-copy view of library-owned device memory for torch.as_tensor."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr or 0, False), "version": 3, "strides": None}


_views = {}     # (device pointer, typestr) -> the longest view made of it so far


def _view(ptr, n, typestr, dtype):
    """A tensor over n elements of library-owned device memory.  Wrapping a raw pointer costs tens of microseconds on the
    host, and a handle hands out the same buffers step after step, so the wrapper is kept per pointer and sliced: the
    view owns nothing, and only the n elements the library has just declared valid are ever reachable through it."""
    torch = _torch()
    if n == 0 or not ptr:
        return torch.zeros(0, dtype=dtype, device="cuda")
    v = _views.get((ptr, typestr))
    if v is None or v.numel() < n:
        if len(_views) >= 512:
            _views.clear()
        v = _views[(ptr, typestr)] = torch.as_tensor(_DevView(ptr, n, typestr), device="cuda")
    return v if v.numel() == n else v[:n]


def _offsets(offsets) -> np.ndarray:
    o = np.ascontiguousarray(offsets, dtype=np.int64)
    if o.ndim != 1 or o.size < 1:
        raise ValueError("offsets must have n_req + 1 entries")
    return o


def _stream_ptr(stream) -> int:
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


class StepResult:
    """Device-resident outputs of one arc_step (torch tensors viewing library-owned memory; valid until the
    next step on the same cache).  The views are made when they are first asked for: a caller that reads only
    `block_id` pays for one view, not for nine."""

    _FIELDS = {"prefix_len": ("prefix_len", "req", "<i4", "int32"), "blk_off": ("blk_off", "req1", "<i8", "int64"),
               "cls": ("cls", "n", "|u1", "uint8"), "block_id": ("block_id", "n", "<i4", "int32"),
               "evicted_id": ("evicted_id", "n", "<i4", "int32"), "p_after": ("p_after", "n", "<i4", "int32"),
               "counts": ("counts", "two", "<i4", "int32"), "chain_state": ("chain_state", "req", "<i8", "int64")}   # chain_state: uint64 bit patterns

    def __init__(self, raw: _StepResult, n_req: int):
        self.n_access = int(raw.n_access)
        self._raw, self._n_req = raw, n_req
        self._alloc_ptr, self._evict_ptr = raw.alloc_ids, raw.evict_ids

    def __getattr__(self, name):
        f = StepResult._FIELDS.get(name)
        if f is None:
            raise AttributeError(name)
        torch = _torch()
        n = {"req": self._n_req, "req1": self._n_req + 1, "n": self.n_access, "two": 2}[f[1]]
        v = _view(getattr(self._raw, f[0]), n, f[2], getattr(torch, f[3]))
        setattr(self, name, v)
        return v

    def to_host(self) -> dict:
        """Synchronising copy of everything to numpy (for tests)."""
        torch = _torch()
        counts = self.counts.cpu().numpy()
        n_alloc, n_evict = int(counts[0]), int(counts[1])
        return dict(n_access=self.n_access, prefix_len=self.prefix_len.cpu().numpy(), blk_off=self.blk_off.cpu().numpy(),
                    cls=self.cls.cpu().numpy(), block_id=self.block_id.cpu().numpy(), evicted_id=self.evicted_id.cpu().numpy(),
                    p_after=self.p_after.cpu().numpy(), chain_state=self.chain_state.cpu().numpy().view(np.uint64),
                    alloc_ids=_view(self._alloc_ptr, n_alloc, "<i4", torch.int32).cpu().numpy(),
                    evict_ids=_view(self._evict_ptr, n_evict, "<i4", torch.int32).cpu().numpy())


class ArcCache:
    """arc_create / arc_step / arc_stats / arc_destroy."""

    def __init__(self, capacity_blocks: int, block_size: int = 16, policy: int = POLICY_ARC):
        _torch().cuda.init()
        self._L = load_library()
        self._h = C.c_void_p()
        rc = self._L.arc_create(capacity_blocks, block_size, policy, C.byref(self._h))
        if rc != OK:
            raise ArcError(rc, self._L.arc_last_error(None).decode())
        self.capacity_blocks, self.block_size, self.policy = capacity_blocks, block_size, policy

    def _check(self, rc):
        if rc != OK:
            raise ArcError(rc, self._L.arc_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.arc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reserve(self, max_req: int, max_blocks_per_step: int):
        self._check(self._L.arc_reserve(self._h, max_req, max_blocks_per_step))

    def step(self, tokens, offsets, stream=None, chain_in=None) -> StepResult:
        """tokens: CUDA int32 tensor (any 4-byte alignment); offsets: host int64[n_req+1].  chain_in (arc_step_resume):
        per request the chain state it continues from - a CUDA int64 tensor of uint64 bit patterns (e.g. gathered from
        an earlier result's chain_state) or a numpy uint64 array; None = new prompts."""
        torch = _torch()
        if not (isinstance(tokens, torch.Tensor) and tokens.is_cuda and tokens.dtype == torch.int32 and tokens.is_contiguous()):
            raise TypeError("tokens must be a contiguous CUDA int32 tensor")
        o = _offsets(offsets)
        if o[-1] > tokens.numel():
            raise ValueError("offsets exceed the token tensor")
        raw = _StepResult()
        if chain_in is None:
            self._check(self._L.arc_step(self._h, tokens.data_ptr(), o.ctypes.data, len(o) - 1, _stream_ptr(stream), C.byref(raw)))
            return StepResult(raw, len(o) - 1)
        if not (hasattr(chain_in, "is_cuda") and chain_in.is_cuda):
            chain_in = torch.from_numpy(np.ascontiguousarray(chain_in, dtype=np.uint64).view(np.int64)).cuda()
        chain_in = chain_in.to(torch.int64).contiguous().clone()     # never the handle's own chain_state buffer
        if chain_in.numel() != len(o) - 1:
            raise ValueError("chain_in needs one state per request")
        self._keep_chain = chain_in
        self._check(self._L.arc_step_resume(self._h, tokens.data_ptr(), o.ctypes.data, chain_in.data_ptr(), len(o) - 1,
                                            _stream_ptr(stream), C.byref(raw)))
        return StepResult(raw, len(o) - 1)

    def step_raw(self, tokens_ptr: int, offsets: np.ndarray, stream_ptr: int) -> int:
        """Marshalling-free variant for benchmarks: returns the error code only (results stay on the device)."""
        raw = _StepResult()
        return self._L.arc_step(self._h, tokens_ptr, offsets.ctypes.data, len(offsets) - 1, stream_ptr, C.byref(raw))

    def step_host(self, tokens: np.ndarray, offsets, stream=None) -> dict:
        """End to end from host memory (H2D of the tokens and D2H of the results inside the call)."""
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        o = _offsets(offsets)
        if o[-1] > t.size:
            raise ValueError("offsets exceed the token array")
        raw = _HostResult()
        self._check(self._L.arc_step_host(self._h, t.ctypes.data, o.ctypes.data, len(o) - 1, _stream_ptr(stream), C.byref(raw)))
        n_req = len(o) - 1
        take = lambda p, n: np.ctypeslib.as_array(p, shape=(n,)).copy() if n else np.zeros(0, np.int32)
        return dict(n_access=int(raw.n_access), prefix_len=take(raw.prefix_len, n_req), alloc_ids=take(raw.alloc_ids, raw.n_alloc),
                    evict_ids=take(raw.evict_ids, raw.n_evict), h2d_bytes=int(raw.h2d_bytes), d2h_bytes=int(raw.d2h_bytes))

    def step_host_async(self, tokens: np.ndarray, offsets, stream=None) -> int:
        """arc_step_host_async: enqueue the step from host memory (pinned memory keeps the copy asynchronous); returns the
        ticket for step_host_wait.  Up to three steps may be in flight."""
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        o = _offsets(offsets)
        if o[-1] > t.size:
            raise ValueError("offsets exceed the token array")
        ticket = C.c_uint32()
        self._check(self._L.arc_step_host_async(self._h, t.ctypes.data, o.ctypes.data, len(o) - 1, _stream_ptr(stream), C.byref(ticket)))
        if not hasattr(self, "_inflight"):
            self._inflight = {}
        self._inflight[ticket.value] = (t, len(o) - 1)          # the tokens stay alive until the step has been waited for
        return ticket.value

    def step_host_wait(self, ticket: int, copy: bool = True) -> dict:
        """arc_step_host_wait: blocks until the step is done; copy=False returns only the counts and byte counts."""
        raw = _HostResult()
        self._check(self._L.arc_step_host_wait(self._h, ticket, C.byref(raw)))
        _, n_req = self._inflight.pop(ticket)
        out = dict(n_access=int(raw.n_access), n_alloc=int(raw.n_alloc), n_evict=int(raw.n_evict), h2d_bytes=int(raw.h2d_bytes), d2h_bytes=int(raw.d2h_bytes))
        if copy:
            take = lambda p, n: np.ctypeslib.as_array(p, shape=(n,)).copy() if n else np.zeros(0, np.int32)
            out.update(prefix_len=take(raw.prefix_len, n_req), alloc_ids=take(raw.alloc_ids, raw.n_alloc), evict_ids=take(raw.evict_ids, raw.n_evict))
        return out

    def stats(self) -> dict:
        s = _Stats()
        self._check(self._L.arc_stats(self._h, C.byref(s)))
        return {n: int(getattr(s, n)) for n in STAT_FIELDS + ["block_size", "policy"]}

    def reset(self):
        self._check(self._L.arc_reset(self._h))

    def set_profiling(self, enabled: bool):
        self._check(self._L.arc_set_profiling(self._h, int(enabled)))

    def last_kernel_times(self) -> dict:
        t = _KernelTimes()
        self._check(self._L.arc_last_kernel_times(self._h, C.byref(t)))
        return {n: float(getattr(t, n)) for n, _ in _KernelTimes._fields_}

    def launch_count(self) -> int:
        return int(self._L.arc_launch_count(self._h))

    def set_pin_scope(self, scope: int):
        self._check(self._L.arc_set_pin_scope(self._h, scope))

    def release(self, block_ids, stream=None):
        """PIN_HELD: one hold back per listed block ID (a CUDA int32 tensor, or anything numpy can read: copied to the
        device first).  Asynchronous on the current stream."""
        torch = _torch()
        if not (hasattr(block_ids, "is_cuda") and block_ids.is_cuda):
            block_ids = torch.from_numpy(np.ascontiguousarray(block_ids, dtype=np.int32)).cuda()
        if block_ids.dtype != torch.int32 or not block_ids.is_contiguous():
            block_ids = block_ids.to(torch.int32).contiguous()
        self._keep_release = block_ids          # stays alive until the kernel has read it (next call replaces it)
        self._check(self._L.arc_release(self._h, block_ids.data_ptr(), block_ids.numel(), _stream_ptr(stream)))

    def hold_units(self) -> int:
        return int(self._L.arc_hold_units(self._h))

    def set_machine(self, which: int):
        self._check(self._L.arc_set_machine(self._h, which))

    DEBUG_COUNTERS = ["win_hit", "win_general", "win_serial", "cut_twin", "cut_conflict", "scan_rounds", "acc_hit_win",
                      "acc_general_win", "cyc_fetch", "cyc_roll", "cyc_scan", "cyc_apply", "cyc_serial", "cyc_total", "roll_calls", "roll_phases",
                      "prov_ok", "prov_miss"]

    def debug_counters(self) -> dict:
        out = np.zeros(len(self.DEBUG_COUNTERS), np.uint64)
        self._check(self._L.arc_debug_counters(self._h, out.ctypes.data, len(out)))
        return {k: int(v) for k, v in zip(self.DEBUG_COUNTERS, out)}

    def debug_latency_hist(self) -> np.ndarray:
        """[5 classes, 16 bins] per-access latency histogram of the by-the-book machine (set_machine(1)); see arc.h."""
        out = np.zeros((5, 16), np.uint32)
        self._check(self._L.arc_debug_latency_hist(self._h, out.ctypes.data))
        return out

    def debug_probe(self, keys, nodes_out=None, stream=None):
        """K2 alone: keys = CUDA int64 tensor holding uint64 bits (>= 2); returns the CUDA int32 tensor of node indices."""
        torch = _torch()
        if nodes_out is None:
            nodes_out = torch.empty(keys.numel(), dtype=torch.int32, device="cuda")
        self._check(self._L.arc_debug_probe(self._h, keys.data_ptr(), keys.numel(), nodes_out.data_ptr(), _stream_ptr(stream)))
        return nodes_out

    def debug_set_key_mask(self, mask: int):
        self._check(self._L.arc_debug_set_key_mask(self._h, mask & 0xFFFFFFFFFFFFFFFF))

    def debug_lists(self) -> dict:
        out = {}
        for name, which in (("T1", 1), ("T2", 2), ("B1", 3), ("B2", 4)):
            cap = 2 * self.capacity_blocks + 8
            keys, blocks, n = np.zeros(cap, np.uint64), np.zeros(cap, np.int32), C.c_uint64()
            self._check(self._L.arc_debug_list(self._h, which, keys.ctypes.data, blocks.ctypes.data, cap, C.byref(n)))
            out[name] = (keys[:n.value].copy(), blocks[:n.value].copy())
        return out


def hash_blocks_static(tokens, offsets, out, block_size: int = 16, stream=None):
    """arc_hash_blocks_static: the same keys as hash_blocks into the caller's `out` (CUDA int64[N]); neither this wrapper
    nor the library allocates (at most 253 requests and 4,096 128-block segments per call, see arc.h)."""
    L = load_library()
    o = _offsets(offsets)
    rc = L.arc_hash_blocks_static(tokens.data_ptr(), o.ctypes.data, len(o) - 1, block_size, out.data_ptr(), _stream_ptr(stream))
    if rc != OK:
        raise ArcError(rc, L.arc_last_error(None).decode())
    return out


def hash_blocks(tokens, offsets, block_size: int = 16, out=None, stream=None):
    """arc_hash_blocks: keys of every full block in natural order, as a CUDA int64 tensor holding the uint64 bits."""
    torch = _torch()
    L = load_library()
    o = _offsets(offsets)
    if out is None:
        out = torch.empty(int((np.diff(o) // block_size).sum()), dtype=torch.int64, device="cuda")
    rc = L.arc_hash_blocks(tokens.data_ptr(), o.ctypes.data, len(o) - 1, block_size, out.data_ptr(), _stream_ptr(stream))
    if rc != OK:
        raise ArcError(rc, L.arc_last_error(None).decode())
    return out


HASH_ITEM = np.dtype([("tok_off", "<i8"), ("key_off", "<i8"), ("n_blocks", "<u4"), ("reserved", "<u4", (3,))])   # arc_hash_item


def hash_items(offsets, block_size: int = 16) -> np.ndarray:
    """The work list arc_hash_blocks builds from host offsets: one HASH_ITEM per request with a full block, requests of
    >= 1024 / 384 / 128 / fewer blocks in that order (input marshalling for arc_hash_blocks_device)."""
    o = _offsets(offsets)
    nb = np.diff(o) // block_size
    key_off = np.concatenate([[0], np.cumsum(nb)])[:-1]
    cls = np.where(nb >= 1024, 0, np.where(nb >= 384, 1, np.where(nb >= 128, 2, 3)))
    idx = np.flatnonzero(nb > 0)
    idx = idx[np.argsort(cls[idx], kind="stable")]
    items = np.zeros(len(idx), HASH_ITEM)
    items["tok_off"], items["key_off"], items["n_blocks"] = o[:-1][idx], key_off[idx], nb[idx]
    return items


def hash_blocks_device(tokens, d_items, n_items: int, tok_lo: int, tok_hi: int, out, ticket, block_size: int = 16, stream=None):
    """arc_hash_blocks_device: d_items = CUDA uint8 tensor holding HASH_ITEM records, ticket a zeroed CUDA int32[2] scratch."""
    L = load_library()
    rc = L.arc_hash_blocks_device(tokens.data_ptr(), d_items.data_ptr(), n_items, tok_lo, tok_hi, block_size, out.data_ptr(),
                                  ticket.data_ptr(), _stream_ptr(stream))
    if rc != OK:
        raise ArcError(rc, L.arc_last_error(None).decode())
    return out


def route_requests(tokens, offsets, world: int, block_size: int = 16, stream=None):
    """arc_route_requests: destination shard of every request, computed on the device from its first block's key; returns a
    CUDA int32 tensor [n_req].  offsets: host int64[n_req+1] (copied to the device here) or a CUDA int64 tensor."""
    torch = _torch()
    L = load_library()
    if not (hasattr(offsets, "is_cuda") and offsets.is_cuda):
        offsets = torch.from_numpy(_offsets(offsets)).to(tokens.device, non_blocking=True)
    n_req = offsets.numel() - 1
    dst = torch.empty(n_req, dtype=torch.int32, device=tokens.device)
    rc = L.arc_route_requests(tokens.data_ptr(), offsets.data_ptr(), n_req, block_size, world, dst.data_ptr(), _stream_ptr(stream))
    if rc != OK:
        raise ArcError(rc, L.arc_last_error(None).decode())
    return dst


def debug_gather_sectors(keys, buf, out=None, stream=None):
    """arc_debug_gather_sectors: the random-32-byte-sector read ceiling K2 is compared with.  keys: CUDA int64 tensor; buf: CUDA
    tensor whose byte size is a power of two (>= 32); returns the CUDA int32 tensor of XORs."""
    torch = _torch()
    L = load_library()
    n_sectors = buf.numel() * buf.element_size() // 32
    if out is None:
        out = torch.empty(keys.numel(), dtype=torch.int32, device="cuda")
    rc = L.arc_debug_gather_sectors(keys.data_ptr(), keys.numel(), buf.data_ptr(), n_sectors, out.data_ptr(), _stream_ptr(stream))
    if rc != OK:
        raise ArcError(rc, L.arc_last_error(None).decode())
    return out


def hash_launch_count() -> int:
    return int(load_library().arc_launch_count(None))
