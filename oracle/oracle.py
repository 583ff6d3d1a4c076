"""ctypes wrapper of the C++ CPU oracle (`arc_oracle.cpp`).  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs
may import this.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "arc_oracle.cpp"
_LIB = _HERE / "liboracle.so"

MISS, HIT_T1, HIT_T2, GHOST_B1, GHOST_B2 = 0, 1, 2, 3, 4
POLICY_ARC, POLICY_LRU, POLICY_DBL = 0, 1, 2
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_REQUEST_TOO_LARGE = 0, -1, -2, -3

STAT_FIELDS = ["steps", "requests", "tokens_seen", "tokens_hashed", "accesses", "hit_t1", "hit_t2", "ghost_b1",
               "ghost_b2", "miss", "evict_t1", "evict_t2", "drop_b1", "drop_b2", "fresh_ids_used",
               "prefix_hit_tokens", "t1", "t2", "b1", "b2", "p", "capacity_blocks"]


class _Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in STAT_FIELDS] + [("block_size", C.c_uint32), ("policy", C.c_int32)]


class _Result(C.Structure):
    _fields_ = [("n_access", C.c_uint64), ("prefix_len", C.POINTER(C.c_int32)), ("blk_off", C.POINTER(C.c_int64)),
                ("cls", C.POINTER(C.c_uint8)), ("block_id", C.POINTER(C.c_int32)), ("evicted_id", C.POINTER(C.c_int32)),
                ("p_after", C.POINTER(C.c_int32)), ("alloc_ids", C.POINTER(C.c_int32)),
                ("evict_ids", C.POINTER(C.c_int32)), ("n_alloc", C.c_uint32), ("n_evict", C.c_uint32),
                ("chain_state", C.POINTER(C.c_uint64))]


def build(force: bool = False) -> Path:
    """g++ -O2, no SIMD intrinsics.  Building the checker is not using it.  With ARC_ORACLE_SANITIZE=1 in
    the environment the library is built and loaded with -fsanitize=address,undefined instead (a separate file; the
    process must then run with libasan preloaded: tests/test_oracle_sanitized.py)."""
    if os.environ.get("ARC_ORACLE_SANITIZE") == "1":
        lib = _HERE / "liboracle_san.so"
        if force or not lib.exists() or lib.stat().st_mtime < _SRC.stat().st_mtime:
            subprocess.check_call(["g++", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                                   "-std=c++17", "-shared", "-fPIC", "-o", str(lib), str(_SRC)])
        return lib
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", str(_LIB), str(_SRC)])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        L.oracle_create.argtypes = [C.c_uint64, C.c_uint32, C.c_int, C.POINTER(C.c_void_p)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_hash_blocks.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p]
        L.oracle_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.POINTER(_Result)]
        L.oracle_step_resume.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.POINTER(_Result)]
        L.oracle_step_keys.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.POINTER(_Result)]
        L.oracle_set_pin_scope.argtypes = [C.c_void_p, C.c_int]
        L.oracle_release.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
        L.oracle_hold_units.argtypes = [C.c_void_p]
        L.oracle_hold_units.restype = C.c_uint64
        L.oracle_stats.argtypes = [C.c_void_p, C.POINTER(_Stats)]
        L.oracle_timing.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.oracle_timing.restype = None
        L.oracle_dump_list.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_uint64]
        L.oracle_dump_list.restype = C.c_uint64
        L.oracle_next_fresh.argtypes = [C.c_void_p]
        L.oracle_next_fresh.restype = C.c_int32
        L.oracle_content_hash.argtypes = [C.c_void_p, C.c_uint32]
        L.oracle_content_hash.restype = C.c_uint64
        L.oracle_key_from_state.argtypes = [C.c_uint64]
        L.oracle_key_from_state.restype = C.c_uint64
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None


def _arr(p, n, dtype):
    if n == 0:
        return np.zeros(0, dtype)
    return np.ctypeslib.as_array(p, shape=(n,)).astype(dtype, copy=True)


def hash_blocks(tokens, offsets, block_size=16):
    """(keys uint64[N], blk_off int64[n_req+1]) in natural order."""
    tokens = np.ascontiguousarray(tokens, dtype=np.int32)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n_req = len(offsets) - 1
    blk_off = np.zeros(n_req + 1, np.int64)
    rc = lib().oracle_hash_blocks(_ptr(tokens), _ptr(offsets), n_req, block_size, None, _ptr(blk_off))
    if rc != OK:
        raise ValueError(f"oracle_hash_blocks: {rc}")
    keys = np.zeros(int(blk_off[-1]), np.uint64)
    lib().oracle_hash_blocks(_ptr(tokens), _ptr(offsets), n_req, block_size, _ptr(keys), None)
    return keys, blk_off


def content_hash(block_tokens):
    t = np.ascontiguousarray(block_tokens, dtype=np.int32)
    return int(lib().oracle_content_hash(_ptr(t), len(t)))


def key_from_state(s):
    return int(lib().oracle_key_from_state(s))


class OracleCache:
    def __init__(self, capacity_blocks, block_size=16, policy=POLICY_ARC):
        self._h = C.c_void_p()
        rc = lib().oracle_create(capacity_blocks, block_size, policy, C.byref(self._h))
        if rc != OK:
            raise ValueError(f"oracle_create: {rc}")
        self.block_size = block_size

    def set_pin_scope(self, scope):
        rc = lib().oracle_set_pin_scope(self._h, scope)
        if rc != OK:
            raise ValueError(f"oracle_set_pin_scope: {rc}")

    def release(self, block_ids):
        """Pin scope 2: one hold back per listed block ID, in order.  Returns 0 or a negative error code (no change)."""
        ids = np.ascontiguousarray(block_ids, dtype=np.int32)
        return int(lib().oracle_release(self._h, _ptr(ids), len(ids)))

    def hold_units(self):
        return int(lib().oracle_hold_units(self._h))

    def close(self):
        if self._h and _lib is not None:      # at interpreter exit the module globals may already be gone
            _lib.oracle_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _unpack(self, res, n_req):
        n = int(res.n_access)
        return dict(n_access=n, prefix_len=_arr(res.prefix_len, n_req, np.int32), blk_off=_arr(res.blk_off, n_req + 1, np.int64),
                    cls=_arr(res.cls, n, np.uint8), block_id=_arr(res.block_id, n, np.int32),
                    evicted_id=_arr(res.evicted_id, n, np.int32), p_after=_arr(res.p_after, n, np.int32),
                    alloc_ids=_arr(res.alloc_ids, res.n_alloc, np.int32), evict_ids=_arr(res.evict_ids, res.n_evict, np.int32))

    def step(self, tokens, offsets, unpack=True, chain_in=None):
        """Returns the outputs dict, or a negative error code (state unchanged).  chain_in: uint64[n_req] H4 states the
        requests continue from (None = every request is a new prompt); the dict then also has chain_state[n_req]."""
        tokens = np.ascontiguousarray(tokens, dtype=np.int32)
        offsets = np.ascontiguousarray(offsets, dtype=np.int64)
        n_req = len(offsets) - 1
        res = _Result()
        ci = None if chain_in is None else np.ascontiguousarray(chain_in, dtype=np.uint64)
        rc = lib().oracle_step_resume(self._h, _ptr(tokens), _ptr(offsets), _ptr(ci), n_req, C.byref(res))
        if rc != OK:
            return rc
        if not unpack:
            return int(res.n_access)
        out = self._unpack(res, n_req)
        out["chain_state"] = _arr(res.chain_state, n_req, np.uint64)
        return out

    def step_keys(self, requests_keys):
        """requests_keys: list of sequences of uint64 keys (block 0 first)."""
        blk_off = np.zeros(len(requests_keys) + 1, np.int64)
        blk_off[1:] = np.cumsum([len(k) for k in requests_keys])
        keys = np.array([k for ks in requests_keys for k in ks], dtype=np.uint64)
        res = _Result()
        rc = lib().oracle_step_keys(self._h, _ptr(keys), _ptr(blk_off), len(requests_keys), C.byref(res))
        if rc != OK:
            return rc
        return self._unpack(res, len(requests_keys))

    def stats(self):
        s = _Stats()
        lib().oracle_stats(self._h, C.byref(s))
        return {n: int(getattr(s, n)) for n in STAT_FIELDS + ["block_size", "policy"]}

    def timing(self):
        a, b = C.c_double(), C.c_double()
        lib().oracle_timing(self._h, C.byref(a), C.byref(b))
        return dict(hash_seconds=a.value, arc_seconds=b.value)

    def lists(self):
        """dict T1/T2/B1/B2 -> (keys, block_ids) LRU -> MRU, plus p and next_fresh."""
        out = {}
        for name, which in (("T1", 1), ("T2", 2), ("B1", 3), ("B2", 4)):
            n = int(lib().oracle_dump_list(self._h, which, None, None, 0))
            keys, blocks = np.zeros(n, np.uint64), np.zeros(n, np.int32)
            lib().oracle_dump_list(self._h, which, _ptr(keys), _ptr(blocks), n)
            out[name] = (keys, blocks)
        out["p"] = self.stats()["p"]
        out["next_fresh"] = int(lib().oracle_next_fresh(self._h))
        return out
