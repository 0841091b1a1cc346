"""ctypes front end of the ring-buffer K/V-cache oracle (oracle/wsref_ring.c, reading R19).

TEST INFRASTRUCTURE, NOT THE PRODUCT (see wsref.py): only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this.  Attention on a ring cache is DEFINED as the plain oracle attention
(wsref.block_causal_attn) on the linearised window."""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

from . import wsref

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wsref_ring.c")
_LIB = os.path.join(_HERE, "libwsref_ring.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-o", tmp, _SRC])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32, i64, vp = ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p
        lib.wsref_ring_state.argtypes = [i64, i64, ctypes.POINTER(i64), ctypes.POINTER(i64)]
        lib.wsref_kv_cache_write_ring.argtypes = [vp, vp, i64, i32, i32, vp, vp, i32, i32, i32, i64, i32]
        lib.wsref_ring_linearise.argtypes = [vp, vp, i64, i32, i32, i64, i64, i32]
        _lib = lib
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what}: invalid arguments (rc={rc})")


def ring_state(rows_written: int, capacity: int):
    """(ring_start, cache_len) of the window after `rows_written` rows of the session."""
    a, b = ctypes.c_int64(), ctypes.c_int64()
    _check(_load().wsref_ring_state(int(rows_written), int(capacity), ctypes.byref(a), ctypes.byref(b)), "ring_state")
    return int(a.value), int(b.value)


def kv_cache_write_ring(k_cache, v_cache, k_src, v_src, head_begin: int, write_pos: int):
    """In place on k_cache/v_cache [H, capacity, d] from k_src/v_src [n_rows, H_src, d]; row r goes to physical row
    (write_pos + r) mod capacity."""
    assert k_cache.flags.c_contiguous and v_cache.flags.c_contiguous
    H, capacity, d = k_cache.shape
    n_rows, H_src, d2 = k_src.shape
    assert d2 == d and v_src.shape == k_src.shape and v_cache.shape == k_cache.shape
    assert k_src.dtype == k_cache.dtype == v_src.dtype == v_cache.dtype
    ks, vs = np.ascontiguousarray(k_src), np.ascontiguousarray(v_src)
    rc = _load().wsref_kv_cache_write_ring(_ptr(k_cache), _ptr(v_cache), capacity, H, d, _ptr(ks), _ptr(vs), n_rows, H_src,
                                           head_begin, int(write_pos), k_cache.dtype.itemsize)
    _check(rc, "kv_cache_write_ring")


def linearise(cache, ring_start: int, cache_len: int):
    """[H, cache_len, d]: the window in timeline order (oldest row first)."""
    cache = np.ascontiguousarray(cache)
    H, capacity, d = cache.shape
    lin = np.empty((H, cache_len, d), cache.dtype)
    _check(_load().wsref_ring_linearise(_ptr(lin), _ptr(cache), capacity, H, d, int(ring_start), int(cache_len),
                                        cache.dtype.itemsize), "ring_linearise")
    return lin


def block_causal_attn_ring(q, k_cache, v_cache, ring_start, cache_len, k_new, v_new, q_block_end, kv_visible, softmax_scale):
    """Block-causal attention whose cache keys are the ring's window in timeline order: the definition is the plain
    oracle on the linearised window.  Returns (out [Lq,H,d] f64, lse [H,Lq] f64)."""
    kl, vl = linearise(k_cache, ring_start, cache_len), linearise(v_cache, ring_start, cache_len)
    return wsref.block_causal_attn(q, kl, vl, cache_len, k_new, v_new, q_block_end, kv_visible, softmax_scale)
