"""ctypes front end of the CPU oracle (oracle/wsref.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg may import this.  Nothing here imports the CUDA package
and the CUDA package never imports this.

All arrays are numpy.  Byte kernels take any dtype (viewed as bytes); attention takes float32
arrays that hold exactly the values the GPU receives (BF16 values widened to float32, or the
FP32 inputs of config 1) and returns float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wsref.c")
_LIB = os.path.join(_HERE, "libwsref.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/wsref.c with gcc -O2 -fopenmp (no -ffast-math). Returns the .so path."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32, i64, dbl = ctypes.c_int32, ctypes.c_int64, ctypes.c_double
        vp = ctypes.c_void_p
        lib.wsref_num_threads.restype = ctypes.c_int
        lib.wsref_kv_cache_write.argtypes = [vp, vp, i64, i32, i32, vp, vp, i32, i32, i32, i64, i32]
        lib.wsref_seq_to_head.argtypes = [vp, vp, i64, i32, i32, i32, i32, i32, i32]
        lib.wsref_head_to_seq.argtypes = [vp, vp, i64, i32, i32, i32, i32, i32, i32]
        lib.wsref_block_causal_attn.argtypes = [vp, vp, vp, vp, vp, i64, i64, vp, vp, i32, i32, i32, i32, i32, vp, vp, dbl, vp]
        lib.wsref_block_causal_attn_rows.argtypes = [vp, vp, vp, vp, vp, i64, i64, vp, vp, i32, i32, i32, i32, i32, vp, vp,
                                                     dbl, i32, vp, vp]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().wsref_num_threads())


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c(a, dtype=None):
    a = np.ascontiguousarray(a) if dtype is None else np.ascontiguousarray(a, dtype=dtype)
    return a


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what}: invalid arguments (rc={rc})")


def kv_cache_write(k_cache, v_cache, k_src, v_src, head_begin: int, row_offset: int):
    """In place on k_cache/v_cache [H, capacity, d] from k_src/v_src [n_rows, H_src, d]."""
    assert k_cache.flags.c_contiguous and v_cache.flags.c_contiguous
    H, capacity, d = k_cache.shape
    n_rows, H_src, d2 = k_src.shape
    assert d2 == d and v_src.shape == k_src.shape and v_cache.shape == k_cache.shape
    assert k_src.dtype == k_cache.dtype == v_src.dtype == v_cache.dtype
    ks, vs = _c(k_src), _c(v_src)
    rc = _load().wsref_kv_cache_write(_ptr(k_cache), _ptr(v_cache), capacity, H, d, _ptr(ks), _ptr(vs), n_rows, H_src,
                                      head_begin, row_offset, k_cache.dtype.itemsize)
    _check(rc, "kv_cache_write")


def seq_to_head(dst, src, P: int, g0: int, G: int):
    """dst [G, n_tok, H/P, d] (written in place) from src [n_tok, H, d]."""
    n_tok, H, d = src.shape
    assert dst.flags.c_contiguous and dst.dtype == src.dtype
    if H % P == 0:
        assert dst.shape == (G, n_tok, H // P, d)
    s = _c(src)
    _check(_load().wsref_seq_to_head(_ptr(dst), _ptr(s), n_tok, H, d, P, g0, G, src.dtype.itemsize), "seq_to_head")


def head_to_seq(dst, src, P: int, g0: int, G: int):
    """dst [n_tok, H, d] (only the selected heads are written) from src [G, n_tok, H/P, d]."""
    n_tok, H, d = dst.shape
    assert dst.flags.c_contiguous and dst.dtype == src.dtype
    if H % P == 0:
        assert src.shape == (G, n_tok, H // P, d)
    s = _c(src)
    _check(_load().wsref_head_to_seq(_ptr(dst), _ptr(s), n_tok, H, d, P, g0, G, src.dtype.itemsize), "head_to_seq")


def _attn_args(q, k_cache, v_cache, cache_len, k_new, v_new, q_block_end, kv_visible):
    q = _c(q, np.float32)
    Lq, H, d = q.shape
    k_cache, v_cache = _c(k_cache, np.float32), _c(v_cache, np.float32)
    assert k_cache.shape == v_cache.shape and k_cache.shape[0] == H and k_cache.shape[2] == d
    capacity = k_cache.shape[1]
    if k_new is None:
        Ln = 0
        k_new = v_new = np.zeros((0, H, d), np.float32)
    else:
        k_new, v_new = _c(k_new, np.float32), _c(v_new, np.float32)
        Ln = k_new.shape[0]
        assert k_new.shape == (Ln, H, d) and v_new.shape == (Ln, H, d)
    qe = _c(q_block_end, np.int32)
    kv = _c(kv_visible, np.int32)
    assert qe.ndim == 1 and qe.shape == kv.shape
    return q, k_cache, v_cache, capacity, int(cache_len), k_new, v_new, Ln, H, d, Lq, qe, kv


def block_causal_attn(q, k_cache, v_cache, cache_len, k_new, v_new, q_block_end, kv_visible, softmax_scale,
                      return_p: bool = False):
    """Returns (out [Lq,H,d] f64, lse [H,Lq] f64[, p [H,Lq,cache_len+Ln] f64])."""
    q, kc, vc, cap, Tc, kn, vn, Ln, H, d, Lq, qe, kv = _attn_args(q, k_cache, v_cache, cache_len, k_new, v_new,
                                                                 q_block_end, kv_visible)
    out = np.empty((Lq, H, d), np.float64)
    lse = np.empty((H, Lq), np.float64)
    p = np.empty((H, Lq, Tc + Ln), np.float64) if return_p else None
    rc = _load().wsref_block_causal_attn(_ptr(out), _ptr(lse), _ptr(q), _ptr(kc), _ptr(vc), cap, Tc, _ptr(kn), _ptr(vn), Ln,
                                         H, d, Lq, len(qe), _ptr(qe), _ptr(kv), float(softmax_scale), _ptr(p))
    _check(rc, "block_causal_attn")
    return (out, lse, p) if return_p else (out, lse)


def block_causal_attn_rows(q, k_cache, v_cache, cache_len, k_new, v_new, q_block_end, kv_visible, softmax_scale,
                           sample_rows, sample_heads):
    """The same definition for a list of (row, head) pairs. Returns (out [n,d] f64, lse [n] f64)."""
    q, kc, vc, cap, Tc, kn, vn, Ln, H, d, Lq, qe, kv = _attn_args(q, k_cache, v_cache, cache_len, k_new, v_new,
                                                                 q_block_end, kv_visible)
    rows, heads = _c(sample_rows, np.int32), _c(sample_heads, np.int32)
    assert rows.shape == heads.shape and rows.ndim == 1
    out = np.empty((len(rows), d), np.float64)
    lse = np.empty((len(rows),), np.float64)
    rc = _load().wsref_block_causal_attn_rows(_ptr(out), _ptr(lse), _ptr(q), _ptr(kc), _ptr(vc), cap, Tc, _ptr(kn), _ptr(vn),
                                              Ln, H, d, Lq, len(qe), _ptr(qe), _ptr(kv), float(softmax_scale), len(rows),
                                              _ptr(rows), _ptr(heads))
    _check(rc, "block_causal_attn_rows")
    return out, lse


def parity_metrics(got, ref):
    """north_star's two attention metrics, in FP64: (max_abs, rel_fro) over the whole tensor."""
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    diff = got - ref
    max_abs = float(np.max(np.abs(diff))) if diff.size else 0.0
    den = float(np.linalg.norm(ref.ravel()))
    rel = float(np.linalg.norm(diff.ravel()) / den) if den > 0 else float(np.linalg.norm(diff.ravel()))
    return max_abs, rel
