"""ctypes front end of the FP8 K/V-cache oracle (oracle/wsref_fp8.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT (see wsref.py): only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this.  Format and quantiser: DESIGN.md readings R17/R18; the C file states them."""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wsref_fp8.c")
_LIB = os.path.join(_HERE, "libwsref_fp8.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32, i64, vp = ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p
        lib.wsref_e4m3_decode.argtypes = [ctypes.c_uint8]
        lib.wsref_e4m3_decode.restype = ctypes.c_double
        lib.wsref_e4m3_encode.argtypes = [ctypes.c_double]
        lib.wsref_e4m3_encode.restype = ctypes.c_uint8
        lib.wsref_fp8_row_exponent.argtypes = [vp, i32]
        lib.wsref_fp8_row_exponent.restype = ctypes.c_int
        lib.wsref_kv_cache_write_fp8.argtypes = [vp, vp, vp, vp, i64, i32, i32, vp, vp, i32, i32, i32, i64]
        lib.wsref_kv_cache_dequant_fp8.argtypes = [vp, vp, vp, i64, i32, i32, i64]
        _lib = lib
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def e4m3_decode(code: int) -> float:
    return float(_load().wsref_e4m3_decode(int(code) & 0xFF))


def e4m3_encode(y: float) -> int:
    return int(_load().wsref_e4m3_encode(float(y)))


def row_exponent(x) -> int:
    x = np.ascontiguousarray(x, np.float32)
    return int(_load().wsref_fp8_row_exponent(_ptr(x), x.size))


def kv_cache_write_fp8(k_cache8, v_cache8, k_exp, v_exp, k_src, v_src, head_begin: int, row_offset: int):
    """In place: cache8 uint8 [H, capacity, d], exp int8 [H, capacity]; src float32 [n_rows, H_src, d]."""
    for a, dt in ((k_cache8, np.uint8), (v_cache8, np.uint8), (k_exp, np.int8), (v_exp, np.int8)):
        assert a.dtype == dt and a.flags.c_contiguous
    H, capacity, d = k_cache8.shape
    assert v_cache8.shape == k_cache8.shape and k_exp.shape == (H, capacity) and v_exp.shape == (H, capacity)
    ks, vs = np.ascontiguousarray(k_src, np.float32), np.ascontiguousarray(v_src, np.float32)
    n_rows, H_src, d2 = ks.shape
    assert d2 == d and vs.shape == ks.shape
    rc = _load().wsref_kv_cache_write_fp8(_ptr(k_cache8), _ptr(v_cache8), _ptr(k_exp), _ptr(v_exp), capacity, H, d, _ptr(ks), _ptr(vs),
                                          n_rows, H_src, head_begin, row_offset)
    if rc != 0:
        raise ValueError(f"oracle kv_cache_write_fp8: invalid arguments (rc={rc})")


def kv_cache_dequant_fp8(cache8, exp, n_rows: int | None = None) -> np.ndarray:
    """float32 [H, capacity, d] with rows [0, n_rows) dequantised (the rest zero)."""
    assert cache8.dtype == np.uint8 and exp.dtype == np.int8 and cache8.flags.c_contiguous and exp.flags.c_contiguous
    H, capacity, d = cache8.shape
    n = capacity if n_rows is None else int(n_rows)
    out = np.zeros((H, capacity, d), np.float32)
    rc = _load().wsref_kv_cache_dequant_fp8(_ptr(out), _ptr(cache8), _ptr(exp), capacity, H, d, n)
    if rc != 0:
        raise ValueError(f"oracle kv_cache_dequant_fp8: invalid arguments (rc={rc})")
    return out
