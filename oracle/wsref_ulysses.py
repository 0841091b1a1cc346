"""ctypes front end of the Ulysses-exchange oracle (oracle/wsref_ulysses.c, reading R20).

TEST INFRASTRUCTURE, NOT THE PRODUCT (see wsref.py): only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline leg may import this.  All ranks' tensors live in one process as lists of numpy arrays."""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wsref_ulysses.c")
_LIB = os.path.join(_HERE, "libwsref_ulysses.so")
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
        pp = ctypes.POINTER(vp)
        lib.wsref_ulysses_seq_to_head.argtypes = [vp, pp, i32, i32, i64, i64, i32, i32, i32]
        lib.wsref_ulysses_head_to_seq.argtypes = [vp, pp, i32, i32, i64, i64, i32, i32, i32]
        lib.wsref_kv_slice_broadcast_write.argtypes = [pp, pp, i32, i64, i32, i32, vp, vp, i32, i64, i32]
        _lib = lib
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _ptrs(arrays):
    return (ctypes.c_void_p * len(arrays))(*[a.ctypes.data for a in arrays])


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what}: invalid arguments (rc={rc})")


def seq_to_head(xs, Ls: int):
    """Exchange #1.  xs: P arrays X_r [Ls + La, H, d] -> P arrays Y_g [P * Ls + La, H / P, d]."""
    P = len(xs)
    xs = [np.ascontiguousarray(x) for x in xs]
    n, H, d = xs[0].shape
    La = n - Ls
    assert all(x.shape == (n, H, d) and x.dtype == xs[0].dtype for x in xs)
    ys = []
    for g in range(P):
        y = np.empty((P * Ls + La, H // P if H % P == 0 else 1, d), xs[0].dtype)
        _check(_load().wsref_ulysses_seq_to_head(_ptr(y), _ptrs(xs), g, P, Ls, La, H, d, xs[0].dtype.itemsize), "ulysses_seq_to_head")
        ys.append(y)
    return ys


def head_to_seq(os_, Ls: int):
    """Exchange #2.  os_: P arrays O_g [P * Ls + La, Hp, d] -> P arrays Z_r [Ls + La, P * Hp, d]."""
    P = len(os_)
    os_ = [np.ascontiguousarray(o) for o in os_]
    n, Hp, d = os_[0].shape
    La = n - P * Ls
    assert all(o.shape == (n, Hp, d) and o.dtype == os_[0].dtype for o in os_)
    zs = []
    for r in range(P):
        z = np.empty((Ls + La, P * Hp, d), os_[0].dtype)
        _check(_load().wsref_ulysses_head_to_seq(_ptr(z), _ptrs(os_), r, P, Ls, La, P * Hp, d, os_[0].dtype.itemsize),
               "ulysses_head_to_seq")
        zs.append(z)
    return zs


def kv_slice_broadcast_write(k_caches, v_caches, k_src, v_src, row_offset: int):
    """In place on the P ranks' caches [Hp, capacity, d] from the thinker's slice [n_rows, P * Hp, d]."""
    P = len(k_caches)
    Hp, capacity, d = k_caches[0].shape
    n_rows = k_src.shape[0]
    assert k_src.shape == (n_rows, P * Hp, d) and v_src.shape == k_src.shape
    assert all(c.flags.c_contiguous and c.shape == (Hp, capacity, d) and c.dtype == k_src.dtype for c in list(k_caches) + list(v_caches))
    ks, vs = np.ascontiguousarray(k_src), np.ascontiguousarray(v_src)
    rc = _load().wsref_kv_slice_broadcast_write(_ptrs(k_caches), _ptrs(v_caches), P, capacity, Hp, d, _ptr(ks), _ptr(vs), n_rows,
                                                int(row_offset), k_src.dtype.itemsize)
    _check(rc, "kv_slice_broadcast_write")
