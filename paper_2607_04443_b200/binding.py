"""ctypes binding of libws.so (include/ws.h): same names, argument marshalling only.

Tensors are torch CUDA tensors (PyTorch is used for device memory and streams, nothing else);
every step of the path runs in the library's own kernels.  There is NO fallback: if libws.so is
missing, or a tensor is not on a CUDA device, the call raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

DTYPE_BF16 = 0
DTYPE_F32 = 1
ABI_VERSION = 300  # WS_VERSION of include/ws.h this binding was written against

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "libws.so")
_lib = None

EXPORTS = (
    "ws_kv_cache_write", "ws_seq_to_head", "ws_head_to_seq", "ws_seq_to_head_multi", "ws_head_to_seq_multi", "ws_block_causal_attn_workspace_bytes",
    "ws_block_causal_attn", "ws_block_causal_attn_seq_layout", "ws_unit_forward_host_staging_bytes", "ws_unit_forward_host", "ws_status_string",
    "ws_version", "ws_last_cuda_error", "ws_kernel_launch_count", "ws_attn_schedule", "ws_kv_cache_write_fp8", "ws_block_causal_attn_fp8kv",
    "ws_kv_cache_write_ring", "ws_ring_state", "ws_block_causal_attn_ring",
    "ws_ulysses_push_seq_to_head", "ws_block_causal_attn_push_out", "ws_kv_slice_broadcast_write",
    "ws_block_causal_attn_static_ws",
)
STATIC_WORKSPACE_BYTES = 64 << 20  # WS_STATIC_WORKSPACE_BYTES of include/ws.h


class WsError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        msg = status_string(status)
        if status == -7:
            msg += f" [cudaError {load().ws_last_cuda_error()}]"
        super().__init__(f"{what}: {msg}")


class _BlockMask(ctypes.Structure):
    _fields_ = [("n_blocks", ctypes.c_int32), ("q_block_end", ctypes.POINTER(ctypes.c_int32)),
                ("kv_visible", ctypes.POINTER(ctypes.c_int32))]


def lib_path() -> str:
    return _LIB_PATH


def load():
    """Loads libws.so.  Raises (loudly) if it has not been built: there is no other path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(f"{_LIB_PATH} not found: build it with `python -m paper_2607_04443_b200.build` "
                           "(there is no CPU or PyTorch fallback)")
    lib = ctypes.CDLL(_LIB_PATH)
    i32, i64, vp, sz, f32 = ctypes.c_int32, ctypes.c_int64, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_float
    lib.ws_kv_cache_write.argtypes = [vp, vp, i64, i32, i32, vp, vp, i32, i32, i32, i64, ctypes.c_int, vp]
    lib.ws_kv_cache_write.restype = ctypes.c_int
    for fn in (lib.ws_seq_to_head, lib.ws_head_to_seq):
        fn.argtypes = [vp, vp, i64, i32, i32, i32, i32, i32, ctypes.c_int, vp]
        fn.restype = ctypes.c_int
    for fn in (lib.ws_seq_to_head_multi, lib.ws_head_to_seq_multi):
        fn.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(vp), i32, i64, i32, i32, i32, i32, i32, ctypes.c_int, vp]
        fn.restype = ctypes.c_int
    lib.ws_block_causal_attn_workspace_bytes.argtypes = [i32, i32, i32, i64, ctypes.c_int]
    lib.ws_block_causal_attn_workspace_bytes.restype = sz
    lib.ws_block_causal_attn.argtypes = [vp, vp, vp, vp, vp, i64, i64, vp, vp, i32, i32, i32, i32,
                                         ctypes.POINTER(_BlockMask), f32, vp, sz, ctypes.c_int, vp]
    lib.ws_block_causal_attn.restype = ctypes.c_int
    lib.ws_block_causal_attn_static_ws.argtypes = [vp, vp, vp, vp, vp, i64, i64, vp, vp, i32, i32, i32, i32,
                                                   ctypes.POINTER(_BlockMask), f32, ctypes.c_int, vp]
    lib.ws_block_causal_attn_static_ws.restype = ctypes.c_int
    lib.ws_block_causal_attn_seq_layout.argtypes = [vp, vp, vp, vp, vp, i64, i64, vp, vp, i32, i32, i32, i32, i32, i32,
                                                    ctypes.POINTER(_BlockMask), f32, vp, sz, ctypes.c_int, vp]
    lib.ws_block_causal_attn_seq_layout.restype = ctypes.c_int
    lib.ws_unit_forward_host_staging_bytes.argtypes = [i32, i32, i32, i32, i32, i64, i32]
    lib.ws_unit_forward_host_staging_bytes.restype = sz
    lib.ws_unit_forward_host.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, i64, vp, vp, i32, i64, i64, i32, i32, f32,
                                         vp, sz, vp]
    lib.ws_unit_forward_host.restype = ctypes.c_int
    lib.ws_attn_schedule.argtypes = [i32, i32, i64, i32, ctypes.POINTER(_BlockMask), i32, ctypes.POINTER(i32), ctypes.POINTER(i32),
                                     ctypes.POINTER(i32), ctypes.POINTER(i32), ctypes.POINTER(i64)]
    lib.ws_attn_schedule.restype = ctypes.c_int
    lib.ws_kv_cache_write_fp8.argtypes = [vp, vp, vp, vp, i64, i32, i32, vp, vp, i32, i32, i32, i64, vp]
    lib.ws_kv_cache_write_fp8.restype = ctypes.c_int
    lib.ws_block_causal_attn_fp8kv.argtypes = [vp, vp, vp, vp, vp, vp, vp, i64, i64, vp, vp, i32, i32, i32, i32, ctypes.POINTER(_BlockMask),
                                               f32, vp, sz, vp]
    lib.ws_block_causal_attn_fp8kv.restype = ctypes.c_int
    lib.ws_kv_cache_write_ring.argtypes = [vp, vp, i64, i32, i32, vp, vp, i32, i32, i32, i64, ctypes.c_int, vp]
    lib.ws_kv_cache_write_ring.restype = ctypes.c_int
    lib.ws_ring_state.argtypes = [i64, i64, ctypes.POINTER(i64), ctypes.POINTER(i64)]
    lib.ws_ring_state.restype = ctypes.c_int
    lib.ws_block_causal_attn_ring.argtypes = [vp, vp, vp, vp, vp, i64, i64, i64, vp, vp, i32, i32, i32, i32,
                                              ctypes.POINTER(_BlockMask), f32, vp, sz, ctypes.c_int, vp]
    lib.ws_block_causal_attn_ring.restype = ctypes.c_int
    lib.ws_ulysses_push_seq_to_head.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(vp), i32, i64, i64, i32, i32, i32, i32, ctypes.c_int, vp]
    lib.ws_ulysses_push_seq_to_head.restype = ctypes.c_int
    lib.ws_block_causal_attn_push_out.argtypes = [ctypes.POINTER(vp), i32, i32, i64, vp, vp, vp, vp, i64, i64, vp, vp, i32, i32, i32, i32,
                                                  ctypes.POINTER(_BlockMask), f32, vp, sz, ctypes.c_int, vp]
    lib.ws_block_causal_attn_push_out.restype = ctypes.c_int
    lib.ws_kv_slice_broadcast_write.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(vp), i32, i64, i32, i32, vp, vp, i32, i64, ctypes.c_int, vp]
    lib.ws_kv_slice_broadcast_write.restype = ctypes.c_int
    lib.ws_status_string.argtypes = [ctypes.c_int]
    lib.ws_status_string.restype = ctypes.c_char_p
    for fn in (lib.ws_version, lib.ws_last_cuda_error, lib.ws_kernel_launch_count):
        fn.argtypes = []
        fn.restype = ctypes.c_int
    if int(lib.ws_version()) != ABI_VERSION:  # a stale build would be called with the wrong argument lists
        raise RuntimeError(f"{_LIB_PATH} reports version {int(lib.ws_version())}, this binding needs {ABI_VERSION}: rebuild it with "
                           "`python -m paper_2607_04443_b200.build --force`")
    _lib = lib
    return lib


def version() -> int:
    return int(load().ws_version())


def status_string(status: int) -> str:
    return load().ws_status_string(int(status)).decode()


def kernel_launch_count() -> int:
    return int(load().ws_kernel_launch_count())


def _dt(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return DTYPE_BF16
    if t.dtype == torch.float32:
        return DTYPE_F32
    raise TypeError(f"unsupported dtype {t.dtype}: the library moves/computes BF16 or FP32")


def _dev(*tensors):
    for t in tensors:
        if t is None:
            continue
        if not t.is_cuda:
            raise RuntimeError("ws: tensors must live on a CUDA device (no CPU fallback exists)")
        if not t.is_contiguous():
            raise ValueError("ws: tensors must be contiguous")


def _p(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream) -> ctypes.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _ok(rc: int, what: str):
    if rc != 0:
        raise WsError(rc, what)


def kv_cache_write(k_cache, v_cache, k_src, v_src, head_begin: int = 0, row_offset: int = 0, stream=None):
    """cache[h, row_offset + r, :] = src[r, head_begin + h, :] for K and V (ws.h a1)."""
    _dev(k_cache, v_cache, k_src, v_src)
    H, capacity, d = k_cache.shape
    n_rows, H_src, d2 = k_src.shape
    if d2 != d or v_cache.shape != k_cache.shape or v_src.shape != k_src.shape:
        raise ValueError("ws_kv_cache_write: shape mismatch")
    if not (k_cache.dtype == v_cache.dtype == k_src.dtype == v_src.dtype):
        raise TypeError("ws_kv_cache_write: dtype mismatch")
    rc = load().ws_kv_cache_write(_p(k_cache), _p(v_cache), capacity, H, d, _p(k_src), _p(v_src), n_rows, H_src, head_begin,
                                  row_offset, _dt(k_cache), _stream(stream))
    _ok(rc, "ws_kv_cache_write")


def seq_to_head(dst, src, P: int, g0: int, G: int, stream=None):
    """dst[g, t, c, :] = src[t, (g0 + g) * H/P + c, :]  (ws.h a2); src [n_tok, H, d]."""
    _dev(dst, src)
    n_tok, H, d = src.shape
    if dst.dtype != src.dtype:
        raise TypeError("ws_seq_to_head: dtype mismatch")
    if P > 0 and H % P == 0 and tuple(dst.shape) != (G, n_tok, H // P, d):
        raise ValueError("ws_seq_to_head: dst must be [G, n_tok, H/P, d]")
    _ok(load().ws_seq_to_head(_p(dst), _p(src), n_tok, H, d, P, g0, G, _dt(src), _stream(stream)), "ws_seq_to_head")


def head_to_seq(dst, src, P: int, g0: int, G: int, stream=None):
    """dst[t, (g0 + g) * H/P + c, :] = src[g, t, c, :]  (ws.h a4); dst [n_tok, H, d]."""
    _dev(dst, src)
    n_tok, H, d = dst.shape
    if dst.dtype != src.dtype:
        raise TypeError("ws_head_to_seq: dtype mismatch")
    if P > 0 and H % P == 0 and tuple(src.shape) != (G, n_tok, H // P, d):
        raise ValueError("ws_head_to_seq: src must be [G, n_tok, H/P, d]")
    _ok(load().ws_head_to_seq(_p(dst), _p(src), n_tok, H, d, P, g0, G, _dt(dst), _stream(stream)), "ws_head_to_seq")


def _multi(fn_name, toks, heads, P, g0, G, stream, to_head):
    """toks: token-major [n_tok, H, d] tensors; heads: head-major [G, n_tok, H/P, d] tensors (same shapes throughout)."""
    if len(toks) != len(heads) or not toks:
        raise ValueError(f"{fn_name}: need as many sources as destinations (at least one)")
    _dev(*toks, *heads)
    n_tok, H, d = toks[0].shape
    for t, h in zip(toks, heads):
        if tuple(t.shape) != (n_tok, H, d) or t.dtype != toks[0].dtype or h.dtype != toks[0].dtype:
            raise ValueError(f"{fn_name}: all tensors must share shape and dtype")
        if P > 0 and H % P == 0 and tuple(h.shape) != (G, n_tok, H // P, d):
            raise ValueError(f"{fn_name}: head-major tensors must be [G, n_tok, H/P, d]")
    n = len(toks)
    dsts, srcs = (heads, toks) if to_head else (toks, heads)
    da = (ctypes.c_void_p * n)(*[t.data_ptr() for t in dsts])
    sa = (ctypes.c_void_p * n)(*[t.data_ptr() for t in srcs])
    rc = getattr(load(), fn_name)(da, sa, n, n_tok, H, d, P, g0, G, _dt(toks[0]), _stream(stream))
    _ok(rc, fn_name)


def seq_to_head_multi(dsts, srcs, P: int, g0: int, G: int, stream=None):
    """ws_seq_to_head on up to four same-shaped tensors in one launch (ws.h)."""
    _multi("ws_seq_to_head_multi", list(srcs), list(dsts), P, g0, G, stream, True)


def head_to_seq_multi(dsts, srcs, P: int, g0: int, G: int, stream=None):
    """ws_head_to_seq on up to four same-shaped tensors in one launch (ws.h)."""
    _multi("ws_head_to_seq_multi", list(dsts), list(srcs), P, g0, G, stream, False)


def block_causal_attn_workspace_bytes(Lq: int, H: int, d: int, kv_total: int, dtype=torch.bfloat16) -> int:
    dt = DTYPE_BF16 if dtype == torch.bfloat16 else DTYPE_F32
    return int(load().ws_block_causal_attn_workspace_bytes(Lq, H, d, kv_total, dt))


def _attn_args(name, out, q, k_cache, v_cache, k_new, v_new, lse, q_block_end, kv_visible, token_major=False, cache_dtype=None):
    """The shape, dtype and mask rules shared by every attention wrapper.  q (and out, k_new, v_new) are [L, Hq, d]; the cache
    is [H, capacity, d] with H == Hq, except for the token-major call (token_major=True) where the cache names the H of the
    Hq heads that take part.  cache_dtype overrides the cache's element type (uint8 codes for the FP8 cache).
    Returns (Lq, H, d, capacity, Ln, mask); `mask` keeps its arrays alive."""
    Lq, Hq, d = q.shape
    capacity = k_cache.shape[1]
    H = k_cache.shape[0] if token_major else Hq
    Ln = 0 if k_new is None else k_new.shape[0]
    if out is not None and (out.shape != q.shape or out.dtype != q.dtype):
        raise ValueError(f"{name}: out must match q")
    if tuple(k_cache.shape) != (H, capacity, d) or v_cache.shape != k_cache.shape:
        raise ValueError(f"{name}: cache must be [H, capacity, d]")
    if k_new is not None and (tuple(k_new.shape) != (Ln, Hq, d) or v_new is None or v_new.shape != k_new.shape):
        raise ValueError(f"{name}: k_new/v_new must be [Ln, {'H_total' if token_major else 'H'}, d]")
    for t, want in ((k_cache, cache_dtype or q.dtype), (v_cache, cache_dtype or q.dtype), (k_new, q.dtype), (v_new, q.dtype)):
        if t is not None and t.dtype != want:
            raise TypeError(f"{name}: dtype mismatch")
    if lse is not None and (lse.dtype != torch.float32 or tuple(lse.shape) != (H, Lq)):
        raise ValueError(f"{name}: lse must be float32 [H, Lq]")
    n = len(q_block_end)
    if len(kv_visible) != n:
        raise ValueError(f"{name}: mask arrays differ in length")
    qe = (ctypes.c_int32 * n)(*[int(x) for x in q_block_end])
    kv = (ctypes.c_int32 * n)(*[int(x) for x in kv_visible])
    mask = _BlockMask(n, qe, kv)
    mask._keep = (qe, kv)
    return Lq, H, d, capacity, Ln, mask


def block_causal_attn(out, q, k_cache, v_cache, cache_len: int, k_new, v_new, q_block_end: Sequence[int],
                      kv_visible: Sequence[int], softmax_scale: float, workspace, lse=None, stream=None):
    """Block-causal unit attention (ws.h a3).  out/q [Lq,H,d]; caches [H,capacity,d]; k_new/v_new [Ln,H,d] or None."""
    _dev(out, q, k_cache, v_cache, k_new, v_new, workspace, lse)
    Lq, H, d, capacity, Ln, mask = _attn_args("ws_block_causal_attn", out, q, k_cache, v_cache, k_new, v_new, lse, q_block_end, kv_visible)
    rc = load().ws_block_causal_attn(_p(out), _p(lse), _p(q), _p(k_cache), _p(v_cache), capacity, int(cache_len), _p(k_new),
                                     _p(v_new), Ln, H, d, Lq, ctypes.byref(mask), float(softmax_scale), _p(workspace),
                                     workspace.numel() * workspace.element_size(), _dt(q), _stream(stream))
    _ok(rc, "ws_block_causal_attn")


def block_causal_attn_static_ws(out, q, k_cache, v_cache, cache_len: int, k_new, v_new, q_block_end: Sequence[int],
                                kv_visible: Sequence[int], softmax_scale: float, lse=None, stream=None):
    """ws_block_causal_attn for callers that cannot allocate device memory (ws.h, ws_block_causal_attn_static_ws).

    Same arguments and results as block_causal_attn, without the workspace: the scratch is a 64 MiB array built into
    libws.so's device image, so neither this wrapper nor the library allocates anything.  It is meant for code that has
    no allocator to turn to -- a plug-in in a serving process whose framework owns all of HBM, the per-unit real-time
    loop where a cudaMalloc would stall the device, set-ups that forbid allocation after start-up.  Problems whose
    scratch need exceeds STATIC_WORKSPACE_BYTES are refused (WsError, status WS_ERR_WORKSPACE, nothing launched).  All
    calls on one device share the array: keep them on one stream (overlapping calls race), and make the first call on
    a device during set-up, before any stream capture."""
    _dev(out, q, k_cache, v_cache, k_new, v_new, lse)
    Lq, H, d, capacity, Ln, mask = _attn_args("ws_block_causal_attn_static_ws", out, q, k_cache, v_cache, k_new, v_new, lse, q_block_end, kv_visible)
    rc = load().ws_block_causal_attn_static_ws(_p(out), _p(lse), _p(q), _p(k_cache), _p(v_cache), capacity, int(cache_len),
                                               _p(k_new), _p(v_new), Ln, H, d, Lq, ctypes.byref(mask), float(softmax_scale),
                                               _dt(q), _stream(stream))
    if rc == -6:
        need = block_causal_attn_workspace_bytes(Lq, H, d, int(cache_len) + Ln, q.dtype)
        raise WsError(rc, f"ws_block_causal_attn_static_ws: this problem needs up to {need} bytes of scratch, the built-in "
                          f"array holds {STATIC_WORKSPACE_BYTES}")
    _ok(rc, "ws_block_causal_attn_static_ws")


def kv_cache_write_ring(k_cache, v_cache, k_src, v_src, head_begin: int = 0, write_pos: int = 0, stream=None):
    """Ring cache write (ws.h ws_kv_cache_write_ring): cache[h, (write_pos + r) mod capacity, :] = src[r, head_begin + h, :]."""
    _dev(k_cache, v_cache, k_src, v_src)
    H, capacity, d = k_cache.shape
    n_rows, H_src, d2 = k_src.shape
    if d2 != d or v_cache.shape != k_cache.shape or v_src.shape != k_src.shape:
        raise ValueError("ws_kv_cache_write_ring: shape mismatch")
    if not (k_cache.dtype == v_cache.dtype == k_src.dtype == v_src.dtype):
        raise TypeError("ws_kv_cache_write_ring: dtype mismatch")
    rc = load().ws_kv_cache_write_ring(_p(k_cache), _p(v_cache), capacity, H, d, _p(k_src), _p(v_src), n_rows, H_src, head_begin,
                                       int(write_pos), _dt(k_cache), _stream(stream))
    _ok(rc, "ws_kv_cache_write_ring")


def ring_state(rows_written: int, capacity: int):
    """(ring_start, cache_len) of a ring cache after rows_written rows of the session (ws.h ws_ring_state; host only)."""
    a, b = ctypes.c_int64(0), ctypes.c_int64(0)
    _ok(load().ws_ring_state(int(rows_written), int(capacity), ctypes.byref(a), ctypes.byref(b)), "ws_ring_state")
    return int(a.value), int(b.value)


def block_causal_attn_ring(out, q, k_cache, v_cache, ring_start: int, cache_len: int, k_new, v_new, q_block_end: Sequence[int],
                           kv_visible: Sequence[int], softmax_scale: float, workspace, lse=None, stream=None):
    """Block-causal unit attention on a ring cache (ws.h ws_block_causal_attn_ring): cache key j is physical row
    (ring_start + j) mod capacity.  Shapes as block_causal_attn."""
    _dev(out, q, k_cache, v_cache, k_new, v_new, workspace, lse)
    Lq, H, d, capacity, Ln, mask = _attn_args("ws_block_causal_attn_ring", out, q, k_cache, v_cache, k_new, v_new, lse, q_block_end, kv_visible)
    rc = load().ws_block_causal_attn_ring(_p(out), _p(lse), _p(q), _p(k_cache), _p(v_cache), capacity, int(ring_start), int(cache_len),
                                          _p(k_new), _p(v_new), Ln, H, d, Lq, ctypes.byref(mask), float(softmax_scale), _p(workspace),
                                          workspace.numel() * workspace.element_size(), _dt(q), _stream(stream))
    _ok(rc, "ws_block_causal_attn_ring")


def _ptr_array(tensors):
    return (ctypes.c_void_p * len(tensors))(*[t.data_ptr() for t in tensors])


def ulysses_push_seq_to_head(peer_dsts, srcs, Ls: int, rank: int, stream=None):
    """Exchange #1 of a Ulysses group, run by rank `rank` (ws.h ws_ulysses_push_seq_to_head).  srcs: this rank's tensors
    X [Ls + La, H, d] (up to 4: Q, K_new, V_new); peer_dsts[i][g]: tensor i's Y_g [P * Ls + La, H / P, d] on peer g
    (a tensor in this process's address space: local, or peer-mapped)."""
    srcs = list(srcs)
    P = len(peer_dsts[0])
    flat = [t for row in peer_dsts for t in row]
    _dev(*srcs, *flat)
    n, H, d = srcs[0].shape
    La = n - Ls
    for x in srcs:
        if tuple(x.shape) != (n, H, d) or x.dtype != srcs[0].dtype:
            raise ValueError("ws_ulysses_push_seq_to_head: sources must share shape and dtype")
    for row in peer_dsts:
        if len(row) != P:
            raise ValueError("ws_ulysses_push_seq_to_head: every tensor needs one destination per peer")
        for y in row:
            if y.dtype != srcs[0].dtype or (H % P == 0 and tuple(y.shape) != (P * Ls + La, H // P, d)):
                raise ValueError("ws_ulysses_push_seq_to_head: destinations must be [P * Ls + La, H / P, d]")
    rc = load().ws_ulysses_push_seq_to_head(_ptr_array(flat), _ptr_array(srcs), len(srcs), int(Ls), int(La), H, d, P, int(rank),
                                            _dt(srcs[0]), _stream(stream))
    _ok(rc, "ws_ulysses_push_seq_to_head")


def block_causal_attn_push_out(peer_outs, rank: int, Ls: int, q, k_cache, v_cache, cache_len: int, k_new, v_new,
                               q_block_end: Sequence[int], kv_visible: Sequence[int], softmax_scale: float, workspace, lse=None,
                               stream=None):
    """Attention of rank `rank` on its heads with exchange #2 fused into the epilogue (ws.h ws_block_causal_attn_push_out).
    peer_outs[r]: peer r's token-major output Z_r [Ls + La, P * H, d]; q [P * Ls + La, H, d]."""
    peer_outs = list(peer_outs)
    _dev(*peer_outs, q, k_cache, v_cache, k_new, v_new, workspace, lse)
    P = len(peer_outs)
    Lq, H, d, capacity, Ln, mask = _attn_args("ws_block_causal_attn_push_out", None, q, k_cache, v_cache, k_new, v_new, lse,
                                              q_block_end, kv_visible)
    La = Lq - P * Ls
    for z in peer_outs:
        if z.dtype != q.dtype or tuple(z.shape) != (Ls + La, P * H, d):
            raise ValueError("ws_block_causal_attn_push_out: peer outputs must be [Ls + La, P * H, d]")
    rc = load().ws_block_causal_attn_push_out(_ptr_array(peer_outs), P, int(rank), int(Ls), _p(lse), _p(q), _p(k_cache), _p(v_cache),
                                              capacity, int(cache_len), _p(k_new), _p(v_new), Ln, H, d, Lq, ctypes.byref(mask),
                                              float(softmax_scale), _p(workspace), workspace.numel() * workspace.element_size(),
                                              _dt(q), _stream(stream))
    _ok(rc, "ws_block_causal_attn_push_out")


def kv_slice_broadcast_write(peer_k_caches, peer_v_caches, k_src, v_src, row_offset: int = 0, stream=None):
    """The thinker's slice [n_rows, P * Hp, d] written into every rank's cache [Hp, capacity, d] by one kernel
    (ws.h ws_kv_slice_broadcast_write)."""
    peer_k_caches, peer_v_caches = list(peer_k_caches), list(peer_v_caches)
    _dev(*peer_k_caches, *peer_v_caches, k_src, v_src)
    P = len(peer_k_caches)
    Hp, capacity, d = peer_k_caches[0].shape
    n_rows = k_src.shape[0]
    if len(peer_v_caches) != P or tuple(k_src.shape) != (n_rows, P * Hp, d) or v_src.shape != k_src.shape:
        raise ValueError("ws_kv_slice_broadcast_write: shape mismatch")
    for c in peer_k_caches + peer_v_caches:
        if tuple(c.shape) != (Hp, capacity, d) or c.dtype != k_src.dtype:
            raise ValueError("ws_kv_slice_broadcast_write: every cache must be [Hp, capacity, d] of the slice's dtype")
    rc = load().ws_kv_slice_broadcast_write(_ptr_array(peer_k_caches), _ptr_array(peer_v_caches), P, capacity, Hp, d, _p(k_src),
                                            _p(v_src), n_rows, int(row_offset), _dt(k_src), _stream(stream))
    _ok(rc, "ws_kv_slice_broadcast_write")


def kv_cache_write_fp8(k_cache8, v_cache8, k_exp, v_exp, k_src, v_src, head_begin: int = 0, row_offset: int = 0, stream=None):
    """FP8 cache write (ws.h ws_kv_cache_write_fp8): cache8 uint8 [H, capacity, d], exp int8 [H, capacity], src BF16 [n_rows, H_src, d]."""
    _dev(k_cache8, v_cache8, k_exp, v_exp, k_src, v_src)
    H, capacity, d = k_cache8.shape
    n_rows, H_src, d2 = k_src.shape
    if d2 != d or v_cache8.shape != k_cache8.shape or v_src.shape != k_src.shape or tuple(k_exp.shape) != (H, capacity) or \
            v_exp.shape != k_exp.shape:
        raise ValueError("ws_kv_cache_write_fp8: shape mismatch")
    if k_cache8.dtype != torch.uint8 or v_cache8.dtype != torch.uint8 or k_exp.dtype != torch.int8 or v_exp.dtype != torch.int8 or \
            k_src.dtype != torch.bfloat16 or v_src.dtype != torch.bfloat16:
        raise TypeError("ws_kv_cache_write_fp8: caches uint8, exponents int8, sources bfloat16")
    rc = load().ws_kv_cache_write_fp8(_p(k_cache8), _p(v_cache8), _p(k_exp), _p(v_exp), capacity, H, d, _p(k_src), _p(v_src), n_rows,
                                      H_src, head_begin, row_offset, _stream(stream))
    _ok(rc, "ws_kv_cache_write_fp8")


def block_causal_attn_fp8kv(out, q, k_cache8, v_cache8, k_exp, v_exp, cache_len: int, k_new, v_new, q_block_end: Sequence[int],
                            kv_visible: Sequence[int], softmax_scale: float, workspace, lse=None, stream=None):
    """Block-causal unit attention on an FP8 cache (ws.h ws_block_causal_attn_fp8kv); q/out/k_new/v_new BF16."""
    _dev(out, q, k_cache8, v_cache8, k_exp, v_exp, k_new, v_new, workspace, lse)
    if q.dtype != torch.bfloat16:
        raise TypeError("ws_block_causal_attn_fp8kv: q, out, k_new, v_new must be bfloat16")
    Lq, H, d, capacity, Ln, mask = _attn_args("ws_block_causal_attn_fp8kv", out, q, k_cache8, v_cache8, k_new, v_new, lse,
                                              q_block_end, kv_visible, cache_dtype=torch.uint8)
    if tuple(k_exp.shape) != (H, capacity) or v_exp.shape != k_exp.shape or k_exp.dtype != torch.int8 or v_exp.dtype != torch.int8:
        raise ValueError("ws_block_causal_attn_fp8kv: exponents must be int8 [H, capacity]")
    rc = load().ws_block_causal_attn_fp8kv(_p(out), _p(lse), _p(q), _p(k_cache8), _p(v_cache8), _p(k_exp), _p(v_exp), capacity,
                                           int(cache_len), _p(k_new), _p(v_new), Ln, H, d, Lq, ctypes.byref(mask), float(softmax_scale),
                                           _p(workspace), workspace.numel() * workspace.element_size(), _stream(stream))
    _ok(rc, "ws_block_causal_attn_fp8kv")


def block_causal_attn_seq_layout(out_seq, q_seq, k_cache, v_cache, cache_len: int, k_new_seq, v_new_seq, head_begin: int,
                                 q_block_end: Sequence[int], kv_visible: Sequence[int], softmax_scale: float, workspace,
                                 lse=None, stream=None):
    """Relayouts fused into attention (ws.h a2+a3+a4): q_seq/out_seq [Lq, H_total, d], k_new_seq/v_new_seq
    [Ln, H_total, d] or None; the cache [H, capacity, d] names the H heads [head_begin, head_begin + H) taken."""
    _dev(out_seq, q_seq, k_cache, v_cache, k_new_seq, v_new_seq, workspace, lse)
    H_total = q_seq.shape[1]
    Lq, H, d, capacity, Ln, mask = _attn_args("ws_block_causal_attn_seq_layout", out_seq, q_seq, k_cache, v_cache, k_new_seq, v_new_seq,
                                              lse, q_block_end, kv_visible, token_major=True)
    rc = load().ws_block_causal_attn_seq_layout(_p(out_seq), _p(lse), _p(q_seq), _p(k_cache), _p(v_cache), capacity, int(cache_len),
                                                _p(k_new_seq), _p(v_new_seq), Ln, H_total, int(head_begin), H, d, Lq,
                                                ctypes.byref(mask), float(softmax_scale), _p(workspace),
                                                workspace.numel() * workspace.element_size(), _dt(q_seq), _stream(stream))
    _ok(rc, "ws_block_causal_attn_seq_layout")


def attn_schedule(Lq: int, H: int, cache_len: int, Ln: int, q_block_end: Sequence[int], kv_visible: Sequence[int], n_sms: int):
    """Host-only: the attention work schedule for a device with n_sms SMs (ws.h ws_attn_schedule).
    Returns dict(grid, n_waves, unit_iters [n_units], unit_kv_tiles [n_units], pool_begin [grid + 1])."""
    n = len(q_block_end)
    qe = (ctypes.c_int32 * n)(*[int(x) for x in q_block_end])
    kv = (ctypes.c_int32 * n)(*[int(x) for x in kv_visible])
    mask = _BlockMask(n, qe, kv)
    n_units = (Lq + 255) // 256
    grid, waves = ctypes.c_int32(0), ctypes.c_int32(0)
    iters = (ctypes.c_int32 * max(n_units, 1))()
    tiles = (ctypes.c_int32 * max(n_units, 1))()
    pool = (ctypes.c_int64 * (n_sms + 1))()
    rc = load().ws_attn_schedule(Lq, H, int(cache_len), Ln, ctypes.byref(mask), n_sms, ctypes.byref(grid), ctypes.byref(waves), iters,
                                 tiles, pool)
    _ok(rc, "ws_attn_schedule")
    return dict(grid=grid.value, n_waves=waves.value, unit_iters=list(iters)[:n_units], unit_kv_tiles=list(tiles)[:n_units],
                pool_begin=list(pool)[:grid.value + 1])


def unit_forward_host_staging_bytes(Lq, Ln, H, d, n_slice_rows, kv_total, n_steps) -> int:
    return int(load().ws_unit_forward_host_staging_bytes(Lq, Ln, H, d, n_slice_rows, kv_total, n_steps))


def unit_forward_host(out_host, q_host, k_new_host, v_new_host, k_cache, v_cache, k_slice_host, v_slice_host,
                      row_offset: int, cache_len_after: int, softmax_scale: float, staging, stream=None):
    """One unit from HOST (pinned CPU) tensors (ws.h a5).  q_host/out_host [n_steps, Lq, H, d] BF16 CPU tensors,
    k_new_host/v_new_host [n_steps, Ln, H, d] or None, slices [n_rows, H, d] or None; caches and staging on the GPU."""
    _dev(k_cache, v_cache, staging)
    for t in (out_host, q_host, k_new_host, v_new_host, k_slice_host, v_slice_host):
        if t is not None and (t.is_cuda or not t.is_contiguous() or t.dtype != torch.bfloat16):
            raise ValueError("ws_unit_forward_host: host tensors must be contiguous BF16 CPU tensors")
    n_steps, Lq, H, d = q_host.shape
    Ln = 0 if k_new_host is None else k_new_host.shape[1]
    n_rows = 0 if k_slice_host is None else k_slice_host.shape[0]
    capacity = k_cache.shape[1]
    rc = load().ws_unit_forward_host(_p(out_host), _p(q_host), _p(k_new_host), _p(v_new_host), Lq, Ln, n_steps, _p(k_cache),
                                     _p(v_cache), capacity, _p(k_slice_host), _p(v_slice_host), n_rows, int(row_offset),
                                     int(cache_len_after), H, d, float(softmax_scale), _p(staging),
                                     staging.numel() * staging.element_size(), _stream(stream))
    _ok(rc, "ws_unit_forward_host")
