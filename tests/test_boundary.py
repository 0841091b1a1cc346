"""The C-ABI boundary without a GPU: libws.so loads, exports every symbol include/ws.h declares,
and rejects bad arguments before touching CUDA (so these calls are safe on a CPU-only box).
No compute call is made here."""
import ctypes
import os
import re

import pytest
import torch

import paper_2607_04443_b200 as ws
from paper_2607_04443_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

OK, INVALID, UNSUPPORTED, ALIGN, RANGE, OVERLAP, WORKSPACE, CUDA = 0, -1, -2, -3, -4, -5, -6, -7


@pytest.fixture(scope="module")
def lib():
    build.build_lib()
    return binding.load()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "ws.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ws_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = declared_functions()
    assert set(names) == set(binding.EXPORTS), (names, binding.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None
    # and nothing from the oracle is linked in
    syms = os.popen(f"nm -D --defined-only {binding.lib_path()}").read()
    assert "wsref" not in syms
    exported = set(re.findall(r" T (ws_[a-z0-9_]+)", syms))
    assert exported == set(names)


def test_version_and_status_strings(lib):
    assert ws.version() == ws.ABI_VERSION == 300
    assert ws.status_string(0) == "WS_OK"
    for code in range(-7, 0):
        assert ws.status_string(code).startswith("WS_ERR_")
    assert ws.status_string(-99) == "WS_ERR_UNKNOWN"


def P(x):
    return ctypes.c_void_p(x)


A, B, C, D = 0x10000000, 0x20000000, 0x30000000, 0x40000000  # fake, 16-byte aligned, far apart


def test_kv_cache_write_rejects_bad_arguments(lib):
    f = lib.ws_kv_cache_write
    good = dict(kc=A, vc=B, cap=1024, H=4, d=128, ks=C, vs=D, n=64, Hs=8, hb=2, off=100, dt=0)

    def call(**kw):
        a = dict(good, **kw)
        return f(P(a["kc"]), P(a["vc"]), a["cap"], a["H"], a["d"], P(a["ks"]), P(a["vs"]), a["n"], a["Hs"], a["hb"], a["off"],
                 a["dt"], None)

    assert call(off=1024 - 63) == RANGE
    assert call(off=-1) == RANGE
    assert call(hb=5) == INVALID          # head_begin + H > H_src
    assert call(kc=0) == INVALID
    assert call(dt=7) == UNSUPPORTED
    assert call(kc=A + 8) == ALIGN
    assert call(d=4) == ALIGN             # 8-byte rows
    assert call(ks=A + 4096) == OVERLAP   # source inside the K cache
    assert call(vc=A + 1024) == OVERLAP   # caches overlap each other
    assert call(n=0) == OK                # no-op, nothing launched


def test_relayout_rejects_bad_arguments(lib):
    for f in (lib.ws_seq_to_head, lib.ws_head_to_seq):
        def call(dst=A, src=B, n_tok=100, H=40, d=128, Pn=4, g0=1, G=1, dt=0):
            return f(P(dst), P(src), n_tok, H, d, Pn, g0, G, dt, None)

        assert call(Pn=3) == INVALID      # H % P != 0
        assert call(g0=4) == INVALID
        assert call(g0=3, G=2) == INVALID
        assert call(Pn=0) == INVALID
        assert call(dst=0) == INVALID
        assert call(dt=5) == UNSUPPORTED
        assert call(src=B + 2) == ALIGN
        assert call(src=A + 256) == OVERLAP
        assert call(n_tok=0) == OK
        assert call(G=0) == OK


def test_attention_rejects_bad_arguments(lib):
    f = lib.ws_block_causal_attn
    Mask = binding._BlockMask

    def call(out=A, q=B, kc=C, vc=D, cap=512, Tc=512, kn=0x50000000, vn=0x60000000, Ln=64, H=2, d=128, Lq=64, qe=(32, 64),
             kv=(544, 576), scale=0.1, wsp=0x70000000, wsb=1 << 30, dt=0, lse=None):
        n = len(qe)
        m = Mask(n, (ctypes.c_int32 * n)(*qe), (ctypes.c_int32 * n)(*kv))
        return f(P(out), lse, P(q), P(kc), P(vc), cap, Tc, P(kn) if kn else None, P(vn) if vn else None, Ln, H, d, Lq,
                 ctypes.byref(m), scale, P(wsp) if wsp else None, wsb, dt, None)

    assert call(d=96) == UNSUPPORTED
    assert call(dt=3) == UNSUPPORTED
    assert call(qe=(32, 63)) == INVALID             # last != Lq
    assert call(qe=(32, 32)) == INVALID             # not strictly increasing
    assert call(kv=(576, 544)) == INVALID           # decreasing visibility
    assert call(kv=(544, 577)) == RANGE             # beyond cache_len + Ln
    assert call(Tc=513) == RANGE                    # cache_len > capacity
    assert call(kn=0) == INVALID                    # Ln > 0 but k_new NULL
    assert call(Ln=0, kv=(100, 512)) == INVALID     # Ln == 0 but k_new given
    assert call(scale=-1.0) == INVALID
    assert call(scale=float("nan")) == INVALID
    assert call(q=B + 8) == ALIGN
    assert call(wsp=0) == WORKSPACE
    assert call(wsb=1024) == WORKSPACE
    assert call(wsp=0x70000010) == WORKSPACE        # not 256-byte aligned
    assert call(qe=tuple(range(1, 131)), kv=tuple([576] * 130), Lq=130) == UNSUPPORTED  # > WS_MAX_MASK_BLOCKS


def test_ring_entry_points_reject_bad_arguments_and_ring_state_is_host_only(lib):
    """the ring cache write / attention check everything before CUDA is touched; ws_ring_state is pure
    host logic and is compared with the rule of DESIGN.md R19 written out again here."""
    i64 = ctypes.c_int64
    for W in list(range(0, 40)) + [10 ** 12 + 3]:
        for cap in (1, 7, 16):
            a, b = i64(-5), i64(-5)
            assert lib.ws_ring_state(W, cap, ctypes.byref(a), ctypes.byref(b)) == OK
            assert (a.value, b.value) == ((0, W) if W < cap else (W % cap, cap))
    a, b = i64(), i64()
    assert lib.ws_ring_state(-1, 4, ctypes.byref(a), ctypes.byref(b)) == INVALID
    assert lib.ws_ring_state(4, 0, ctypes.byref(a), ctypes.byref(b)) == INVALID
    assert lib.ws_ring_state(4, 4, None, ctypes.byref(b)) == INVALID

    w = lib.ws_kv_cache_write_ring
    good = dict(kc=A, vc=B, cap=1024, H=4, d=128, ks=C, vs=D, n=64, Hs=8, hb=2, pos=1000, dt=0)

    def wcall(**kw):
        a = dict(good, **kw)
        return w(P(a["kc"]), P(a["vc"]), a["cap"], a["H"], a["d"], P(a["ks"]), P(a["vs"]), a["n"], a["Hs"], a["hb"], a["pos"],
                 a["dt"], None)

    assert wcall(pos=-1) == RANGE
    assert wcall(n=1025) == RANGE             # more rows than the ring holds
    assert wcall(cap=0) == INVALID
    assert wcall(hb=5) == INVALID
    assert wcall(dt=7) == UNSUPPORTED
    assert wcall(kc=A + 8) == ALIGN
    assert wcall(ks=A + 4096) == OVERLAP
    assert wcall(n=0) == OK                   # nothing launched
    if not torch.cuda.is_available():
        assert wcall() == CUDA                # a valid (wrapping) write reaches CUDA: no CPU fallback

    f = lib.ws_block_causal_attn_ring
    Mask = binding._BlockMask

    def acall(cap=512, start=100, Tc=512, Ln=64, kv=(544, 576), q=B, d=128):
        m = Mask(2, (ctypes.c_int32 * 2)(32, 64), (ctypes.c_int32 * 2)(*kv))
        return f(P(A), None, P(q), P(C), P(D), cap, start, Tc, P(0x50000000), P(0x60000000), Ln, 2, d, 64, ctypes.byref(m), 0.1,
                 P(0x70000000), 1 << 30, 0, None)

    assert acall(start=-1) == RANGE
    assert acall(start=512) == RANGE
    assert acall(Tc=513) == RANGE
    assert acall(kv=(544, 577)) == RANGE
    assert acall(q=B + 8) == ALIGN
    assert acall(d=96) == UNSUPPORTED
    if not torch.cuda.is_available():
        assert acall() == CUDA


def test_ulysses_exchange_entry_points_reject_bad_arguments(lib):
    """every argument error of the peer-memory exchange calls comes back before CUDA is touched."""
    vp = ctypes.c_void_p

    def arr(*ptrs):
        return (vp * len(ptrs))(*ptrs)

    push = lib.ws_ulysses_push_seq_to_head

    def pcall(dsts=(A, B), srcs=(C,), n=1, Ls=16, La=4, H=8, d=64, Pn=2, rank=0, dt=0):
        return push(arr(*dsts), arr(*srcs), n, Ls, La, H, d, Pn, rank, dt, None)

    assert pcall(rank=2) == INVALID
    assert pcall(rank=-1) == INVALID
    assert pcall(H=7) == INVALID                       # H % P != 0
    assert pcall(dsts=(A, 0)) == INVALID               # NULL peer pointer
    assert pcall(dsts=(A, B + 8)) == ALIGN
    assert pcall(dsts=(A, A)) == OVERLAP               # two peers, one buffer
    assert pcall(dsts=(A, C + 256)) == OVERLAP         # a destination inside the source
    assert pcall(Pn=9, H=72, dsts=tuple([A] * 9)) == UNSUPPORTED
    assert pcall(n=5, srcs=tuple([C] * 5), dsts=tuple([A] * 10)) == UNSUPPORTED
    assert pcall(dt=4) == UNSUPPORTED
    assert pcall(n=0) == OK
    assert pcall(Ls=0, La=0) == OK                     # nothing to move, nothing launched

    bw = lib.ws_kv_slice_broadcast_write

    def bcall(kcs=(A, B), vcs=(C, D), Pn=2, cap=256, Hp=2, d=64, ks=0x50000000, vs=0x60000000, n=8, off=10, dt=0):
        return bw(arr(*kcs), arr(*vcs), Pn, cap, Hp, d, vp(ks), vp(vs), n, off, dt, None)

    assert bcall(off=250) == RANGE
    assert bcall(kcs=(A, 0)) == INVALID
    assert bcall(kcs=(A, A)) == OVERLAP                # two ranks sharing one cache
    assert bcall(vcs=(C, A)) == OVERLAP
    assert bcall(ks=A + 1024) == OVERLAP
    assert bcall(kcs=(A, B + 4)) == ALIGN
    assert bcall(Pn=9, kcs=tuple([A] * 9), vcs=tuple([C] * 9)) == UNSUPPORTED
    assert bcall(n=0) == OK

    po = lib.ws_block_causal_attn_push_out
    Mask = binding._BlockMask

    def ocall(outs=(A, B), Pn=2, rank=1, Ls=30, Lq=64, H=2, d=128, q=C, lse=None):
        m = Mask(1, (ctypes.c_int32 * 1)(Lq), (ctypes.c_int32 * 1)(512))
        return po(arr(*outs), Pn, rank, Ls, vp(lse) if lse else None, vp(q), vp(D), vp(0x40000000), 512, 512, None, None, 0, H, d, Lq, ctypes.byref(m), 0.1,
                  vp(0x70000000), 1 << 30, 0, None)

    assert ocall(rank=2) == INVALID
    assert ocall(outs=(A, 0)) == INVALID
    assert ocall(Ls=33) == RANGE                       # P * Ls > Lq
    assert ocall(outs=(A, A + 64)) == OVERLAP
    assert ocall(outs=(A, B + 2)) == ALIGN
    assert ocall(d=96) == UNSUPPORTED
    assert ocall(Pn=9, outs=tuple([A] * 9), Ls=7) == UNSUPPORTED
    # a peer output on top of anything the call reads or uses as scratch (the epilogue would overwrite live data)
    assert ocall(outs=(A, C + 64)) == OVERLAP           # inside q
    assert ocall(outs=(C - 64, B)) == OVERLAP           # its tail reaches into q
    assert ocall(outs=(A, D + 1024)) == OVERLAP         # inside the caches
    assert ocall(outs=(A, 0x70000000 + 4096)) == OVERLAP  # inside the workspace
    assert ocall(outs=(A, B), lse=B + 1024) == OVERLAP  # lse inside a peer output
    if not torch.cuda.is_available():
        assert ocall() == CUDA and pcall() == CUDA and bcall() == CUDA     # valid calls reach CUDA: no CPU fallback


def test_fp8kv_rejects_exponent_arrays_under_the_output_or_the_scratch(lib):
    """The per-row exponents of the FP8 cache are read for the whole launch; an output, LSE or workspace laid over them is refused."""
    f = lib.ws_block_causal_attn_fp8kv
    Mask = binding._BlockMask

    def call(out=A, lse=None, ke=0x50000000, ve=0x58000000, wsp=0x70000000, cap=512):
        m = Mask(1, (ctypes.c_int32 * 1)(64), (ctypes.c_int32 * 1)(512))
        return f(P(out), P(lse) if lse else None, P(B), P(C), P(D), P(ke) if ke else None, P(ve) if ve else None, cap, 512, None, None, 0,
                 2, 128, 64, ctypes.byref(m), 0.1, P(wsp), 1 << 30, None)

    assert call(ke=0) == INVALID
    assert call(ke=0x50000004) == ALIGN
    assert call(cap=520) == ALIGN                      # capacity must be a multiple of 16
    assert call(ke=A + 256) == OVERLAP                 # K exponents inside the output
    assert call(ve=A - 512) == OVERLAP                 # V exponents run into the output
    assert call(ve=0x70000000 + 4096) == OVERLAP       # inside the workspace
    assert call(lse=0x50000000 + 128) == OVERLAP       # LSE over the K exponents
    if not torch.cuda.is_available():
        assert call() == CUDA


def test_unit_forward_host_checks_everything_before_enqueueing(lib):
    """ws_unit_forward_host runs every check of the calls it is made of (cache write, attention) up front, so a call
    that will fail enqueues no copy and forks no helper stream.  On this CPU-only box that is observable: every
    argument error comes back as itself, never as WS_ERR_CUDA from a first CUDA call."""
    f = lib.ws_unit_forward_host
    sb = lib.ws_unit_forward_host_staging_bytes

    def call(out=0x1000, q=0x2000, kn=0x3000, vn=0x4000, Lq=300, Ln=300, steps=2, kc=A, vc=B, cap=4096, ks=0x5000, vs=0x6000, n=100,
             off=500, Tc=600, H=8, d=64, scale=0.125, st=0x70000000, stb=None):
        need = sb(Lq, Ln, H, d, n, Tc + Ln, steps) if (Lq > 0 and steps > 0 and H > 0 and Tc + Ln >= 0 and n >= 0 and Ln >= 0) else 0
        return f(P(out), P(q), P(kn) if kn else None, P(vn) if vn else None, Lq, Ln, steps, P(kc), P(vc), cap, P(ks) if ks else None,
                 P(vs) if vs else None, n, off, Tc, H, d, scale, P(st) if st else None, need if stb is None else stb, None)

    assert call(kc=A + 8) == ALIGN                  # misaligned cache pointer: found by the cache-write / attention checks
    assert call(vc=B + 2) == ALIGN
    assert call(Lq=256 * 256 + 1, Ln=0, kn=0, vn=0) == UNSUPPORTED   # more than 256 Q-tile pairs
    assert call(cap=1 << 24, Tc=(0x7fffffff // 256), n=0, ks=0, vs=0, off=0) == UNSUPPORTED  # beyond the attention kernel's key limit
    assert call(scale=float("nan")) == INVALID
    assert call(scale=-0.5) == INVALID
    assert call(vc=A + 4096) == OVERLAP             # K and V cache ranges intersect
    assert call(kc=0x70000000) == OVERLAP           # staging (where the slice lands) inside the K cache
    assert call(off=4096 - 99) == RANGE
    assert call(Tc=4097) == RANGE
    assert call(d=96) == UNSUPPORTED
    assert call(kn=0) == INVALID
    assert call(ks=0) == INVALID
    assert call(st=0) == WORKSPACE
    assert call(st=0x70000010) == WORKSPACE
    assert call(stb=4096) == WORKSPACE
    assert call(steps=0) == INVALID
    if not torch.cuda.is_available():
        assert call() == CUDA                       # a valid call reaches CUDA and fails there: no CPU fallback


def test_attention_accepts_more_than_65535_work_items(lib):
    """H * ceil(Lq / 256) above 65535 used to overflow the combine kernel's gridDim.y after the attention kernel had
    already run; the item index now sits on gridDim.x.  The schedule for such a problem must build."""
    n_sms = 148
    grid, n_waves = ctypes.c_int32(), ctypes.c_int32()
    iters, tiles = (ctypes.c_int32 * 4)(), (ctypes.c_int32 * 4)()
    pool = (ctypes.c_int64 * (n_sms + 1))()
    Mask = binding._BlockMask
    m = Mask(1, (ctypes.c_int32 * 1)(520), (ctypes.c_int32 * 1)(300))
    H = 40000  # x 3 units = 120000 items
    assert lib.ws_attn_schedule(520, H, 300, 0, ctypes.byref(m), n_sms, ctypes.byref(grid), ctypes.byref(n_waves), iters, tiles, pool) == OK
    assert grid.value == n_sms and n_waves.value == (H * 3) // n_sms


def test_workspace_bytes_is_sane(lib):
    f = lib.ws_block_causal_attn_workspace_bytes
    assert f(0, 1, 128, 10, 0) == 0
    b3 = f(970, 40, 128, 17354, 0)
    assert 20 << 20 < b3 < 200 << 20
    assert f(970, 40, 128, 17354, 1) > b3 + 2 * 40 * 17354 * 128 * 2  # FP32 staging on top
    assert f(3680, 10, 128, 20064, 0) >= f(970, 10, 128, 20064, 0)
    g = lib.ws_unit_forward_host_staging_bytes
    assert g(970, 970, 40, 128, 1024, 17354, 1) > b3 + 3 * 970 * 40 * 128 * 2


def test_binding_refuses_cpu_tensors_no_fallback(lib):
    kc = torch.zeros(2, 8, 64, dtype=torch.bfloat16)
    ks = torch.zeros(4, 2, 64, dtype=torch.bfloat16)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        ws.kv_cache_write(kc, kc.clone(), ks, ks.clone(), 0, 0)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        ws.seq_to_head(torch.zeros(1, 4, 1, 64, dtype=torch.bfloat16), ks, 2, 0, 1)


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", "/nonexistent/libws.so")
    with pytest.raises(RuntimeError, match="no CPU or PyTorch fallback"):
        binding.load()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_04443_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "wsref" not in text and "import oracle" not in text and "from oracle" not in text, fn
    hdr = open(os.path.join(ROOT, "include", "ws.h")).read()
    assert "wsref" not in hdr
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_2607_04443_b200 import" not in text.replace("never imports", "") or fn == "__init__.py"
            assert "ws.h" not in text or "includes nothing from include/" in text
