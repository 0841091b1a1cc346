"""GPU parity of the ring (sliding-window) K/V-cache row (R19) against the CPU oracle
(oracle/wsref_ring.c + wsref.c), through the C ABI.

  * ws_kv_cache_write_ring: whole cache images BIT-EXACT against the oracle, wrapping and non-wrapping slices, a whole
    session of writes;
  * ws_block_causal_attn_ring: against the FP64 oracle attention on the linearised window at north_star's tolerance
    (max-abs 2e-2, rel-Frobenius 1e-2), ring_start unaligned, partially visible windows, spike keys on both sides of the
    wrap seam, FP32, and a config-3-sized streaming session whose window has wrapped;
  * ws_ring_state against the oracle's state rule."""
import math
import zlib

import numpy as np
import pytest
import torch

import paper_2607_04443_b200 as ws
from oracle import wsref, wsref_ring
from paper_2607_04443_b200 import workloads as wl

from gpu_helpers import raw_bytes, to_dev, to_host, workspace_for

pytestmark = pytest.mark.gpu

MAX_ABS, REL_FRO = 2e-2, 1e-2


def rnd(rng, *s):
    return wl.bf16_round(rng.standard_normal(s, dtype=np.float32))


def gpu_ring_attention(q, k_cache, v_cache, ring_start, cache_len, k_new, v_new, qe, kv, scale, dtype="bf16"):
    tq, tkc, tvc = to_dev(q, dtype), to_dev(k_cache, dtype), to_dev(v_cache, dtype)
    tkn = to_dev(k_new, dtype) if k_new is not None and len(k_new) else None
    tvn = to_dev(v_new, dtype) if v_new is not None and len(v_new) else None
    Lq, H, d = q.shape
    Ln = 0 if tkn is None else tkn.shape[0]
    out = torch.full_like(tq, float("nan"))
    lse = torch.full((H, Lq), float("nan"), dtype=torch.float32, device="cuda")
    wsp = workspace_for(Lq, H, d, cache_len + Ln, tq.dtype)
    ws.block_causal_attn_ring(out, tq, tkc, tvc, ring_start, cache_len, tkn, tvn, list(qe), list(kv), scale, wsp, lse=lse)
    torch.cuda.synchronize()
    return to_host(out), lse.cpu().numpy()


def check(got, got_lse, ref, ref_lse, what):
    assert np.all(np.isfinite(got)), what
    ma, rf = wsref.parity_metrics(got, ref)
    assert ma <= MAX_ABS and rf <= REL_FRO, f"{what}: max_abs={ma:.3e} rel_fro={rf:.3e}"
    fin = np.isfinite(ref_lse)
    assert np.array_equal(np.isfinite(got_lse), fin), what
    if fin.any():
        assert np.max(np.abs(got_lse[fin] - ref_lse[fin])) <= 2e-2, what


# ================================================================================================ state
def test_ring_state_matches_oracle():
    for cap in (1, 7, 128, 16384):
        for W in (0, 1, cap - 1, cap, cap + 1, 3 * cap + 5, 10 ** 12 + 17):
            if W < 0:
                continue
            assert ws.ring_state(W, cap) == wsref_ring.ring_state(W, cap)
    with pytest.raises(ws.WsError):
        ws.ring_state(-1, 4)
    with pytest.raises(ws.WsError):
        ws.ring_state(4, 0)


# ================================================================================================ write
@pytest.mark.parametrize("H,cap,d,n,Hs,hb,pos,dtype", [
    (3, 50, 64, 7, 5, 1, 0, "bf16"),          # no wrap
    (3, 50, 64, 7, 5, 1, 46, "bf16"),         # wraps: 4 rows at the end, 3 at the start
    (2, 33, 128, 33, 2, 0, 20, "bf16"),       # a whole lap in one call
    (2, 40, 64, 9, 4, 2, 10 ** 9 + 35, "f32"),  # far into the session, FP32
    (4, 1024, 128, 970, 4, 0, 600, "bf16"),   # a unit's rows wrapping a 1024-row ring
    (1, 16, 8, 0, 1, 0, 5, "f32"),            # nothing to write
])
def test_ring_write_bit_exact_whole_image(H, cap, d, n, Hs, hb, pos, dtype):
    rng = np.random.default_rng(n + cap)
    gen = (lambda *s: rnd(rng, *s)) if dtype == "bf16" else (lambda *s: rng.standard_normal(s, dtype=np.float32))
    k0, v0, ks, vs = gen(H, cap, d), gen(H, cap, d), gen(n, Hs, d), gen(n, Hs, d)
    tk, tv = to_dev(k0, dtype), to_dev(v0, dtype)
    ws.kv_cache_write_ring(tk, tv, to_dev(ks, dtype), to_dev(vs, dtype), hb, pos)
    torch.cuda.synchronize()
    rk, rv = k0.copy(), v0.copy()
    wsref_ring.kv_cache_write_ring(rk, rv, ks, vs, hb, pos)
    assert np.array_equal(raw_bytes(tk), raw_bytes(to_dev(rk, dtype))) and np.array_equal(raw_bytes(tv), raw_bytes(to_dev(rv, dtype)))


def test_ring_write_errors_launch_nothing():
    k = torch.zeros((2, 8, 64), dtype=torch.bfloat16, device="cuda")
    v = torch.zeros_like(k)
    src = torch.ones((9, 2, 64), dtype=torch.bfloat16, device="cuda")
    n0 = ws.kernel_launch_count()
    with pytest.raises(ws.WsError) as e:
        ws.kv_cache_write_ring(k, v, src, src.clone(), 0, 0)        # 9 rows into a ring of 8
    assert e.value.status == -4
    with pytest.raises(ws.WsError) as e:
        ws.kv_cache_write_ring(k, v, src[:4].contiguous(), src[:4].clone(), 0, -1)
    assert e.value.status == -4
    with pytest.raises(ws.WsError) as e:
        ws.kv_cache_write_ring(k, v, src[:4].contiguous(), src[:4].clone(), 1, 0)   # heads [1, 3) of 2
    assert e.value.status == -1
    torch.cuda.synchronize()
    assert ws.kernel_launch_count() == n0 and float(k.abs().sum()) == 0.0


# ================================================================================================ attention
RING_SHAPES = [
    # H, d, blocks, cap, ring_start, cache_len, Ln, visible-as-offsets-from-cache_len
    (2, 128, [200], 640, 0, 640, 200, [200]),            # ring_start 0 == the linear call
    (2, 128, [200], 640, 129, 640, 200, [200]),          # full ring, unaligned start
    (3, 64, [100, 60], 300, 299, 300, 160, [100, 160]),  # run A is a single row
    (2, 128, [130, 126], 512, 384, 512, 256, [130, 256]),  # aligned start: run A exactly one tile
    (2, 128, [256], 1000, 77, 1000, 0, [0]),             # cache only
    (2, 128, [300], 1000, 500, 1000, 300, [-700]),       # the visible prefix ends inside run B... of the window
    (2, 128, [300], 1000, 500, 1000, 300, [-450]),       # ends one row past the wrap seam's tile
    (2, 64, [64, 64, 64], 700, 650, 700, 192, [-690, 0, 192]),  # first block sees 10 rows (all in run A), then all
    (1, 128, [128], 256, 255, 256, 128, [128]),          # smallest wrap: one row, then 255
    (2, 128, [970], 2048, 1500, 2048, 970, [970]),       # unit-sized queries, odd number of Q tiles (single unit)
    (2, 128, [150], 400, 100, 250, 100, [100]),          # ring_start > 0 but the window does not reach the end: no wrap
    (2, 128, [150], 400, 300, 250, 100, [100]),          # wraps without filling the ring: rows 150..299 lie outside the window
]


@pytest.mark.parametrize("case", RING_SHAPES)
def test_ring_attention_whole_tensor(case):
    H, d, blocks, cap, start, clen, Ln, vis_off = case
    rng = np.random.default_rng(zlib.crc32(str(case).encode()))
    qe = np.cumsum(blocks).astype(np.int32)
    kv = np.asarray([clen + o for o in vis_off], np.int32)
    Lq = int(qe[-1])
    q, kc, vc = rnd(rng, Lq, H, d), rnd(rng, H, cap, d), rnd(rng, H, cap, d)
    kn, vn = (rnd(rng, Ln, H, d), rnd(rng, Ln, H, d)) if Ln else (None, None)
    scale = 1.0 / math.sqrt(d)
    got, got_lse = gpu_ring_attention(q, kc, vc, start, clen, kn, vn, qe, kv, scale)
    ref, ref_lse = wsref_ring.block_causal_attn_ring(q, kc, vc, start, clen, kn, vn, qe, kv, scale)
    check(got, got_lse, ref, ref_lse, str(case))


def test_ring_attention_fp32_inputs():
    rng = np.random.default_rng(5)
    H, d, cap, start, Ln = 2, 64, 200, 150, 64
    q, kc, vc = [rng.standard_normal(s, dtype=np.float32) for s in ((64, H, d), (H, cap, d), (H, cap, d))]
    kn, vn = rng.standard_normal((Ln, H, d), dtype=np.float32), rng.standard_normal((Ln, H, d), dtype=np.float32)
    qe, kv = [32, 64], [cap + 32, cap + 64]
    got, got_lse = gpu_ring_attention(q, kc, vc, start, cap, kn, vn, qe, kv, 0.125, dtype="f32")
    ref, ref_lse = wsref_ring.block_causal_attn_ring(q, kc, vc, start, cap, kn, vn, qe, kv, 0.125)
    check(got, got_lse, ref, ref_lse, "fp32 ring")


@pytest.mark.parametrize("cap,start", [(384, 200), (300, 172), (256, 128), (131, 130)])
def test_spike_key_on_both_sides_of_the_wrap_seam(cap, start):
    """A key with logit +40 planted at timeline index vis - 1 must dominate (O ~= its value row); planted at index vis it
    must have no effect.  vis runs over the seam (timeline index cap - start is physical row 0), the tile edges of both
    runs and the ends of the window."""
    rng = np.random.default_rng(cap)
    H, d, Lq = 1, 128, 4
    seam = cap - start
    q = np.zeros((Lq, H, d), np.float32); q[:, 0, 0] = 1.0
    interesting = sorted({1, seam - 1, seam, seam + 1, min(128, cap - 1), min(seam + 128, cap - 1), cap - 1, cap})
    for vis in interesting:
        if not (1 <= vis <= cap):
            continue
        for spike_j, dominated in ((vis - 1, True), (vis, False)):
            if spike_j >= cap:
                continue
            kc, vc = wl.bf16_round(0.01 * rnd(rng, H, cap, d)), rnd(rng, H, cap, d)
            phys = (start + spike_j) % cap
            kc[0, phys, :] = 0.0; kc[0, phys, 0] = 40.0
            vc[0, phys, :] = 7.0
            got, _ = gpu_ring_attention(q, kc, vc, start, cap, None, None, [Lq], [vis], 1.0)
            ref, _ = wsref_ring.block_causal_attn_ring(q, kc, vc, start, cap, None, None, [Lq], [vis], 1.0)
            ma, _ = wsref.parity_metrics(got, ref)
            assert ma <= MAX_ABS, (vis, spike_j, ma)
            if dominated:
                assert np.max(np.abs(got - 7.0)) < 0.05, (vis, spike_j)
            else:
                assert np.max(np.abs(got)) < 6.0, (vis, spike_j)


def test_streaming_session_config3_sized_window_that_has_wrapped():
    """A session at config-3 width (40 heads would take the oracle a minute; 6 heads here): units of 970 rows are
    written into a 4096-row ring until it has wrapped twice, then the unit's 970 queries attend to the window plus their
    own K/V.  The cache image is compared bit for bit after every write, attention whole-tensor at the end."""
    rng = np.random.default_rng(33)
    H, d, cap, unit = 6, 128, 4096, 970
    k = np.zeros((H, cap, d), np.float32); v = np.zeros((H, cap, d), np.float32)
    tk, tv = to_dev(k, "bf16"), to_dev(v, "bf16")
    W = 0
    for _ in range(10):                                   # 9700 rows: the ring wraps twice
        ks, vs = rnd(rng, unit, H, d), rnd(rng, unit, H, d)
        ws.kv_cache_write_ring(tk, tv, to_dev(ks, "bf16"), to_dev(vs, "bf16"), 0, W)
        wsref_ring.kv_cache_write_ring(k, v, ks, vs, 0, W)
        W += unit
        assert np.array_equal(to_host(tk), k) and np.array_equal(to_host(tv), v)
    start, clen = ws.ring_state(W, cap)
    assert (start, clen) == (W % cap, cap) and start % 128 != 0
    q, kn, vn = rnd(rng, unit, H, d), rnd(rng, unit, H, d), rnd(rng, unit, H, d)
    Lq = unit
    out = torch.full((Lq, H, d), float("nan"), dtype=torch.bfloat16, device="cuda")
    lse = torch.empty((H, Lq), dtype=torch.float32, device="cuda")
    wsp = workspace_for(Lq, H, d, clen + unit)
    ws.block_causal_attn_ring(out, to_dev(q, "bf16"), tk, tv, start, clen, to_dev(kn, "bf16"), to_dev(vn, "bf16"), [Lq], [clen + unit],
                              1.0 / math.sqrt(d), wsp, lse=lse)
    torch.cuda.synchronize()
    ref, ref_lse = wsref_ring.block_causal_attn_ring(q, k, v, start, clen, kn, vn, [Lq], [clen + unit], 1.0 / math.sqrt(d))
    check(to_host(out), lse.cpu().numpy(), ref, ref_lse, "session")


def test_config3_full_size_on_a_wrapped_ring_whole_tensor():
    """BASELINE.json config 3 at full size (970 queries x 40 heads, 16384 cached rows + the unit's own 970), the cache held as a
    16384-row ring whose window starts at an unaligned row: whole [Lq, H, d] tensor and LSE against the FP64 oracle on the
    linearised window -- the launch configuration bench.py times in aux.ring_and_ulysses.ring_cfg3."""
    cfg = wl.CONFIGS["cfg3"]
    x = wl.generate(cfg)
    kc, vc = x["k_cache"].copy(), x["v_cache"].copy()
    wsref.kv_cache_write(kc, vc, x["k_slice"], x["v_slice"], 0, cfg.write_offset)          # the linear timeline: 16384 valid rows
    cap = cfg.cache_len
    start = ws.ring_state(23 * 970, cap)[0]
    assert start % 128 != 0
    ring_k = np.ascontiguousarray(np.roll(kc[:, :cap], start, axis=1))                      # timeline row j sits at (start + j) % cap
    ring_v = np.ascontiguousarray(np.roll(vc[:, :cap], start, axis=1))
    q, kn, vn = x["q"][0], x["k_new"][0], x["v_new"][0]
    got, got_lse = gpu_ring_attention(q, ring_k, ring_v, start, cap, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale)
    ref, ref_lse = wsref.block_causal_attn(q, kc, vc, cap, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale)
    check(got, got_lse, ref, ref_lse, "cfg3 on a ring")
    # and the ring oracle agrees with the linear one on this window (the roll above is the inverse of its linearisation)
    assert np.array_equal(wsref_ring.linearise(ring_k, start, cap), kc[:, :cap])


def test_ring_attention_errors_launch_nothing():
    H, d, cap = 2, 128, 256
    q = torch.zeros((16, H, d), dtype=torch.bfloat16, device="cuda")
    kc = torch.zeros((H, cap, d), dtype=torch.bfloat16, device="cuda")
    out = torch.full_like(q, 3.0)
    wsp = workspace_for(16, H, d, cap)
    n0 = ws.kernel_launch_count()
    for start in (-1, cap, cap + 5):
        with pytest.raises(ws.WsError) as e:
            ws.block_causal_attn_ring(out, q, kc, kc.clone(), start, cap, None, None, [16], [cap], 1.0, wsp)
        assert e.value.status == -4
    torch.cuda.synchronize()
    assert ws.kernel_launch_count() == n0 and float((out - 3.0).abs().sum()) == 0.0
