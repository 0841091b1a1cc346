"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Bit-exact for the cache write and the relayouts; max-abs <= 2e-2 AND
rel-Frobenius <= 1e-2 for attention (north_star; BF16 in, FP32 accumulate).  Off-by-one errors in
the mask / seam / tile tails are pinned by config 1 and the spike-key tests."""
import math

import numpy as np
import pytest
import torch

import paper_2607_04443_b200 as ws
from oracle import wsref
from paper_2607_04443_b200 import workloads as wl

from gpu_helpers import gpu_attention, raw_bytes, to_dev, to_host, workspace_for

pytestmark = pytest.mark.gpu

MAX_ABS, REL_FRO = 2e-2, 1e-2


def check_attn(got, ref, got_lse=None, ref_lse=None, max_abs=MAX_ABS, rel_fro=REL_FRO, what=""):
    assert np.all(np.isfinite(got)), f"{what}: non-finite output"
    ma, rf = wsref.parity_metrics(got, ref)
    assert ma <= max_abs and rf <= rel_fro, f"{what}: max_abs={ma:.3e} rel_fro={rf:.3e}"
    if got_lse is not None:
        fin = np.isfinite(ref_lse)
        assert np.array_equal(np.isfinite(got_lse), fin), f"{what}: lse finiteness"
        assert np.all(np.isneginf(got_lse[~fin]))
        if fin.any():
            assert np.max(np.abs(got_lse[fin] - ref_lse[fin])) <= 2e-2, f"{what}: lse"
    return ma, rf


def rand_case(seed, H, d, blocks, vis, Tc, Ln, cap=None, q_mul=1.0):
    rng = np.random.default_rng(seed)
    cap = cap or max(Tc, 1)
    qe = np.cumsum(blocks).astype(np.int32)
    Lq = int(qe[-1])
    r = lambda *s: wl.bf16_round(rng.standard_normal(s, dtype=np.float32))
    return dict(q=wl.bf16_round(r(Lq, H, d) * np.float32(q_mul)), k_cache=r(H, cap, d), v_cache=r(H, cap, d), cache_len=Tc,
                k_new=r(Ln, H, d) if Ln else None, v_new=r(Ln, H, d) if Ln else None, q_block_end=qe,
                kv_visible=np.asarray(vis, np.int32), scale=1.0 / math.sqrt(d))


def both(c, dtype="bf16"):
    got, got_lse = gpu_attention(c["q"], c["k_cache"], c["v_cache"], c["cache_len"], c["k_new"], c["v_new"], c["q_block_end"],
                                 c["kv_visible"], c["scale"], dtype)
    ref, ref_lse = wsref.block_causal_attn(c["q"], c["k_cache"], c["v_cache"], c["cache_len"], c["k_new"], c["v_new"],
                                           c["q_block_end"], c["kv_visible"], c["scale"])
    return got, got_lse, ref, ref_lse


# ================================================================================================
# a1: KV cache write -- bit-exact, whole buffers, sentinel outside
# ================================================================================================
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg5_small"])
def test_cache_write_bit_exact(name):
    cfg = wl.CONFIGS[name]
    x = wl.generate(cfg)
    dt = cfg.dtype
    kc, vc = to_dev(x["k_cache"], dt), to_dev(x["v_cache"], dt)
    ws.kv_cache_write(kc, vc, to_dev(x["k_slice"], dt), to_dev(x["v_slice"], dt), 0, cfg.write_offset)
    torch.cuda.synchronize()
    rk, rv = wl.device_array(x["k_cache"], dt), wl.device_array(x["v_cache"], dt)
    wsref.kv_cache_write(rk, rv, wl.device_array(x["k_slice"], dt), wl.device_array(x["v_slice"], dt), 0, cfg.write_offset)
    assert np.array_equal(raw_bytes(kc), rk.view(np.uint8).reshape(-1))
    assert np.array_equal(raw_bytes(vc), rv.view(np.uint8).reshape(-1))


@pytest.mark.parametrize("H,cap,d,n,Hs,hb,off,dtype", [
    (3, 1000, 128, 257, 7, 2, 700, torch.bfloat16),   # head sub-range of a wider slice, ragged rows
    (5, 64, 64, 1, 5, 0, 63, torch.bfloat16),         # one row, last slot
    (2, 300, 64, 300, 2, 0, 0, torch.float32),        # whole cache, FP32
    (1, 17, 8, 5, 3, 1, 9, torch.bfloat16),           # 16-byte rows (dv = 1)
])
def test_cache_write_shapes_and_untouched_regions(H, cap, d, n, Hs, hb, off, dtype):
    g = torch.Generator().manual_seed(n)
    np_dt = np.uint16 if dtype == torch.bfloat16 else np.uint32
    bits = lambda *s: torch.randint(0, 2 ** 15, s, generator=g, dtype=torch.int32).numpy().astype(np_dt)
    kc, vc, ks, vs = bits(H, cap, d), bits(H, cap, d), bits(n, Hs, d), bits(n, Hs, d)
    t = lambda a: torch.from_numpy(a.view(np.int16 if np_dt == np.uint16 else np.int32)).cuda().view(dtype)
    tk, tv = t(kc), t(vc)
    ws.kv_cache_write(tk, tv, t(ks), t(vs), hb, off)
    torch.cuda.synchronize()
    wsref.kv_cache_write(kc, vc, ks, vs, hb, off)
    assert np.array_equal(raw_bytes(tk), kc.view(np.uint8).reshape(-1))
    assert np.array_equal(raw_bytes(tv), vc.view(np.uint8).reshape(-1))


# ================================================================================================
# a2 / a4: relayouts -- bit-exact, round trip, other heads untouched
# ================================================================================================
@pytest.mark.parametrize("n_tok,H,d,P,g0,G,dtype", [
    (3680, 40, 128, 4, 0, 1, "bf16"), (3680, 40, 128, 4, 1, 1, "bf16"), (3680, 40, 128, 4, 2, 1, "bf16"),
    (3680, 40, 128, 4, 3, 1, "bf16"),                       # config 4, every rank
    (920, 40, 128, 4, 0, 4, "bf16"),                        # true rank-local pack, G = P
    (333, 6, 64, 1, 0, 1, "bf16"), (77, 8, 64, 2, 1, 1, "f32"), (1, 4, 8, 4, 3, 1, "bf16"), (1000, 12, 128, 3, 1, 2, "bf16"),
])
def test_relayouts_bit_exact_and_round_trip(n_tok, H, d, P, g0, G, dtype):
    Hp = H // P
    np_dt = np.uint16 if dtype == "bf16" else np.uint32
    th = torch.bfloat16 if dtype == "bf16" else torch.float32
    src = (np.arange(n_tok * H * d, dtype=np.uint64) * 2654435761 % 65521).astype(np_dt).reshape(n_tok, H, d)
    t = lambda a: torch.from_numpy(a.view(np.int16 if np_dt == np.uint16 else np.int32)).cuda().view(th)
    dst = np.full((G, n_tok, Hp, d), 0x7BCD, np_dt)
    tdst = t(dst)
    ws.seq_to_head(tdst, t(src), P, g0, G)
    wsref.seq_to_head(dst, src, P, g0, G)
    assert np.array_equal(raw_bytes(tdst), dst.view(np.uint8).reshape(-1))
    back = np.full((n_tok, H, d), 0x7EEE, np_dt)
    tback = t(back)
    ws.head_to_seq(tback, tdst, P, g0, G)
    wsref.head_to_seq(back, dst, P, g0, G)
    assert np.array_equal(raw_bytes(tback), back.view(np.uint8).reshape(-1))
    sel = np.zeros(H, bool)
    sel[g0 * Hp:(g0 + G) * Hp] = True
    got = tback.view(torch.int16 if np_dt == np.uint16 else torch.int32).cpu().numpy().view(np_dt)
    assert np.array_equal(got[:, sel], src[:, sel]) and np.all(got[:, ~sel] == 0x7EEE)


def test_multi_tensor_relayouts_equal_single_calls():
    """ws_seq_to_head_multi / ws_head_to_seq_multi: three tensors in one launch == three single calls == oracle."""
    n_tok, H, d, P, g0, G = 970, 40, 128, 4, 1, 2
    rng = np.random.default_rng(21)
    srcs_np = [wl.bf16_round(rng.standard_normal((n_tok, H, d), dtype=np.float32)) for _ in range(3)]
    srcs = [to_dev(a, "bf16") for a in srcs_np]
    one = [torch.full((G, n_tok, H // P, d), 7.0, dtype=torch.bfloat16, device="cuda") for _ in range(3)]
    many = [torch.full_like(o, 9.0) for o in one]
    for o, a in zip(one, srcs):
        ws.seq_to_head(o, a, P, g0, G)
    ws.seq_to_head_multi(many, srcs, P, g0, G)
    torch.cuda.synchronize()
    for o, m, a in zip(one, many, srcs_np):
        assert np.array_equal(raw_bytes(o), raw_bytes(m))
        ref = np.empty((G, n_tok, H // P, d), np.float32)
        wsref.seq_to_head(ref, a, P, g0, G)
        assert np.array_equal(to_host(m), ref)
    back_one = [torch.full((n_tok, H, d), 3.0, dtype=torch.bfloat16, device="cuda") for _ in range(3)]
    back_many = [torch.full_like(b, 3.0) for b in back_one]
    for b, m in zip(back_one, many):
        ws.head_to_seq(b, m, P, g0, G)
    ws.head_to_seq_multi(back_many, many, P, g0, G)
    torch.cuda.synchronize()
    for b, m in zip(back_one, back_many):
        assert np.array_equal(raw_bytes(b), raw_bytes(m))
    # errors: too many tensors, overlapping destinations -- nothing is written
    with pytest.raises(ws.WsError) as e:
        ws.seq_to_head_multi(many + many[:2], srcs + srcs[:2], P, g0, G)
    assert e.value.status == -2
    before = raw_bytes(many[0]).copy()
    with pytest.raises(ws.WsError) as e:
        ws.seq_to_head_multi([many[0], many[0]], srcs[:2], P, g0, G)
    assert e.value.status == -5
    torch.cuda.synchronize()
    assert np.array_equal(raw_bytes(many[0]), before)


# ================================================================================================
# a3: attention -- BASELINE.json configs (1-4 and step 0 of 5 whole at full size; steps 1-7 of 5 sampled; reduced copies whole)
# ================================================================================================
def run_config(cfg, x, step=0):
    """cache write (if any) + relayout (if any) + attention through the library; returns device tensors."""
    dt = cfg.dtype
    kc, vc = to_dev(x["k_cache"], dt), to_dev(x["v_cache"], dt)
    if cfg.write_rows:
        ws.kv_cache_write(kc, vc, to_dev(x["k_slice"], dt), to_dev(x["v_slice"], dt), 0, cfg.write_offset)
    q, kn, vn = to_dev(x["q"][step], dt), None, None
    if cfg.Ln:
        kn, vn = to_dev(x["k_new"][step], dt), to_dev(x["v_new"][step], dt)
    if cfg.P > 1:
        def relay(t):
            o = torch.empty((cfg.G, t.shape[0], cfg.H, cfg.d), dtype=t.dtype, device="cuda")
            ws.seq_to_head(o, t, cfg.P, cfg.g0, cfg.G)
            return o[0]
        q, kn, vn = relay(q), relay(kn), relay(vn)
    out = torch.full_like(q, float("nan"))
    lse = torch.full((cfg.H, cfg.Lq), float("nan"), dtype=torch.float32, device="cuda")
    wsp = workspace_for(cfg.Lq, cfg.H, cfg.d, cfg.cache_len + cfg.Ln, q.dtype)
    ws.block_causal_attn(out, q, kc, vc, cfg.cache_len, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale, wsp, lse=lse)
    torch.cuda.synchronize()
    return out, lse, kc, vc


def oracle_inputs(cfg, x, step=0):
    kc, vc = x["k_cache"].copy(), x["v_cache"].copy()
    if cfg.write_rows:
        wsref.kv_cache_write(kc, vc, x["k_slice"], x["v_slice"], 0, cfg.write_offset)
    q = x["q"][step]
    kn = x["k_new"][step] if cfg.Ln else None
    vn = x["v_new"][step] if cfg.Ln else None
    if cfg.P > 1:
        def relay(a):
            o = np.empty((cfg.G, a.shape[0], cfg.H, cfg.d), np.float32)
            wsref.seq_to_head(o, a, cfg.P, cfg.g0, cfg.G)
            return o[0]
        q, kn, vn = relay(q), relay(kn), relay(vn)
    return q, kc, vc, kn, vn


@pytest.mark.parametrize("name", ["cfg1", "cfg1_split", "cfg2_small", "cfg3_small", "cfg4_small", "cfg5_small"])
def test_config_whole_tensor_parity(name):
    cfg = wl.CONFIGS[name]
    x = wl.generate(cfg)
    for step in range(cfg.steps):
        out, lse, _, _ = run_config(cfg, x, step)
        q, kc, vc, kn, vn = oracle_inputs(cfg, x, step)
        ref, ref_lse = wsref.block_causal_attn(q, kc, vc, cfg.cache_len, kn, vn, cfg.q_block_end, cfg.kv_visible,
                                               cfg.softmax_scale)
        check_attn(to_host(out), ref, lse.cpu().numpy(), ref_lse, what=f"{name} step {step}")


@pytest.mark.parametrize("name,g0", [("cfg4_small", 0), ("cfg4_small", 3), ("cfg4", 1)])
def test_relayouts_fused_into_attention(name, g0):
    """ws_block_causal_attn_seq_layout (a2 + a3 + a4 in one call) on the token-major [L, H_total, d] tensors:
    bit-identical to seq->head x3 + attention + head->seq through the library, heads of other ranks untouched,
    and within tolerance of the oracle's composition of the same three definitions."""
    cfg = wl.CONFIGS[name]
    x = wl.generate(cfg)
    dt = cfg.dtype
    P, Hp, H_total = cfg.P, cfg.H, cfg.H * cfg.P
    kc, vc = to_dev(x["k_cache"], dt), to_dev(x["v_cache"], dt)
    q, kn, vn = to_dev(x["q"][0], dt), to_dev(x["k_new"][0], dt), to_dev(x["v_new"][0], dt)
    assert tuple(q.shape) == (cfg.Lq, H_total, cfg.d)
    wsp = workspace_for(cfg.Lq, Hp, cfg.d, cfg.cache_len + cfg.Ln, q.dtype)
    # unfused: three packs, attention, unpack into a sentinel-filled token-major tensor
    def relay(t):
        o = torch.empty((1, t.shape[0], Hp, cfg.d), dtype=t.dtype, device="cuda")
        ws.seq_to_head(o, t, P, g0, 1)
        return o[0]
    out_h = torch.empty((cfg.Lq, Hp, cfg.d), dtype=q.dtype, device="cuda")
    lse_a = torch.empty((Hp, cfg.Lq), dtype=torch.float32, device="cuda")
    ws.block_causal_attn(out_h, relay(q), kc, vc, cfg.cache_len, relay(kn), relay(vn), cfg.q_block_end, cfg.kv_visible,
                         cfg.softmax_scale, wsp, lse=lse_a)
    sentinel = 1.0 / 64.0
    out_a = torch.full_like(q, sentinel)
    ws.head_to_seq(out_a, out_h[None], P, g0, 1)
    # fused
    out_b = torch.full_like(q, sentinel)
    lse_b = torch.empty_like(lse_a)
    ws.block_causal_attn_seq_layout(out_b, q, kc, vc, cfg.cache_len, kn, vn, g0 * Hp, cfg.q_block_end, cfg.kv_visible,
                                    cfg.softmax_scale, wsp, lse=lse_b)
    torch.cuda.synchronize()
    assert np.array_equal(raw_bytes(out_a), raw_bytes(out_b)), "fused and unfused paths must agree bit for bit"
    assert torch.equal(lse_a, lse_b)
    got = to_host(out_b)
    others = np.ones(H_total, bool)
    others[g0 * Hp:(g0 + 1) * Hp] = False
    assert np.all(got[:, others] == sentinel), "heads of other ranks must not be touched"
    # oracle: definitions composed (relayout -> attention), sampled rows at full size
    def relay_ref(a):
        o = np.empty((1, a.shape[0], Hp, cfg.d), np.float32)
        wsref.seq_to_head(o, a, P, g0, 1)
        return o[0]
    rq, rkn, rvn = relay_ref(x["q"][0]), relay_ref(x["k_new"][0]), relay_ref(x["v_new"][0])
    mine = got[:, g0 * Hp:(g0 + 1) * Hp]
    if name.endswith("_small"):
        ref, ref_lse = wsref.block_causal_attn(rq, x["k_cache"], x["v_cache"], cfg.cache_len, rkn, rvn, cfg.q_block_end,
                                               cfg.kv_visible, cfg.softmax_scale)
        check_attn(mine, ref, lse_b.cpu().numpy(), ref_lse, what=f"{name} fused g0={g0}")
    else:
        rows, heads = wl.sample_pairs(cfg, 256)
        ref, ref_lse = wsref.block_causal_attn_rows(rq, x["k_cache"], x["v_cache"], cfg.cache_len, rkn, rvn, cfg.q_block_end,
                                                    cfg.kv_visible, cfg.softmax_scale, rows, heads)
        check_attn(mine[rows, heads], ref, lse_b.cpu().numpy()[heads, rows], ref_lse, what=f"{name} fused g0={g0} (sampled)")


def test_config1_also_in_bf16():
    cfg = wl.CONFIGS["cfg1_split"]
    x = wl.generate(cfg)
    c = dict(q=wl.bf16_round(x["q"][0]), k_cache=wl.bf16_round(x["k_cache"]), v_cache=wl.bf16_round(x["v_cache"]),
             cache_len=cfg.cache_len, k_new=wl.bf16_round(x["k_new"][0]), v_new=wl.bf16_round(x["v_new"][0]),
             q_block_end=cfg.q_block_end, kv_visible=cfg.kv_visible, scale=cfg.softmax_scale)
    got, got_lse, ref, ref_lse = both(c)
    check_attn(got, ref, got_lse, ref_lse, what="cfg1 bf16")


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4"])
def test_config_full_size_whole_tensor_parity(name):
    """BASELINE.json's full sizes in the launch configuration bench.py times, compared with the oracle over the
    WHOLE [Lq, H, d] output and the whole LSE (full comparison of configs 2-4)."""
    cfg = wl.CONFIGS[name]
    x = wl.generate(cfg)
    out, lse, kc, vc = run_config(cfg, x, 0)
    q, rkc, rvc, kn, vn = oracle_inputs(cfg, x, 0)
    if cfg.write_rows:  # the cache image itself, bit-exact at full size
        assert np.array_equal(raw_bytes(kc), wl.device_array(rkc, cfg.dtype).view(np.uint8).reshape(-1))
        assert np.array_equal(raw_bytes(vc), wl.device_array(rvc, cfg.dtype).view(np.uint8).reshape(-1))
    ref, ref_lse = wsref.block_causal_attn(q, rkc, rvc, cfg.cache_len, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale)
    check_attn(to_host(out), ref, lse.cpu().numpy(), ref_lse, what=f"{name} (whole tensor)")
    # per head as well: one wrong work item (one head x 256 rows) must not hide inside the whole-tensor norm
    got = to_host(out)
    for h in range(cfg.H):
        check_attn(got[:, h], ref[:, h], what=f"{name} head {h}")


def test_config5_full_size_eager_and_graph():
    """Config 5 at full size (65536-row cache, 8 denoising steps): step 0 against the oracle over the whole tensor,
    steps 1-7 on a sample of (row, head) outputs the oracle computes one by one; then the unit as
    bench.py times it -- cache write + 8 attention calls under ONE CUDA graph -- replayed and compared the same way."""
    cfg = wl.CONFIGS["cfg5"]
    x = wl.generate(cfg)
    dt = cfg.dtype
    q0, rkc, rvc, kn0, vn0 = oracle_inputs(cfg, x, 0)
    ref0, ref0_lse = wsref.block_causal_attn(q0, rkc, rvc, cfg.cache_len, kn0, vn0, cfg.q_block_end, cfg.kv_visible,
                                             cfg.softmax_scale)
    rows, heads = wl.sample_pairs(cfg, 256)
    samples = {0: None}
    for s in range(1, cfg.steps):
        samples[s] = wsref.block_causal_attn_rows(x["q"][s], rkc, rvc, cfg.cache_len, x["k_new"][s], x["v_new"][s], cfg.q_block_end,
                                                  cfg.kv_visible, cfg.softmax_scale, rows, heads)

    def compare(outs, lses, what):
        check_attn(to_host(outs[0]), ref0, None if lses is None else lses[0].cpu().numpy(), ref0_lse, what=f"cfg5 {what} step 0 (whole)")
        got0 = to_host(outs[0])
        for h in range(cfg.H):
            check_attn(got0[:, h], ref0[:, h], what=f"cfg5 {what} step 0 head {h}")
        for s in range(1, cfg.steps):
            got = to_host(outs[s])
            assert np.all(np.isfinite(got)) and np.abs(got).max() <= 4.0, "whole output must be written and inside the value range"
            check_attn(got[rows, heads], samples[s][0], None if lses is None else lses[s].cpu().numpy()[heads, rows], samples[s][1],
                       what=f"cfg5 {what} step {s} (sampled)")

    # ---- eager ----
    kc, vc = to_dev(x["k_cache"], dt), to_dev(x["v_cache"], dt)
    ks, vs = to_dev(x["k_slice"], dt), to_dev(x["v_slice"], dt)
    qs = [to_dev(a, dt) for a in x["q"]]
    kns = [to_dev(a, dt) for a in x["k_new"]]
    vns = [to_dev(a, dt) for a in x["v_new"]]
    outs = [torch.full_like(q, float("nan")) for q in qs]
    lses = [torch.full((cfg.H, cfg.Lq), float("nan"), dtype=torch.float32, device="cuda") for _ in qs]
    wsp = workspace_for(cfg.Lq, cfg.H, cfg.d, cfg.cache_len + cfg.Ln)
    ws.kv_cache_write(kc, vc, ks, vs, 0, cfg.write_offset)
    for s in range(cfg.steps):
        ws.block_causal_attn(outs[s], qs[s], kc, vc, cfg.cache_len, kns[s], vns[s], cfg.q_block_end, cfg.kv_visible,
                             cfg.softmax_scale, wsp, lse=lses[s])
    torch.cuda.synchronize()
    assert np.array_equal(raw_bytes(kc), wl.device_array(rkc, dt).view(np.uint8).reshape(-1)), "cache image, bit-exact at full size"
    compare(outs, lses, "eager")
    # ---- the same unit under one CUDA graph (what bench.py's cfg5_unit_graph times) ----
    kc2, vc2 = to_dev(x["k_cache"], dt), to_dev(x["v_cache"], dt)
    stream = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(graph, stream=stream):
        ws.kv_cache_write(kc2, vc2, ks, vs, 0, cfg.write_offset)
        for s in range(cfg.steps):
            ws.block_causal_attn(outs[s], qs[s], kc2, vc2, cfg.cache_len, kns[s], vns[s], cfg.q_block_end, cfg.kv_visible,
                                 cfg.softmax_scale, wsp)
    for o in outs:
        o.fill_(float("nan"))
    graph.replay()
    graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(raw_bytes(vc2), wl.device_array(rvc, dt).view(np.uint8).reshape(-1))
    compare(outs, None, "graph")


# ================================================================================================
# closed forms, boundaries and degenerate cases on the GPU
# ================================================================================================
SHAPES = [
    # seed, H, d, blocks, kv_visible, Tc, Ln
    (1, 2, 128, [128], [128], 128, 0),                     # exactly one tile
    (2, 2, 128, [100], [300], 200, 100),                   # ragged everything
    (3, 3, 64, [64, 64], [160, 192], 128, 64),             # d = 64, config-1 structure
    (4, 1, 128, [130, 127, 259], [1, 129, 777], 500, 277),  # tile-straddling blocks, 1 visible key, partial cache tile
    (5, 2, 128, [300], [520], 0, 520),                     # no cache at all
    (6, 2, 128, [257], [1000], 1000, 0),                   # no new rows, Q tail of one row
    (7, 1, 128, [50, 50], [0, 64], 64, 0),                 # first block sees nothing
    (8, 5, 64, [700], [2500], 1900, 600),                  # d = 64 multi-tile with split-KV
    (9, 1, 128, [512], [40000], 39500, 500),               # long KV, few Q tiles: deep split-KV + combine
    # more (head, Q-pair) work items than SMs: whole-item waves first, stream-K only on the remainder
    (10, 40, 128, [1100], [400], 300, 100),                # 200 equal items: one wave + a 52-item pool
    (11, 160, 64, [256, 300], [0, 450], 200, 250),         # 480 items, three waves; every pair 0 sees no key at all
    (12, 30, 128, [256] * 6, [300, 600, 900, 1200, 1500, 1800], 1500, 300),  # 180 items of very unequal length
    (13, 2, 128, [100, 100], [128, 256], 256, 50),         # own K/V rows passed but never visible; limits on tile multiples
    (14, 3, 64, [1], [1], 1, 0),                           # one query, one key
]


@pytest.mark.parametrize("case", SHAPES)
def test_random_shapes_whole_tensor(case):
    c = rand_case(*case)
    got, got_lse, ref, ref_lse = both(c)
    check_attn(got, ref, got_lse, ref_lse, what=str(case))


def test_peaked_logits_exercise_running_max_and_rescale():
    """Q x 4 (logit sigma ~4): O(1) outputs, the running max moves across tiles, lazy rescale fires."""
    c = rand_case(11, 2, 128, [300], [3000], 2500, 500, q_mul=4.0)
    got, got_lse, ref, ref_lse = both(c)
    check_attn(got, ref, got_lse, ref_lse, what="peaked")
    # increasing key norm along the timeline forces the max to grow by > 2^8 between tiles
    c = rand_case(12, 1, 128, [200], [1500], 1500, 0)
    c["k_cache"] = wl.bf16_round(c["k_cache"] * np.linspace(0.05, 6.0, c["k_cache"].shape[1], dtype=np.float32)[None, :, None])
    got, got_lse, ref, ref_lse = both(c)
    check_attn(got, ref, got_lse, ref_lse, what="growing max")


def test_unit_values_give_ones_and_equal_keys_give_mean():
    c = rand_case(13, 2, 128, [150, 150], [400, 900], 600, 300)
    ones = dict(c, v_cache=np.ones_like(c["v_cache"]), v_new=np.ones_like(c["v_new"]))
    got, _ = gpu_attention(ones["q"], ones["k_cache"], ones["v_cache"], 600, ones["k_new"], ones["v_new"], c["q_block_end"],
                           c["kv_visible"], c["scale"])
    assert np.max(np.abs(got - 1.0)) <= 1e-2      # softmax rows sum to 1 (BF16 P rounding only)
    eq = dict(c, k_cache=np.full_like(c["k_cache"], 0.25), k_new=np.full_like(c["k_new"], 0.25))
    got, _ = gpu_attention(eq["q"], eq["k_cache"], eq["v_cache"], 600, eq["k_new"], eq["v_new"], c["q_block_end"],
                           c["kv_visible"], c["scale"])
    V = np.concatenate([c["v_cache"][:, :600], np.transpose(c["v_new"], (1, 0, 2))], axis=1).astype(np.float64)
    for rows, n in ((slice(0, 150), 400), (slice(150, 300), 900)):
        want = V[:, :n].mean(axis=1)  # [H, d]
        assert np.max(np.abs(got[rows] - want[None])) <= 2e-3, "mean of exactly the visible value rows"


@pytest.mark.parametrize("Tc,Ln", [(300, 200), (256, 128), (130, 126)])
def test_spike_key_at_every_boundary(Tc, Ln):
    """+40-logit key at kv_visible[b]-1 dominates block b; at kv_visible[b] it must not be seen.
    Also at the cache/new seam and either side of every 128-key tile edge."""
    H, d = 1, 128
    blocks = [96, 64, 140]
    vis = [Tc - 45, Tc + 1, Tc + Ln]
    base = rand_case(14, H, d, blocks, vis, Tc, Ln)
    base["q"] = np.ones_like(base["q"])
    scale = base["scale"]

    def run(j=None):
        c = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in base.items()}
        if j is not None:
            big = np.full(d, wl.bf16_round(np.float32(40.0 / (d * scale))), np.float32)
            val = np.full(d, 100.0, np.float32)
            if j < Tc:
                c["k_cache"][0, j], c["v_cache"][0, j] = big, val
            else:
                c["k_new"][j - Tc, 0], c["v_new"][j - Tc, 0] = big, val
        return gpu_attention(c["q"], c["k_cache"], c["v_cache"], Tc, c["k_new"], c["v_new"], c["q_block_end"],
                             c["kv_visible"], scale)[0]

    ref = run()
    edges = np.cumsum([0] + blocks)
    probes = set()
    for n in vis:
        probes.update([n - 1, n])
    probes.update([Tc - 1, Tc, 127, 128, 255, 256])
    for j in sorted(p for p in probes if 0 <= p < Tc + Ln):
        got = run(j)
        for b, n in enumerate(vis):
            rows = slice(edges[b], edges[b + 1])
            if j < n:
                assert np.all(np.abs(got[rows] - 100.0) < 0.5), f"key {j} must dominate block {b}"
            else:
                assert np.array_equal(got[rows], ref[rows]), f"key {j} must be invisible to block {b}"


def test_stale_cache_rows_beyond_cache_len_are_never_read():
    c = rand_case(15, 2, 128, [200], [100 + 64], 100, 64, cap=512)
    got, _, ref, _ = both(c)
    poisoned = dict(c, k_cache=c["k_cache"].copy(), v_cache=c["v_cache"].copy())
    poisoned["k_cache"][:, 100:] = np.nan
    poisoned["v_cache"][:, 100:] = np.inf
    got2, _ = gpu_attention(poisoned["q"], poisoned["k_cache"], poisoned["v_cache"], 100, c["k_new"], c["v_new"],
                            c["q_block_end"], c["kv_visible"], c["scale"])
    assert np.array_equal(got, got2)
    check_attn(got, ref, what="stale rows")


def test_scale_zero_is_uniform_and_lse_is_log_n():
    c = rand_case(16, 1, 64, [10], [333], 333, 0)
    got, lse = gpu_attention(c["q"], c["k_cache"], c["v_cache"], 333, None, None, c["q_block_end"], c["kv_visible"], 0.0)
    want = c["v_cache"][:, :333].astype(np.float64).mean(axis=1)
    assert np.max(np.abs(got - want[None])) <= 2e-3
    assert np.max(np.abs(lse - math.log(333))) <= 1e-3


# ================================================================================================
# errors on the GPU box, CUDA-graph capture, end-to-end host entry
# ================================================================================================
def test_errors_leave_outputs_untouched():
    q = torch.zeros(64, 2, 128, dtype=torch.bfloat16, device="cuda")
    kc = torch.zeros(2, 256, 128, dtype=torch.bfloat16, device="cuda")
    out = torch.full_like(q, 7.0)
    wsp = workspace_for(64, 2, 128, 256)
    with pytest.raises(ws.WsError) as e:
        ws.block_causal_attn(out, q, kc, kc.clone(), 256, None, None, [64], [257], 0.1, wsp)
    assert e.value.status == -4
    with pytest.raises(ws.WsError) as e:
        ws.block_causal_attn(out, q, kc, kc.clone(), 256, None, None, [64], [256], 0.1, wsp[:1024])
    assert e.value.status == -6
    with pytest.raises(ws.WsError) as e:
        ws.kv_cache_write(kc, kc.clone(), q, q.clone(), 0, 200)
    assert e.value.status == -4
    torch.cuda.synchronize()
    assert torch.all(out == 7.0) and torch.all(kc == 0)


def test_cuda_graph_capture_of_the_unit_loop():
    """config-5 structure (reduced): cache write + N attention steps captured once, replayed."""
    cfg = wl.CONFIGS["cfg5_small"]
    x = wl.generate(cfg)
    dt = cfg.dtype
    kc, vc = to_dev(x["k_cache"], dt), to_dev(x["v_cache"], dt)
    ks, vs = to_dev(x["k_slice"], dt), to_dev(x["v_slice"], dt)
    qs = [to_dev(a, dt) for a in x["q"]]
    kns = [to_dev(a, dt) for a in x["k_new"]]
    vns = [to_dev(a, dt) for a in x["v_new"]]
    outs = [torch.zeros_like(q) for q in qs]
    wsp = workspace_for(cfg.Lq, cfg.H, cfg.d, cfg.cache_len + cfg.Ln)
    stream = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.graph(graph, stream=stream):
        ws.kv_cache_write(kc, vc, ks, vs, 0, cfg.write_offset)
        for s in range(cfg.steps):
            ws.block_causal_attn(outs[s], qs[s], kc, vc, cfg.cache_len, kns[s], vns[s], cfg.q_block_end, cfg.kv_visible,
                                 cfg.softmax_scale, wsp)
    for o in outs:
        o.fill_(float("nan"))
    graph.replay()
    graph.replay()
    torch.cuda.synchronize()
    for s in range(cfg.steps):
        q, rkc, rvc, kn, vn = oracle_inputs(cfg, x, s)
        ref, _ = wsref.block_causal_attn(q, rkc, rvc, cfg.cache_len, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale)
        check_attn(to_host(outs[s]), ref, what=f"graph step {s}")


def test_unit_forward_host_matches_oracle():
    cfg = wl.CONFIGS["cfg5_small"]
    x = wl.generate(cfg)
    host = lambda a: torch.from_numpy(wl.bf16_bits(a).view(np.int16)).view(torch.bfloat16).pin_memory()
    kc, vc = to_dev(x["k_cache"], "bf16"), to_dev(x["v_cache"], "bf16")
    qh = host(np.stack(x["q"]))
    knh, vnh = host(np.stack(x["k_new"])), host(np.stack(x["v_new"]))
    outh = torch.zeros_like(qh).pin_memory()
    nbytes = ws.unit_forward_host_staging_bytes(cfg.Lq, cfg.Ln, cfg.H, cfg.d, cfg.write_rows, cfg.cache_len + cfg.Ln, cfg.steps)
    staging = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ws.unit_forward_host(outh, qh, knh, vnh, kc, vc, host(x["k_slice"]), host(x["v_slice"]), cfg.write_offset, cfg.cache_len,
                         cfg.softmax_scale, staging)
    torch.cuda.synchronize()
    got = wl.bf16_from_bits(outh.view(torch.int16).numpy().view(np.uint16))
    for s in range(cfg.steps):
        q, rkc, rvc, kn, vn = oracle_inputs(cfg, x, s)
        ref, _ = wsref.block_causal_attn(q, rkc, rvc, cfg.cache_len, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale)
        check_attn(got[s], ref, what=f"host entry step {s}")


def test_unit_forward_host_two_steps_and_reuse_of_the_helper_streams():
    """ws_unit_forward_host with d = 64, two steps, called twice: contiguous copies on the internal streams, cache write,
    attention against the cache and against the unit's own rows merged by LSE; cache and every step's output against the oracle."""
    rng = np.random.default_rng(31)
    H, d, Lq, Tc0, n_w, cap, steps = 8, 64, 300, 500, 100, 700, 2
    r = lambda *s: wl.bf16_round(rng.standard_normal(s, dtype=np.float32))
    k_cache, v_cache = np.zeros((H, cap, d), np.float32), np.zeros((H, cap, d), np.float32)
    k_cache[:, :Tc0], v_cache[:, :Tc0] = r(H, Tc0, d), r(H, Tc0, d)
    k_slice, v_slice = r(n_w, H, d), r(n_w, H, d)
    q, kn, vn = r(steps, Lq, H, d), r(steps, Lq, H, d), r(steps, Lq, H, d)
    Tc, scale = Tc0 + n_w, 1.0 / math.sqrt(d)
    host = lambda a: torch.from_numpy(wl.bf16_bits(a).view(np.int16)).view(torch.bfloat16).pin_memory()
    kc, vc = to_dev(k_cache, "bf16"), to_dev(v_cache, "bf16")
    outh = torch.zeros((steps, Lq, H, d), dtype=torch.bfloat16).pin_memory()
    staging = torch.empty(ws.unit_forward_host_staging_bytes(Lq, Lq, H, d, n_w, Tc + Lq, steps), dtype=torch.uint8, device="cuda")
    for _ in range(2):  # twice: the helper streams and events are reused across calls
        ws.unit_forward_host(outh, host(q), host(kn), host(vn), kc, vc, host(k_slice), host(v_slice), Tc0, Tc, scale, staging)
        torch.cuda.synchronize()
    rk, rv = k_cache.copy(), v_cache.copy()
    wsref.kv_cache_write(rk, rv, k_slice, v_slice, 0, Tc0)
    assert np.array_equal(to_host(kc), rk) and np.array_equal(to_host(vc), rv)
    got = wl.bf16_from_bits(outh.view(torch.int16).numpy().view(np.uint16))
    for s in range(steps):
        ref, _ = wsref.block_causal_attn(q[s], rk, rv, Tc, kn[s], vn[s], [Lq], [Tc + Lq], scale)
        check_attn(got[s], ref, what=f"pipelined host entry step {s}")


def test_unit_forward_host_is_as_accurate_as_the_single_pass_call():
    """ws_unit_forward_host splits the keys by source (cache | the unit's own rows) and merges the two attentions by LSE.  The
    partial results stay FP32 until the merge, so its output carries ONE rounding to BF16, like ws_block_causal_attn's: its
    error against the oracle may not exceed the single-pass call's by more than a tenth, and the two GPU results agree far
    inside the oracle tolerance (they differ by FP32 summation order and by which running maximum P was rounded against)."""
    rng = np.random.default_rng(41)
    H, d, Lq, Tc, cap = 6, 128, 300, 640, 640
    r = lambda *s: wl.bf16_round(rng.standard_normal(s, dtype=np.float32))
    k_cache, v_cache, q, kn, vn = r(H, cap, d), r(H, cap, d), r(1, Lq, H, d), r(1, Lq, H, d), r(1, Lq, H, d)
    scale = 1.0 / math.sqrt(d)
    host = lambda a: torch.from_numpy(wl.bf16_bits(a).view(np.int16)).view(torch.bfloat16).pin_memory()
    kc, vc = to_dev(k_cache, "bf16"), to_dev(v_cache, "bf16")
    outh = torch.zeros((1, Lq, H, d), dtype=torch.bfloat16).pin_memory()
    staging = torch.empty(ws.unit_forward_host_staging_bytes(Lq, Lq, H, d, 0, Tc + Lq, 1), dtype=torch.uint8, device="cuda")
    ws.unit_forward_host(outh, host(q), host(kn), host(vn), kc, vc, None, None, 0, Tc, scale, staging)
    torch.cuda.synchronize()
    got_host = wl.bf16_from_bits(outh.view(torch.int16).numpy().view(np.uint16))[0]
    got_single, _ = gpu_attention(q[0], k_cache, v_cache, Tc, kn[0], vn[0], [Lq], [Tc + Lq], scale, want_lse=False)
    ref, _ = wsref.block_causal_attn(q[0], k_cache, v_cache, Tc, kn[0], vn[0], [Lq], [Tc + Lq], scale)
    _, rf_host = wsref.parity_metrics(got_host, ref)
    _, rf_single = wsref.parity_metrics(got_single, ref)
    ma_pair, rf_pair = wsref.parity_metrics(got_host, got_single.astype(np.float64))
    assert rf_host <= 1.1 * rf_single + 2e-4, (rf_host, rf_single)
    assert rf_pair <= 4e-3 and ma_pair <= 4e-3, (ma_pair, rf_pair)


def test_fused_relayout_attention_in_fp32():
    """Config-1 arithmetic (FP32 in, rounded to BF16 on the device, FP32 out) through the token-major call:
    the staging cast gathers the rank's heads token by token."""
    rng = np.random.default_rng(32)
    H_total, Hp, d, Lq, Tc, g0 = 4, 2, 64, 64, 128, 1
    r = lambda *s: rng.standard_normal(s, dtype=np.float32)
    q, kn, vn = r(Lq, H_total, d), r(Lq, H_total, d), r(Lq, H_total, d)
    k_cache, v_cache = r(Hp, Tc, d), r(Hp, Tc, d)
    qe, kv, scale = [32, 64], [Tc + 32, Tc + 64], 1.0 / math.sqrt(d)
    tq, tkn, tvn = to_dev(q, "f32"), to_dev(kn, "f32"), to_dev(vn, "f32")
    tkc, tvc = to_dev(k_cache, "f32"), to_dev(v_cache, "f32")
    wsp = workspace_for(Lq, Hp, d, Tc + Lq, torch.float32)
    out = torch.full_like(tq, 5.0)
    lse = torch.empty((Hp, Lq), dtype=torch.float32, device="cuda")
    ws.block_causal_attn_seq_layout(out, tq, tkc, tvc, Tc, tkn, tvn, g0 * Hp, qe, kv, scale, wsp, lse=lse)
    torch.cuda.synchronize()
    got = to_host(out)
    sel = slice(g0 * Hp, (g0 + 1) * Hp)
    ref, ref_lse = wsref.block_causal_attn(np.ascontiguousarray(q[:, sel]), k_cache, v_cache, Tc, np.ascontiguousarray(kn[:, sel]),
                                           np.ascontiguousarray(vn[:, sel]), qe, kv, scale)
    check_attn(got[:, sel], ref, lse.cpu().numpy(), ref_lse, what="fused fp32")
    assert np.all(got[:, :g0 * Hp] == 5.0), "heads of other ranks must not be touched"


def test_per_device_state_survives_device_round_trips():
    """The SM count and the kernels' shared-memory attribute are kept per device (ws.h conventions): the library is
    called on every visible device in turn, twice, each time after a cudaSetDevice; on a one-GPU box this walks the
    per-device table path for device 0 after set_device round trips."""
    c = rand_case(41, 3, 128, [300], [700], 500, 200)
    ref, _ = wsref.block_causal_attn(c["q"], c["k_cache"], c["v_cache"], c["cache_len"], c["k_new"], c["v_new"], c["q_block_end"],
                                     c["kv_visible"], c["scale"])
    n_dev = torch.cuda.device_count()
    try:
        for _ in range(2):
            for dev in range(n_dev):
                torch.cuda.set_device(dev)
                got, _ = gpu_attention(c["q"], c["k_cache"], c["v_cache"], c["cache_len"], c["k_new"], c["v_new"], c["q_block_end"],
                                       c["kv_visible"], c["scale"])
                check_attn(got, ref, what=f"device {dev}")
    finally:
        torch.cuda.set_device(0)


@pytest.mark.parametrize("Tc0,n_w,Ln", [(0, 0, 200), (300, 0, 0), (0, 0, 0), (100, 28, 77)])
def test_unit_forward_host_degenerate_key_sources(Tc0, n_w, Ln):
    """No cache at all (only the unit's own rows), no own rows (only the cache), no key whatsoever (zeros), and a ragged
    mix: the single-source cases skip the merge."""
    rng = np.random.default_rng(33)
    H, d, Lq, cap = 3, 128, 150, 512
    r = lambda *s: wl.bf16_round(rng.standard_normal(s, dtype=np.float32))
    k_cache, v_cache = np.zeros((H, cap, d), np.float32), np.zeros((H, cap, d), np.float32)
    k_cache[:, :Tc0], v_cache[:, :Tc0] = r(H, Tc0, d), r(H, Tc0, d)
    q = r(1, Lq, H, d)
    kn, vn = (r(1, Ln, H, d), r(1, Ln, H, d)) if Ln else (None, None)
    ks, vs = (r(n_w, H, d), r(n_w, H, d)) if n_w else (None, None)
    Tc, scale = Tc0 + n_w, 1.0 / math.sqrt(d)
    host = lambda a: None if a is None else torch.from_numpy(wl.bf16_bits(a).view(np.int16)).view(torch.bfloat16).pin_memory()
    kc, vc = to_dev(k_cache, "bf16"), to_dev(v_cache, "bf16")
    outh = torch.full((1, Lq, H, d), 9.0, dtype=torch.bfloat16).pin_memory()
    staging = torch.empty(ws.unit_forward_host_staging_bytes(Lq, Ln, H, d, n_w, Tc + Ln, 1), dtype=torch.uint8, device="cuda")
    ws.unit_forward_host(outh, host(q), host(kn), host(vn), kc, vc, host(ks), host(vs), Tc0, Tc, scale, staging)
    torch.cuda.synchronize()
    rk, rv = k_cache.copy(), v_cache.copy()
    if n_w:
        wsref.kv_cache_write(rk, rv, ks, vs, 0, Tc0)
    got = wl.bf16_from_bits(outh.view(torch.int16).numpy().view(np.uint16))[0]
    ref, _ = wsref.block_causal_attn(q[0], rk, rv, Tc, None if kn is None else kn[0], None if vn is None else vn[0], [Lq], [Tc + Ln], scale)
    check_attn(got, ref, what=f"host entry Tc0={Tc0} n_w={n_w} Ln={Ln}")
    if Tc + Ln == 0:
        assert np.all(got == 0.0)


# ================================================================================================
# split work items: partial records, combine kernel, scratch workspace
# ================================================================================================
def attention_with_workspace_fill(c, fill):
    """The plain call, with the workspace pre-filled by `fill(workspace)` (its contents are scratch by contract)."""
    tq, tkc, tvc = to_dev(c["q"], "bf16"), to_dev(c["k_cache"], "bf16"), to_dev(c["v_cache"], "bf16")
    tkn = to_dev(c["k_new"], "bf16") if c["k_new"] is not None else None
    tvn = to_dev(c["v_new"], "bf16") if c["v_new"] is not None else None
    Lq, H, d = c["q"].shape
    Ln = 0 if tkn is None else tkn.shape[0]
    out = torch.full_like(tq, float("nan"))
    lse = torch.full((H, Lq), float("nan"), dtype=torch.float32, device="cuda")
    wsp = workspace_for(Lq, H, d, c["cache_len"] + Ln)
    fill(wsp)
    ws.block_causal_attn(out, tq, tkc, tvc, c["cache_len"], tkn, tvn, list(c["q_block_end"]), list(c["kv_visible"]), c["scale"], wsp, lse=lse)
    torch.cuda.synchronize()
    return to_host(out), lse.cpu().numpy()


@pytest.mark.parametrize("Lq,H,Tc", [(268, 79, 300), (893, 40, 300), (369, 79, 1000)])
def test_split_item_whose_cta_span_contains_an_empty_cta(Lq, H, Tc):
    """Shapes for which (on 148 SMs) the cost-aware partition leaves a CTA without pool work INSIDE the CTA span of a split
    item: that CTA writes no partial record, and the merge must not read one.  The workspace is filled with NaN bytes so a
    stale read cannot pass by luck."""
    c = rand_case(Lq + H, H, 128, [Lq], [Tc], Tc, 0)
    got, got_lse = attention_with_workspace_fill(c, lambda w: w.fill_(0xFF))
    ref, ref_lse = wsref.block_causal_attn(c["q"], c["k_cache"], c["v_cache"], Tc, None, None, c["q_block_end"], c["kv_visible"], c["scale"])
    check_attn(got, ref, got_lse, ref_lse, what=f"Lq={Lq} H={H} Tc={Tc}")


@pytest.mark.parametrize("fill", ["zeros", "ones", "random"])
def test_workspace_contents_are_scratch(fill):
    """The split-KV partial records live in the caller's workspace, whose contents are scratch: it may hold anything."""
    c = rand_case(77, 24, 128, [292], [2048 + 292], 2048, 292)          # config-2-like: every item is split over several CTAs
    fills = {"zeros": lambda w: w.zero_(), "ones": lambda w: w.fill_(0xFF),
             "random": lambda w: w.copy_(torch.randint(0, 256, w.shape, dtype=torch.uint8, device="cuda"))}
    got, got_lse = attention_with_workspace_fill(c, fills[fill])
    ref, ref_lse = wsref.block_causal_attn(c["q"], c["k_cache"], c["v_cache"], 2048, c["k_new"], c["v_new"], c["q_block_end"],
                                           c["kv_visible"], c["scale"])
    check_attn(got, ref, got_lse, ref_lse, what=fill)


def test_graph_replays_of_a_split_item_shape():
    """Two calls that share one workspace inside one CUDA graph, replayed with fresh queries: every replay must stand on its
    own (no state survives in the workspace from one call or replay to the next)."""
    c = rand_case(78, 10, 128, [700], [1500 + 700], 1500, 700)
    tq, tkc, tvc = to_dev(c["q"], "bf16"), to_dev(c["k_cache"], "bf16"), to_dev(c["v_cache"], "bf16")
    tkn, tvn = to_dev(c["k_new"], "bf16"), to_dev(c["v_new"], "bf16")
    out = torch.empty_like(tq)
    wsp = workspace_for(700, 10, 128, 2200)
    args = (tkc, tvc, 1500, tkn, tvn, [700], [2200], c["scale"], wsp)
    ws.block_causal_attn(out, tq, *args)
    torch.cuda.synchronize()
    st, cg = torch.cuda.Stream(), torch.cuda.CUDAGraph()
    with torch.cuda.graph(cg, stream=st):
        ws.block_causal_attn(out, tq, *args)
        ws.block_causal_attn(out, tq, *args)      # two calls in one graph share the workspace
    rng = np.random.default_rng(5)
    for rep in range(4):
        q = wl.bf16_round(rng.standard_normal(c["q"].shape, dtype=np.float32))
        tq.copy_(to_dev(q, "bf16"))
        out.fill_(float("nan"))
        cg.replay()
        torch.cuda.synchronize()
        ref, _ = wsref.block_causal_attn(q, c["k_cache"], c["v_cache"], 1500, c["k_new"], c["v_new"], [700], [2200], c["scale"])
        check_attn(to_host(out), ref, what=f"replay {rep}")
