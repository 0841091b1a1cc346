"""GPU parity of the FP8 K/V-cache row against the CPU oracle (oracle/wsref_fp8.c + wsref.c).

  * ws_kv_cache_write_fp8: codes and exponents BIT-EXACT against the oracle's quantiser, whole buffers, untouched regions;
  * ws_block_causal_attn_fp8kv: the codes are expanded to BF16 exactly, so the reference is the FP64 oracle attention on
    the DEQUANTISED cache, at north_star's tolerance (max-abs 2e-2, rel-Frobenius 1e-2); the expansion itself is checked
    exactly for all 256 codes (a query that sees one key returns that key's value row);
  * the quantisation error against the BF16 cache is reported and bounded separately (it is a property of the format)."""
import math

import numpy as np
import pytest
import torch

import paper_2607_04443_b200 as ws
from oracle import wsref, wsref_fp8
from paper_2607_04443_b200 import workloads as wl

from gpu_helpers import to_dev, to_host, workspace_for

pytestmark = pytest.mark.gpu

MAX_ABS, REL_FRO = 2e-2, 1e-2


def dev_u8(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_write(k_src, v_src, H, cap, hb, off, fill=(0xAB, 0xCD, 55, -66)):
    d = k_src.shape[2]
    kc8 = torch.full((H, cap, d), fill[0], dtype=torch.uint8, device="cuda")
    vc8 = torch.full((H, cap, d), fill[1], dtype=torch.uint8, device="cuda")
    ke = torch.full((H, cap), fill[2], dtype=torch.int8, device="cuda")
    ve = torch.full((H, cap), fill[3], dtype=torch.int8, device="cuda")
    ws.kv_cache_write_fp8(kc8, vc8, ke, ve, to_dev(k_src, "bf16"), to_dev(v_src, "bf16"), hb, off)
    torch.cuda.synchronize()
    return kc8, vc8, ke, ve


def ref_write(k_src, v_src, H, cap, hb, off, fill=(0xAB, 0xCD, 55, -66)):
    d = k_src.shape[2]
    kc8, vc8 = np.full((H, cap, d), fill[0], np.uint8), np.full((H, cap, d), fill[1], np.uint8)
    ke, ve = np.full((H, cap), fill[2], np.int8), np.full((H, cap), fill[3], np.int8)
    wsref_fp8.kv_cache_write_fp8(kc8, vc8, ke, ve, k_src, v_src, hb, off)
    return kc8, vc8, ke, ve


def test_fp8_cache_nan_source_is_contained_and_not_propagated():
    """ws.h: FP8-cache sources must be finite.  What a NaN does is pinned here so that it cannot change unnoticed: the NaN
    element is stored as the E4M3 NaN code (0x7f / 0xff), every OTHER (row, head) group is bit-exact as if the NaN were
    not there, and ws_block_causal_attn_fp8kv does NOT hand the NaN on -- it reads the NaN code as a finite number (the
    BF16 cache would return NaN rows).  Only the poisoned group's own exponent and codes are unspecified."""
    n, H, d, cap = 64, 3, 128, 128
    rng = np.random.default_rng(77)
    k = wl.bf16_round(rng.standard_normal((n, H, d), dtype=np.float32))
    v = wl.bf16_round(rng.standard_normal((n, H, d), dtype=np.float32))
    tk, tv = to_dev(k, "bf16"), to_dev(v, "bf16")
    tk[10, 1, 5] = float("nan")
    tv[20, 2, 9] = float("nan")
    kc8, vc8 = (torch.full((H, cap, d), 0xAB, dtype=torch.uint8, device="cuda") for _ in range(2))
    ke, ve = (torch.full((H, cap), 55, dtype=torch.int8, device="cuda") for _ in range(2))
    ws.kv_cache_write_fp8(kc8, vc8, ke, ve, tk, tv, 0, 0)
    torch.cuda.synchronize()
    want = ref_write(k, v, H, cap, 0, 0, fill=(0xAB, 0xAB, 55, 55))   # the oracle on the finite rows
    for got, ref, (r, h, c) in ((kc8, want[0], (10, 1, 5)), (vc8, want[1], (20, 2, 9))):
        g = got.cpu().numpy()
        assert g[h, r, c] & 0x7f == 0x7f                     # the E4M3 NaN pattern
        g[h, r, :] = ref[h, r, :]
        assert np.array_equal(g, ref)                        # no other group is disturbed
    for got, ref, (r, h) in ((ke, want[2], (10, 1)), (ve, want[3], (20, 2))):
        g = got.cpu().numpy()
        g[h, r] = ref[h, r]
        assert np.array_equal(g, ref)
    q = to_dev(wl.bf16_round(rng.standard_normal((40, H, d), dtype=np.float32)), "bf16")
    out = torch.full_like(q, float("nan"))
    ws.block_causal_attn_fp8kv(out, q, kc8, vc8, ke, ve, n, None, None, [40], [n], d ** -0.5, workspace_for(40, H, d, n))
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out.float()).all())           # the documented hazard: a NaN in the source is silently finite here


@pytest.mark.parametrize("n,Hs,d,H,cap,hb,off,spread", [
    (1024, 40, 128, 40, 2048, 0, 512, 0),     # cfg3's slice shape
    (257, 7, 128, 3, 1008, 2, 700, 3),        # head sub-range of a wider slice, ragged rows, rows of very different magnitude
    (300, 2, 64, 2, 304, 0, 0, 5),            # d = 64, (almost) the whole cache
    (1, 5, 64, 5, 64, 0, 63, 0),              # one row, last slot
])
def test_fp8_cache_write_bit_exact(n, Hs, d, H, cap, hb, off, spread):
    rng = np.random.default_rng(n + d)
    mag = np.float32(10.0) ** rng.uniform(-spread, spread, (n, Hs, 1)).astype(np.float32)
    k = wl.bf16_round(rng.standard_normal((n, Hs, d), dtype=np.float32) * mag)
    v = wl.bf16_round(rng.standard_normal((n, Hs, d), dtype=np.float32) * mag[::-1])
    if n > 5:
        k[3] = 0.0                                   # all-zero rows: exponent -100, codes 0
        v[4, :, : d // 2] = 0.0
        k[5, :, 0] = wl.bf16_round(np.float32(3e38))  # beyond 448 * 2^7: the exponent clamps and the codes saturate
        v[5, :, 1] = -448.0 * 128                    # exactly the largest representable magnitude
        k[2, :, 3] = np.float32(2.0 ** -130)         # BF16 subnormal
    got = gpu_write(k, v, H, cap, hb, off)
    want = ref_write(k, v, H, cap, hb, off)
    for g, w, name in zip(got, want, ("k codes", "v codes", "k exponents", "v exponents")):
        assert np.array_equal(g.cpu().numpy(), w), name


def test_fp8_expansion_is_exact_for_all_256_codes():
    """A query block that sees ONE key returns that key's value row: P = 1 exactly, so O = decode(code) * 2^e rounded
    to BF16, which must be the oracle's dequantised value bit for bit -- for every code (NaN codes excepted), several
    exponents (incl. both clamps), and both through a whole-unit CTA and the K side (a huge key must win the softmax)."""
    d, H = 128, 8
    codes = np.array([c for c in range(256) if c not in (0x7F, 0xFF)], np.uint8)
    exps = [-100, -9, -8, 0, 3, 7, -50, 1]
    vc8 = np.zeros((H, 16, d), np.uint8)
    ve = np.zeros((H, 16), np.int8)
    rng = np.random.default_rng(7)
    for h in range(H):
        row = rng.permutation(np.resize(codes, d * 2))[:d]
        vc8[h, 0] = row
        ve[h, 0] = exps[h]
    vc8[:, 0, :4] = np.array([0x00, 0x80, 0x01, 0x7E], np.uint8)   # +0, -0, smallest subnormal, 448
    kc8 = np.full((H, 16, d), 0x38, np.uint8)                      # code 0x38 = 1.0
    ke = np.zeros((H, 16), np.int8)
    want = wsref_fp8.kv_cache_dequant_fp8(vc8, ve, 1)[:, 0]        # [H, d]
    q = torch.ones((5, H, d), dtype=torch.bfloat16, device="cuda")
    out = torch.full_like(q, float("nan"))
    wsp = workspace_for(5, H, d, 16)
    ws.block_causal_attn_fp8kv(out, q, dev_u8(kc8), dev_u8(vc8), dev_u8(ke), dev_u8(ve), 16, None, None, [5], [1], 0.01, wsp)
    torch.cuda.synchronize()
    got = to_host(out)
    for r in range(5):
        assert np.array_equal(got[r], want), "dequantised value rows must come back bit for bit"
    # K side: key 3 of every head is 448 * 2^e in every element, the others are tiny: with all-ones queries it takes all the weight
    kc8[:, :, :] = 0x08
    kc8[:, 3, :] = 0x7E
    ke[:, :] = -6
    for h in range(H):
        ke[h, 3] = [-3, -2, -1, 0, 1, 2, 3, 4][h]
    vc8[:, :, :] = 0x38
    vc8[:, 3, :] = 0x40                                            # 2.0
    ve[:, :] = 0
    ws.block_causal_attn_fp8kv(out, q, dev_u8(kc8), dev_u8(vc8), dev_u8(ke), dev_u8(ve), 16, None, None, [5], [16], 1.0, wsp)
    torch.cuda.synchronize()
    assert np.all(to_host(out) == 2.0)


def fp8_case(seed, H, d, blocks, vis, Tc, Ln, cap, q_mul=1.0, kv_mag_spread=0.0):
    rng = np.random.default_rng(seed)
    qe = np.cumsum(blocks).astype(np.int32)
    Lq = int(qe[-1])
    r = lambda *s: wl.bf16_round(rng.standard_normal(s, dtype=np.float32))
    # rows of very different magnitude exercise the per-row exponents; V stays below ~2 so that BF16 rounding of the
    # OUTPUT (half an ulp is 2^-8 of the value's binade) stays inside north_star's absolute tolerance
    kmag = np.float32(4.0) ** rng.uniform(-kv_mag_spread, 0.5 * kv_mag_spread, (max(Tc, 1), H, 1)).astype(np.float32)
    vmag = np.float32(4.0) ** rng.uniform(-2 * kv_mag_spread, -0.5, (max(Tc, 1), H, 1)).astype(np.float32)
    return dict(q=wl.bf16_round(r(Lq, H, d) * np.float32(q_mul)), k_rows=wl.bf16_round(r(max(Tc, 1), H, d) * kmag),
                v_rows=wl.bf16_round(r(max(Tc, 1), H, d) * vmag), cache_len=Tc, cap=cap,
                k_new=r(Ln, H, d) if Ln else None, v_new=r(Ln, H, d) if Ln else None, q_block_end=qe,
                kv_visible=np.asarray(vis, np.int32), scale=1.0 / math.sqrt(d))


def run_fp8(c, want_bf16_reference=False):
    """-> (gpu out, gpu lse, oracle out on the dequantised cache, oracle lse[, oracle out on the unquantised rows])."""
    H, d, Tc, cap = c["q"].shape[1], c["q"].shape[2], c["cache_len"], c["cap"]
    kc8, vc8, ke, ve = gpu_write(c["k_rows"][:Tc], c["v_rows"][:Tc], H, cap, 0, 0, fill=(0x7F, 0xFF, 120, -120)) if Tc else \
        tuple(torch.zeros(s, dtype=t, device="cuda") for s, t in (((H, cap, d), torch.uint8),) * 2 + (((H, cap), torch.int8),) * 2)
    if Tc:
        w = ref_write(c["k_rows"][:Tc], c["v_rows"][:Tc], H, cap, 0, 0, fill=(0x7F, 0xFF, 120, -120))
        for g, ww in zip((kc8, vc8, ke, ve), w):
            assert np.array_equal(g.cpu().numpy(), ww), "cache image (codes, exponents), bit-exact"
        kd, vd = wsref_fp8.kv_cache_dequant_fp8(w[0], w[2], Tc), wsref_fp8.kv_cache_dequant_fp8(w[1], w[3], Tc)
    else:
        kd = vd = np.zeros((H, cap, d), np.float32)
    q = to_dev(c["q"], "bf16")
    kn = to_dev(c["k_new"], "bf16") if c["k_new"] is not None else None
    vn = to_dev(c["v_new"], "bf16") if c["v_new"] is not None else None
    Lq, Ln = q.shape[0], 0 if kn is None else kn.shape[0]
    out = torch.full_like(q, float("nan"))
    lse = torch.full((H, Lq), float("nan"), dtype=torch.float32, device="cuda")
    wsp = workspace_for(Lq, H, d, Tc + Ln)
    ws.block_causal_attn_fp8kv(out, q, kc8, vc8, ke, ve, Tc, kn, vn, list(c["q_block_end"]), list(c["kv_visible"]), c["scale"], wsp, lse=lse)
    torch.cuda.synchronize()
    ref, ref_lse = wsref.block_causal_attn(c["q"], kd, vd, Tc, c["k_new"], c["v_new"], c["q_block_end"], c["kv_visible"], c["scale"])
    res = [to_host(out), lse.cpu().numpy(), ref, ref_lse]
    if want_bf16_reference:
        kb, vb = np.zeros((H, cap, d), np.float32), np.zeros((H, cap, d), np.float32)
        kb[:, :Tc], vb[:, :Tc] = np.transpose(c["k_rows"][:Tc], (1, 0, 2)), np.transpose(c["v_rows"][:Tc], (1, 0, 2))
        res.append(wsref.block_causal_attn(c["q"], kb, vb, Tc, c["k_new"], c["v_new"], c["q_block_end"], c["kv_visible"], c["scale"])[0])
    return res


def check(got, got_lse, ref, ref_lse, what):
    assert np.all(np.isfinite(got)), f"{what}: non-finite output"
    ma, rf = wsref.parity_metrics(got, ref)
    assert ma <= MAX_ABS and rf <= REL_FRO, f"{what}: max_abs={ma:.3e} rel_fro={rf:.3e}"
    fin = np.isfinite(ref_lse)
    assert np.array_equal(np.isfinite(got_lse), fin) and np.all(np.isneginf(got_lse[~fin]))
    if fin.any():
        assert np.max(np.abs(got_lse[fin] - ref_lse[fin])) <= 2e-2, f"{what}: lse"


FP8_SHAPES = [
    # seed, H, d, blocks, kv_visible, Tc, Ln, cap
    (1, 2, 128, [128], [128], 128, 0, 128),                       # exactly one cache tile
    (2, 2, 128, [100], [300], 200, 100, 208),                     # ragged everything; single unit, cache + own rows
    (3, 3, 64, [64, 64], [160, 192], 128, 64, 256),               # d = 64, config-1 structure
    (4, 1, 128, [130, 127, 259], [1, 129, 777], 500, 277, 512),   # tile-straddling blocks, partial cache tile
    (5, 2, 128, [300], [520], 0, 520, 16),                        # no cache at all
    (6, 2, 128, [257], [1000], 1000, 0, 1008),                    # no new rows; a pair and a single unit
    (7, 5, 64, [700], [2500], 1900, 600, 1904),                   # d = 64 multi-tile with split-KV
    (8, 1, 128, [512], [40000], 39500, 500, 39504),               # long KV, few Q tiles: deep split-KV + combine
    (9, 40, 128, [1100], [400], 300, 100, 304),                   # more units than SMs: whole-item waves + pool
    (10, 3, 128, [100, 100], [128, 256], 256, 50, 256),           # own rows passed but never visible
]


@pytest.mark.parametrize("case", FP8_SHAPES)
def test_fp8_attention_matches_oracle_on_dequantised_cache(case):
    c = fp8_case(*case, kv_mag_spread=1.5)
    got, got_lse, ref, ref_lse = run_fp8(c)
    check(got, got_lse, ref, ref_lse, str(case))


@pytest.mark.parametrize("name", ["cfg2", "cfg3"])
def test_fp8_attention_full_size_configs(name):
    """BASELINE.json configs 2 and 3 with the cache held in FP8: whole-tensor parity against the oracle on the dequantised
    cache, and the error the format itself introduces against the BF16 cache (reported; bounded loosely)."""
    cfg = wl.CONFIGS[name]
    x = wl.generate(cfg)
    kc, vc = x["k_cache"].copy(), x["v_cache"].copy()
    if cfg.write_rows:
        wsref.kv_cache_write(kc, vc, x["k_slice"], x["v_slice"], 0, cfg.write_offset)
    Tc = cfg.cache_len
    c = dict(q=x["q"][0], k_rows=np.ascontiguousarray(np.transpose(kc[:, :Tc], (1, 0, 2))),
             v_rows=np.ascontiguousarray(np.transpose(vc[:, :Tc], (1, 0, 2))), cache_len=Tc, cap=cfg.capacity, k_new=x["k_new"][0],
             v_new=x["v_new"][0], q_block_end=np.asarray(cfg.q_block_end, np.int32), kv_visible=np.asarray(cfg.kv_visible, np.int32),
             scale=cfg.softmax_scale)
    got, got_lse, ref, ref_lse, ref_bf16 = run_fp8(c, want_bf16_reference=True)
    check(got, got_lse, ref, ref_lse, f"{name} fp8 cache (whole tensor)")
    for h in range(cfg.H):
        ma, rf = wsref.parity_metrics(got[:, h], ref[:, h])
        assert ma <= MAX_ABS and rf <= REL_FRO, f"{name} head {h}"
    _, q_err = wsref.parity_metrics(ref, ref_bf16)   # what quantising the cache costs, oracle vs oracle
    print(f"{name}: rel-Frobenius error of E4M3 + per-row scale against the BF16 cache = {q_err:.3e}")
    assert q_err < 6e-2    # 4 significant bits: about 2^-5 per element, averaged over thousands of keys


def test_fp8_attention_config5_step0_sampled():
    """BASELINE.json config 5 (65536 cached rows, 970 x 40 x 128 queries) with the cache held in FP8 -- the launch bench.py times
    in aux.fp8_kv_cache.cfg5.  The cache image (codes and exponents written by ws_kv_cache_write_fp8) is compared bit for bit with
    the oracle's; the attention output of step 0 is compared on 1024 sampled (row, head) outputs that the oracle computes one by
    one on the dequantised cache (full size -> sampled outputs), and the whole output must be written and in range."""
    cfg = wl.CONFIGS["cfg5"]
    x = wl.generate(cfg)
    kc, vc = x["k_cache"].copy(), x["v_cache"].copy()
    wsref.kv_cache_write(kc, vc, x["k_slice"], x["v_slice"], 0, cfg.write_offset)
    Tc, H, d, cap = cfg.cache_len, cfg.H, cfg.d, cfg.capacity
    k_rows = np.ascontiguousarray(np.transpose(kc[:, :Tc], (1, 0, 2)))
    v_rows = np.ascontiguousarray(np.transpose(vc[:, :Tc], (1, 0, 2)))
    del kc, vc
    kc8, vc8, ke, ve = gpu_write(k_rows, v_rows, H, cap, 0, 0, fill=(0, 0, 0, 0))
    w = ref_write(k_rows, v_rows, H, cap, 0, 0, fill=(0, 0, 0, 0))
    del k_rows, v_rows
    for g, ww, what in zip((kc8, vc8, ke, ve), w, ("k codes", "v codes", "k exponents", "v exponents")):
        assert np.array_equal(g.cpu().numpy(), ww), f"cfg5 cache image, {what}"
    kd, vd = wsref_fp8.kv_cache_dequant_fp8(w[0], w[2], Tc), wsref_fp8.kv_cache_dequant_fp8(w[1], w[3], Tc)
    del w
    q, kn, vn = x["q"][0], x["k_new"][0], x["v_new"][0]
    tq, tkn, tvn = to_dev(q, "bf16"), to_dev(kn, "bf16"), to_dev(vn, "bf16")
    out = torch.full_like(tq, float("nan"))
    lse = torch.full((H, cfg.Lq), float("nan"), dtype=torch.float32, device="cuda")
    wsp = workspace_for(cfg.Lq, H, d, Tc + cfg.Ln)
    wsp.fill_(0xFF)
    ws.block_causal_attn_fp8kv(out, tq, kc8, vc8, ke, ve, Tc, tkn, tvn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale, wsp, lse=lse)
    torch.cuda.synchronize()
    got = to_host(out)
    assert np.all(np.isfinite(got)) and np.abs(got).max() <= 4.0, "whole output must be written and inside the value range"
    rows, heads = wl.sample_pairs(cfg, 1024)
    ref, ref_lse = wsref.block_causal_attn_rows(q, kd, vd, Tc, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale, rows, heads)
    check(got[rows, heads], lse.cpu().numpy()[heads, rows], ref, ref_lse, "cfg5 fp8 cache, step 0 (sampled)")


def test_fp8_errors_leave_outputs_untouched():
    q = torch.zeros(64, 2, 128, dtype=torch.bfloat16, device="cuda")
    kc8 = torch.zeros(2, 256, 128, dtype=torch.uint8, device="cuda")
    ke = torch.zeros(2, 256, dtype=torch.int8, device="cuda")
    out = torch.full_like(q, 7.0)
    wsp = workspace_for(64, 2, 128, 256)
    with pytest.raises(ws.WsError) as e:
        ws.block_causal_attn_fp8kv(out, q, kc8, kc8.clone(), ke, ke.clone(), 256, None, None, [64], [257], 0.1, wsp)
    assert e.value.status == -4
    with pytest.raises(ws.WsError) as e:   # capacity not a multiple of 16
        ws.block_causal_attn_fp8kv(out, q, kc8[:, :250].contiguous(), kc8[:, :250].contiguous(), ke[:, :250].contiguous(),
                                   ke[:, :250].contiguous(), 250, None, None, [64], [250], 0.1, wsp)
    assert e.value.status == -3
    src = torch.zeros(8, 2, 128, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(ws.WsError) as e:
        ws.kv_cache_write_fp8(kc8, kc8.clone(), ke, ke.clone(), src, src.clone(), 0, 250)
    assert e.value.status == -4
    torch.cuda.synchronize()
    assert torch.all(out == 7.0) and torch.all(kc8 == 0)
