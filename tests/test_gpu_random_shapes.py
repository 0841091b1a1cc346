"""Seeded sweep of the attention work schedule: 64 random problem shapes, 16 through each of the four entry-point families
(plain, ring cache, FP8 cache, exchange-in-epilogue), every call with a NaN-filled workspace, every output against the FP64
CPU oracle at north_star's tolerance (max-abs 2e-2, rel-Frobenius 1e-2; LSE 2e-2).

Why it exists: the one wrong-result bug of round 2 (a CTA left without pool work inside the CTA span of a split item; the
combine kernel read a partial record nobody wrote) was found by a random sweep, not by the hand-picked shapes.  The shapes
here aim where the schedule has its case distinctions: the number of work items H * ceil(Lq / 256) from 1 to a little over
twice the SM count (whole-item waves, pool, both), ragged last Q tiles (single units), cache lengths below / around / far
above one KV tile, masks that hide the cache or the unit's own rows.  Sizes are kept to what the oracle finishes in well
under a second each."""
import math

import numpy as np
import pytest
import torch

import paper_2607_04443_b200 as ws
from oracle import wsref, wsref_fp8, wsref_ring
from paper_2607_04443_b200 import workloads as wl

from gpu_helpers import to_dev, to_host, workspace_for

pytestmark = pytest.mark.gpu

MAX_ABS, REL_FRO, LSE_ABS = 2e-2, 1e-2, 2e-2
VARIANTS = ("plain", "ring", "fp8", "push_out")
N_CASES = 64
MAX_PAIRS = 3e7   # Lq * H * keys: about 15 GFLOP of FP64 for the oracle


def make_cases():
    rng = np.random.default_rng(20261106)
    cases = []
    for i in range(N_CASES):
        d = 64 if rng.random() < 0.25 else 128
        Lq = int(rng.integers(1, 1000))
        n_units = (Lq + 255) // 256
        H = max(1, int(rng.integers(1, 330)) // n_units)
        Tc = int((0, int(rng.integers(1, 129)), int(rng.integers(129, 1600)))[int(rng.integers(0, 3))])
        Ln = int((0, int(rng.integers(1, 400)))[int(rng.integers(0, 2))])
        if Tc + Ln == 0:
            Ln = Lq
        while Lq * H * (Tc + Ln) > MAX_PAIRS and H > 1:
            H = H * 3 // 4
        n_blocks = int(rng.integers(1, 4))
        cuts = sorted(set(int(x) for x in rng.integers(1, Lq + 1, n_blocks - 1)) - {Lq}) + [Lq] if Lq > 1 else [Lq]
        vis = sorted(int(x) for x in rng.integers(0, Tc + Ln + 1, len(cuts)))
        if rng.random() < 0.7:
            vis[-1] = Tc + Ln
        cases.append(dict(i=i, variant=VARIANTS[i % 4], seed=1000 + i, Lq=Lq, H=H, d=d, Tc=Tc, Ln=Ln, qe=cuts, kv=vis,
                          extra=int(rng.integers(0, 1 << 30))))
    return cases


CASES = make_cases()


def rnd(rng, *s):
    return wl.bf16_round(rng.standard_normal(s, dtype=np.float32))


def nan_workspace(Lq, H, d, kv_total):
    w = workspace_for(Lq, H, d, kv_total)
    w.fill_(0xFF)
    return w


def check(got, got_lse, ref, ref_lse, what):
    assert np.all(np.isfinite(got)), what
    ma, rf = wsref.parity_metrics(got, ref)
    assert ma <= MAX_ABS and rf <= REL_FRO, f"{what}: max_abs={ma:.3e} rel_fro={rf:.3e}"
    fin = np.isfinite(ref_lse)
    assert np.array_equal(np.isfinite(got_lse), fin), f"{what}: lse finiteness"
    if fin.any():
        assert np.max(np.abs(got_lse[fin] - ref_lse[fin])) <= LSE_ABS, f"{what}: lse"


@pytest.mark.parametrize("c", CASES, ids=lambda c: f"{c['i']:02d}-{c['variant']}-Lq{c['Lq']}-H{c['H']}-d{c['d']}-Tc{c['Tc']}-Ln{c['Ln']}")
def test_random_shape(c):
    rng = np.random.default_rng(c["seed"])
    Lq, H, d, Tc, Ln, qe, kv, variant = (c[k] for k in ("Lq", "H", "d", "Tc", "Ln", "qe", "kv", "variant"))
    scale = 1.0 / math.sqrt(d)
    q = rnd(rng, Lq, H, d)
    k_new, v_new = (rnd(rng, Ln, H, d), rnd(rng, Ln, H, d)) if Ln else (None, None)
    tq = to_dev(q, "bf16")
    tkn, tvn = (to_dev(k_new, "bf16"), to_dev(v_new, "bf16")) if Ln else (None, None)
    out = torch.full_like(tq, float("nan"))
    lse = torch.full((H, Lq), float("nan"), dtype=torch.float32, device="cuda")
    wsp = nan_workspace(Lq, H, d, Tc + Ln)
    what = f"case {c}"

    if variant in ("plain", "push_out"):
        cap = Tc + c["extra"] % 40
        kc, vc = rnd(rng, H, max(cap, 1), d), rnd(rng, H, max(cap, 1), d)
        ref, ref_lse = wsref.block_causal_attn(q, kc, vc, Tc, k_new, v_new, qe, kv, scale)
        tkc, tvc = to_dev(kc, "bf16"), to_dev(vc, "bf16")
        if variant == "plain":
            ws.block_causal_attn(out, tq, tkc, tvc, Tc, tkn, tvn, qe, kv, scale, wsp, lse=lse)
            torch.cuda.synchronize()
            check(to_host(out), lse.cpu().numpy(), ref, ref_lse, what)
            return
        # exchange #2 in the epilogue: P peers, this rank's heads land in columns [rank * H, (rank + 1) * H) of every Z_r
        P = 1 + c["extra"] % 4
        Ls = max(1, (Lq // P) - (c["extra"] >> 4) % 3) if Lq >= P else 0
        if Ls == 0:
            P, Ls = 1, Lq
        La, rank = Lq - P * Ls, (c["extra"] >> 8) % P
        zs = [torch.full((Ls + La, P * H, d), 3.0, dtype=torch.bfloat16, device="cuda") for _ in range(P)]
        ws.block_causal_attn_push_out(zs, rank, Ls, tq, tkc, tvc, Tc, tkn, tvn, qe, kv, scale, wsp, lse=lse)
        torch.cuda.synchronize()
        got = np.empty((Lq, H, d), np.float32)
        for r in range(P):
            z = to_host(zs[r])
            mine = z[:, rank * H:(rank + 1) * H]
            got[r * Ls:(r + 1) * Ls] = mine[:Ls]
            assert np.array_equal(mine[Ls:], to_host(zs[0])[Ls:, rank * H:(rank + 1) * H]), f"{what}: gathered rows differ on peer {r}"
            others = np.delete(z, np.s_[rank * H:(rank + 1) * H], axis=1)
            assert np.all(others == 3.0), f"{what}: peer {r}: another rank's heads were written"
        got[P * Ls:] = to_host(zs[0])[Ls:, rank * H:(rank + 1) * H]
        check(got, lse.cpu().numpy(), ref, ref_lse, what)
    elif variant == "ring":
        cap = max(Tc + c["extra"] % 50, 1)
        start = (c["extra"] >> 8) % cap if Tc else 0
        kc, vc = rnd(rng, H, cap, d), rnd(rng, H, cap, d)
        ref, ref_lse = wsref_ring.block_causal_attn_ring(q, kc, vc, start, Tc, k_new, v_new, qe, kv, scale)
        ws.block_causal_attn_ring(out, tq, to_dev(kc, "bf16"), to_dev(vc, "bf16"), start, Tc, tkn, tvn, qe, kv, scale, wsp, lse=lse)
        torch.cuda.synchronize()
        check(to_host(out), lse.cpu().numpy(), ref, ref_lse, what)
    else:  # fp8: the oracle quantises, the GPU attends on the oracle's codes, the reference attends on the dequantised rows
        cap = max(16, (Tc + 15) // 16 * 16)
        mag = np.float32(10.0) ** rng.uniform(-0.5, 0.5, (max(Tc, 1), H, 1)).astype(np.float32)
        ks, vs = rnd(rng, max(Tc, 1), H, d) * mag, rnd(rng, max(Tc, 1), H, d)
        kc8, vc8 = np.zeros((H, cap, d), np.uint8), np.zeros((H, cap, d), np.uint8)
        ke, ve = np.zeros((H, cap), np.int8), np.zeros((H, cap), np.int8)
        wsref_fp8.kv_cache_write_fp8(kc8, vc8, ke, ve, wl.bf16_round(ks), vs, 0, 0)
        kd, vd = wsref_fp8.kv_cache_dequant_fp8(kc8, ke, max(Tc, 1)), wsref_fp8.kv_cache_dequant_fp8(vc8, ve, max(Tc, 1))
        ref, ref_lse = wsref.block_causal_attn(q, kd, vd, Tc, k_new, v_new, qe, kv, scale)
        dev8 = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        ws.block_causal_attn_fp8kv(out, tq, dev8(kc8), dev8(vc8), dev8(ke), dev8(ve), Tc, tkn, tvn, qe, kv, scale, wsp, lse=lse)
        torch.cuda.synchronize()
        check(to_host(out), lse.cpu().numpy(), ref, ref_lse, what)
