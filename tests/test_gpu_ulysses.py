"""GPU parity of the Ulysses-exchange row (R20) against the CPU oracle
(oracle/wsref_ulysses.c + wsref.c), through the C ABI.

One GPU stands in for the P performer ranks: every rank's buffers live on cuda:0 and the ranks' calls run one after the
other on one stream (no kernel ever waits for another rank), so "peer pointers" are plain local pointers -- the same
kernels store through peer-mapped pointers on a multi-GPU node.

  * ws_ulysses_push_seq_to_head (exchange #1) and ws_kv_slice_broadcast_write: whole destination images BIT-EXACT;
  * ws_block_causal_attn_push_out (attention + exchange #2 in its epilogue): bit-identical to ws_block_causal_attn followed
    by the oracle's exchange #2 of those outputs, other ranks' heads untouched, and within north_star's tolerance of the
    oracle pipeline (exchange #1 -> FP64 attention per rank -> exchange #2) == single-rank attention on all heads."""
import math

import numpy as np
import pytest
import torch

import paper_2607_04443_b200 as ws
from oracle import wsref, wsref_ulysses as uly
from paper_2607_04443_b200 import workloads as wl

from gpu_helpers import raw_bytes, to_dev, to_host, workspace_for

pytestmark = pytest.mark.gpu

MAX_ABS, REL_FRO = 2e-2, 1e-2


def gen(rng, dtype, *s):
    x = rng.standard_normal(s, dtype=np.float32)
    return wl.bf16_round(x) if dtype == "bf16" else x


def make_rank_inputs(rng, P, Ls, La, H, d, dtype):
    """X_r [Ls + La, H, d] per rank; the La audio rows are the same on every rank."""
    audio = gen(rng, dtype, La, H, d)
    return [np.concatenate([gen(rng, dtype, Ls, H, d), audio]) for _ in range(P)]


# ================================================================================================ exchange #1
@pytest.mark.parametrize("P,Ls,La,H,d,n_t,dtype", [
    (4, 920, 50, 40, 128, 3, "bf16"),     # config 4's rank group: Q, K_new, V_new of four 920-token shards + 50 audio tokens
    (2, 33, 0, 6, 64, 1, "bf16"),
    (8, 17, 5, 16, 64, 3, "bf16"),        # 24 (tensor, peer) pairs: more than one launch
    (1, 40, 7, 3, 128, 2, "bf16"),        # a group of one: a plain copy
    (4, 19, 3, 8, 32, 4, "f32"),
    (2, 0, 9, 4, 64, 2, "bf16"),          # nothing sharded
])
def test_push_seq_to_head_bit_exact_whole_images(P, Ls, La, H, d, n_t, dtype):
    rng = np.random.default_rng(P * 1000 + Ls)
    Hp = H // P
    xs = [make_rank_inputs(rng, P, Ls, La, H, d, dtype) for _ in range(n_t)]          # xs[i][r]
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    ys = [[torch.full((P * Ls + La, Hp, d), -3.0, dtype=tdt, device="cuda") for _ in range(P)] for _ in range(n_t)]
    for r in range(P):                                                                # each rank pushes its shard to every peer
        ws.ulysses_push_seq_to_head(ys, [to_dev(xs[i][r], dtype) for i in range(n_t)], Ls, r)
    torch.cuda.synchronize()
    for i in range(n_t):
        want = uly.seq_to_head(xs[i], Ls)
        for g in range(P):
            assert np.array_equal(raw_bytes(ys[i][g]), raw_bytes(to_dev(want[g], dtype))), (i, g)


def test_push_seq_to_head_of_one_rank_touches_only_its_rows():
    rng = np.random.default_rng(4)
    P, Ls, La, H, d, r = 4, 10, 3, 8, 64, 2
    x = make_rank_inputs(rng, P, Ls, La, H, d, "bf16")[r]
    ys = [[torch.full((P * Ls + La, H // P, d), 5.0, dtype=torch.bfloat16, device="cuda") for _ in range(P)]]
    ws.ulysses_push_seq_to_head(ys, [to_dev(x, "bf16")], Ls, r)
    torch.cuda.synchronize()
    for g in range(P):
        y = to_host(ys[0][g])
        mine = np.zeros(P * Ls + La, bool)
        mine[r * Ls:(r + 1) * Ls] = True
        if g == r:
            mine[P * Ls:] = True
        assert np.all(y[~mine] == 5.0)
        assert np.array_equal(y[r * Ls:(r + 1) * Ls], x[:Ls, g * 2:(g + 1) * 2])
    assert np.array_equal(to_host(ys[0][r])[P * Ls:], x[Ls:, r * 2:(r + 1) * 2])


# ================================================================================================ broadcast write
@pytest.mark.parametrize("P,Hp,cap,d,n,off,dtype", [(4, 10, 2048, 128, 1024, 1000, "bf16"), (8, 2, 64, 64, 9, 55, "bf16"),
                                                    (2, 3, 40, 32, 7, 0, "f32"), (1, 4, 32, 64, 5, 3, "bf16")])
def test_slice_broadcast_write_bit_exact(P, Hp, cap, d, n, off, dtype):
    rng = np.random.default_rng(cap + n)
    ks, vs = gen(rng, dtype, n, P * Hp, d), gen(rng, dtype, n, P * Hp, d)
    k0 = [gen(rng, dtype, Hp, cap, d) for _ in range(P)]
    v0 = [gen(rng, dtype, Hp, cap, d) for _ in range(P)]
    tk, tv = [to_dev(c, dtype) for c in k0], [to_dev(c, dtype) for c in v0]
    n0 = ws.kernel_launch_count()
    ws.kv_slice_broadcast_write(tk, tv, to_dev(ks, dtype), to_dev(vs, dtype), off)
    torch.cuda.synchronize()
    assert ws.kernel_launch_count() == n0 + 1                                        # one kernel feeds every rank
    uly.kv_slice_broadcast_write(k0, v0, ks, vs, off)
    for g in range(P):
        assert np.array_equal(raw_bytes(tk[g]), raw_bytes(to_dev(k0[g], dtype))) and np.array_equal(raw_bytes(tv[g]), raw_bytes(to_dev(v0[g], dtype)))


# ================================================================================================ attention + exchange #2
def group_case(seed, P, Ls, La, Hp, d, Tc, blocks=None, dtype="bf16"):
    rng = np.random.default_rng(seed)
    H, L = P * Hp, P * Ls + La
    q_r, k_r, v_r = (make_rank_inputs(rng, P, Ls, La, H, d, dtype) for _ in range(3))
    kc, vc = gen(rng, dtype, H, max(Tc, 1), d), gen(rng, dtype, H, max(Tc, 1), d)
    if blocks is None:
        qe, kv = [L], [Tc + L]
    else:
        qe = list(np.cumsum(blocks))
        kv = [Tc + e for e in qe]
    return dict(P=P, Ls=Ls, La=La, Hp=Hp, H=H, d=d, L=L, Tc=Tc, q_r=q_r, k_r=k_r, v_r=v_r, kc=kc, vc=vc, qe=qe, kv=kv,
                scale=1.0 / math.sqrt(d), dtype=dtype)


def run_group(c, only_rank=None, fill=7.0):
    """The whole exchange on the GPU.  Returns (Z_r tensors, O_g of the plain attention call for comparison)."""
    P, Ls, La, Hp, H, d, L, Tc, dtype = (c[k] for k in ("P", "Ls", "La", "Hp", "H", "d", "L", "Tc", "dtype"))
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    ys = [[torch.empty((L, Hp, d), dtype=tdt, device="cuda") for _ in range(P)] for _ in range(3)]
    for r in range(P):
        ws.ulysses_push_seq_to_head(ys, [to_dev(c[k][r], dtype) for k in ("q_r", "k_r", "v_r")], Ls, r)
    zs = [torch.full((Ls + La, H, d), fill, dtype=tdt, device="cuda") for _ in range(P)]
    plain = []
    wsp = workspace_for(L, Hp, d, Tc + L, tdt)
    for g in range(P):
        if only_rank is not None and g != only_rank:
            plain.append(None)
            continue
        kc, vc = to_dev(c["kc"][g * Hp:(g + 1) * Hp], dtype), to_dev(c["vc"][g * Hp:(g + 1) * Hp], dtype)
        lse = torch.empty((Hp, L), dtype=torch.float32, device="cuda")
        ws.block_causal_attn_push_out(zs, g, Ls, ys[0][g], kc, vc, Tc, ys[1][g], ys[2][g], c["qe"], c["kv"], c["scale"], wsp, lse=lse)
        o = torch.empty((L, Hp, d), dtype=tdt, device="cuda")
        lse2 = torch.empty_like(lse)
        ws.block_causal_attn(o, ys[0][g], kc, vc, Tc, ys[1][g], ys[2][g], c["qe"], c["kv"], c["scale"], wsp, lse=lse2)
        torch.cuda.synchronize()
        assert torch.equal(lse, lse2)
        plain.append(o)
    torch.cuda.synchronize()
    return zs, plain


def oracle_group(c):
    """All heads in one place (FP64), cut into the ranks' token shards: what every Z_r must hold."""
    P, Ls = c["P"], c["Ls"]
    cat = lambda xs: np.concatenate([x[:Ls] for x in xs] + [xs[0][Ls:]])
    want, _ = wsref.block_causal_attn(cat(c["q_r"]), c["kc"], c["vc"], c["Tc"], cat(c["k_r"]), cat(c["v_r"]), c["qe"], c["kv"], c["scale"])
    return [np.concatenate([want[r * Ls:(r + 1) * Ls], want[P * Ls:]]) for r in range(P)]


GROUPS = [
    dict(seed=1, P=4, Ls=230, La=13, Hp=2, d=128, Tc=1024),                       # 4 x 230 + 13 = 933 rows: odd number of Q tiles
    dict(seed=2, P=2, Ls=150, La=0, Hp=3, d=64, Tc=300, blocks=[150, 150]),       # two causal blocks = the two shards
    dict(seed=3, P=8, Ls=40, La=24, Hp=1, d=128, Tc=2000),                        # split-KV work items -> the combine kernel's stores
    dict(seed=4, P=1, Ls=200, La=56, Hp=4, d=128, Tc=512),                        # a group of one: the plain call
    dict(seed=5, P=3, Ls=100, La=7, Hp=2, d=64, Tc=0, blocks=[100, 100, 107]),    # no cache
    dict(seed=6, P=4, Ls=64, La=5, Hp=2, d=64, Tc=128, dtype="f32"),
]


@pytest.mark.parametrize("kw", GROUPS)
def test_attention_with_fused_exchange_2_matches_plain_attention_and_the_oracle_pipeline(kw):
    c = group_case(**kw)
    zs, plain = run_group(c)
    # (1) data movement, exactly: Z_r is the oracle's exchange #2 of the plain call's outputs
    moved = uly.head_to_seq([to_host(o) for o in plain], c["Ls"])
    for r in range(c["P"]):
        assert np.array_equal(to_host(zs[r]), moved[r]), f"rank {r}"
    # (2) arithmetic: against FP64 attention on all heads in one place
    want = oracle_group(c)
    for r in range(c["P"]):
        ma, rf = wsref.parity_metrics(to_host(zs[r]), want[r])
        assert ma <= MAX_ABS and rf <= REL_FRO, f"rank {r}: max_abs={ma:.3e} rel_fro={rf:.3e}"


def test_a_rank_writes_only_its_own_heads_on_every_peer():
    c = group_case(seed=9, P=4, Ls=70, La=9, Hp=2, d=64, Tc=256)
    zs, _ = run_group(c, only_rank=2, fill=7.0)
    for r in range(4):
        z = to_host(zs[r])
        assert np.all(z[:, :4] == 7.0) and np.all(z[:, 6:] == 7.0)        # heads of ranks 0, 1 and 3 untouched
        assert not np.any(z[:, 4:6] == 7.0)                                # every row of rank 2's heads written, audio rows too


def test_config4_sized_group_whole_pipeline():
    """Config 4's geometry with the real exchange: P = 4 ranks, 4 x 920 video tokens + 50 audio tokens, 16384 cached rows,
    8 heads here (2 per rank; 40 heads take the FP64 oracle minutes)."""
    c = group_case(seed=11, P=4, Ls=920, La=50, Hp=2, d=128, Tc=16384, blocks=[920, 920, 920, 970])
    zs, plain = run_group(c)
    moved = uly.head_to_seq([to_host(o) for o in plain], c["Ls"])
    want = oracle_group(c)
    for r in range(4):
        assert np.array_equal(to_host(zs[r]), moved[r])
        ma, rf = wsref.parity_metrics(to_host(zs[r]), want[r])
        assert ma <= MAX_ABS and rf <= REL_FRO, f"rank {r}: max_abs={ma:.3e} rel_fro={rf:.3e}"


def test_config4_full_width_rank_against_the_oracle():
    """One rank of config 4's group at FULL width -- 10 heads, 4 x 920 + 50 queries, 16384 cached rows, four causal blocks --
    through exchange #1, attention with exchange #2 in its epilogue, against the FP64 oracle on that rank's heads: the launch
    configuration bench.py times in aux.ring_and_ulysses.ulysses_attention_rank."""
    rng = np.random.default_rng(21)
    P, Ls, La, Hp, d, Tc, g = 4, 920, 50, 10, 128, 16384, 1
    H, L = P * Hp, P * Ls + La
    q_r, k_r, v_r = (make_rank_inputs(rng, P, Ls, La, H, d, "bf16") for _ in range(3))
    kc, vc = gen(rng, "bf16", Hp, Tc, d), gen(rng, "bf16", Hp, Tc, d)
    qe = [Ls, 2 * Ls, 3 * Ls, L]
    kv = [Tc + e for e in qe]
    scale = 1.0 / math.sqrt(d)
    ys = [[torch.empty((L, Hp, d), dtype=torch.bfloat16, device="cuda") for _ in range(P)] for _ in range(3)]
    for r in range(P):
        ws.ulysses_push_seq_to_head(ys, [to_dev(t[r], "bf16") for t in (q_r, k_r, v_r)], Ls, r)
    zs = [torch.full((Ls + La, H, d), 7.0, dtype=torch.bfloat16, device="cuda") for _ in range(P)]
    wsp = workspace_for(L, Hp, d, Tc + L)
    ws.block_causal_attn_push_out(zs, g, Ls, ys[0][g], to_dev(kc, "bf16"), to_dev(vc, "bf16"), Tc, ys[1][g], ys[2][g], qe, kv, scale, wsp)
    torch.cuda.synchronize()
    yq, yk, yv = (uly.seq_to_head(t, Ls)[g] for t in (q_r, k_r, v_r))
    ref, _ = wsref.block_causal_attn(yq, kc, vc, Tc, yk, yv, qe, kv, scale)
    filler = np.full((L, Hp, d), 7.0, np.float32)
    want = uly.head_to_seq([ref.astype(np.float32) if i == g else filler for i in range(P)], Ls)
    for r in range(P):
        z = to_host(zs[r])
        assert np.all(np.delete(z, np.s_[g * Hp:(g + 1) * Hp], axis=1) == 7.0), f"rank {r}: other ranks' heads touched"
        ma, rf = wsref.parity_metrics(z[:, g * Hp:(g + 1) * Hp], want[r][:, g * Hp:(g + 1) * Hp])
        assert ma <= MAX_ABS and rf <= REL_FRO, f"rank {r}: max_abs={ma:.3e} rel_fro={rf:.3e}"


def test_exchange_errors_launch_nothing():
    P, Ls, La, H, d = 2, 8, 2, 4, 64
    x = torch.zeros((Ls + La, H, d), dtype=torch.bfloat16, device="cuda")
    ys = [[torch.full((P * Ls + La, H // P, d), 3.0, dtype=torch.bfloat16, device="cuda") for _ in range(P)]]
    n0 = ws.kernel_launch_count()
    with pytest.raises(ws.WsError) as e:
        ws.ulysses_push_seq_to_head(ys, [x], Ls, 2)                       # rank outside the group
    assert e.value.status == -1
    with pytest.raises(ws.WsError) as e:
        ws.ulysses_push_seq_to_head([[ys[0][0], ys[0][0]]], [x], Ls, 0)   # two peers given the same buffer
    assert e.value.status == -5
    q = torch.zeros((P * Ls + La, 2, d), dtype=torch.bfloat16, device="cuda")
    kc = torch.zeros((2, 16, d), dtype=torch.bfloat16, device="cuda")
    zs = [torch.full((Ls + La, H, d), 3.0, dtype=torch.bfloat16, device="cuda") for _ in range(P)]
    wsp = workspace_for(P * Ls + La, 2, d, 16)
    with pytest.raises(ws.WsError) as e:
        ws.block_causal_attn_push_out(zs, 5, Ls, q, kc, kc.clone(), 16, None, None, [P * Ls + La], [16], 1.0, wsp)
    assert e.value.status == -1
    with pytest.raises(ws.WsError) as e:
        ws.block_causal_attn_push_out([zs[0], zs[0]], 0, Ls, q, kc, kc.clone(), 16, None, None, [P * Ls + La], [16], 1.0, wsp)
    assert e.value.status == -5
    # a peer output laid over the queries, or over the workspace: the epilogue would overwrite what other CTAs still read
    pool = torch.zeros(8192, dtype=torch.bfloat16, device="cuda")
    q_in = pool[:q.numel()].view_as(q)
    z_over_q = pool[1024:1024 + zs[0].numel()].view_as(zs[0])
    with pytest.raises(ws.WsError) as e:
        ws.block_causal_attn_push_out([zs[0], z_over_q], 0, Ls, q_in, kc, kc.clone(), 16, None, None, [P * Ls + La], [16], 1.0, wsp)
    assert e.value.status == -5
    z_in_wsp = wsp[4096:4096 + 2 * zs[0].numel()].view(torch.bfloat16).view_as(zs[0])
    with pytest.raises(ws.WsError) as e:
        ws.block_causal_attn_push_out([z_in_wsp, zs[1]], 0, Ls, q, kc, kc.clone(), 16, None, None, [P * Ls + La], [16], 1.0, wsp)
    assert e.value.status == -5
    torch.cuda.synchronize()
    assert ws.kernel_launch_count() == n0
    assert all(float((t - 3.0).abs().sum()) == 0.0 for t in ys[0] + zs)
