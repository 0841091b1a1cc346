"""Pins for the CPU oracle (oracle/wsref.c) against things other than itself.

No GPU needed.  Each test is chosen so a plausible mistake in the oracle (dropped term, wrong
sign/index, transposed operand, off-by-one in the visible prefix, wrong source at the
cache/new seam, wrong head stride) fails at least one of them.  SURVEY.md section 8(c).
"""
import math
import os

import numpy as np
import pytest

from oracle import dense_twin, wsref
from paper_2607_04443_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
TOL = 1e-12


def rand_problem(seed, H, d, Lq_blocks, vis, Tc, Ln, cap=None):
    rng = np.random.default_rng(seed)
    cap = cap or Tc + 3
    qe = np.cumsum(Lq_blocks).astype(np.int32)
    Lq = int(qe[-1])
    q = rng.standard_normal((Lq, H, d)).astype(np.float32)
    kc = rng.standard_normal((H, cap, d)).astype(np.float32)
    vc = rng.standard_normal((H, cap, d)).astype(np.float32)
    kn = rng.standard_normal((Ln, H, d)).astype(np.float32) if Ln else None
    vn = rng.standard_normal((Ln, H, d)).astype(np.float32) if Ln else None
    return dict(q=q, k_cache=kc, v_cache=vc, cache_len=Tc, k_new=kn, v_new=vn, q_block_end=qe,
                kv_visible=np.asarray(vis, np.int32), softmax_scale=1.0 / math.sqrt(d))


def run(p, **kw):
    return wsref.block_causal_attn(p["q"], p["k_cache"], p["v_cache"], p["cache_len"], p["k_new"], p["v_new"],
                                   p["q_block_end"], p["kv_visible"], p["softmax_scale"], **kw)


def pure_python_attention(p):
    """The definition with nothing but Python floats and math.exp (tiny inputs only)."""
    q, kc, vc, Tc = p["q"], p["k_cache"], p["v_cache"], p["cache_len"]
    kn, vn = p["k_new"], p["v_new"]
    Lq, H, d = q.shape
    out = [[[0.0] * d for _ in range(H)] for _ in range(Lq)]
    lse = [[-math.inf] * Lq for _ in range(H)]
    for i in range(Lq):
        b = next(bb for bb, e in enumerate(p["q_block_end"]) if i < e)
        n = int(p["kv_visible"][b])
        for h in range(H):
            keys = [kc[h][j] if j < Tc else kn[j - Tc][h] for j in range(n)]
            vals = [vc[h][j] if j < Tc else vn[j - Tc][h] for j in range(n)]
            if n == 0:
                continue
            s = [p["softmax_scale"] * sum(float(q[i][h][c]) * float(keys[j][c]) for c in range(d)) for j in range(n)]
            m = max(s)
            e = [math.exp(x - m) for x in s]
            l = sum(e)
            for c in range(d):
                out[i][h][c] = sum(e[j] * float(vals[j][c]) for j in range(n)) / l
            lse[h][i] = m + math.log(l)
    return np.asarray(out), np.asarray(lse)


# ----------------------------------------------------------------------------------------------
# golden fixture: hand-worked rationals
# ----------------------------------------------------------------------------------------------
def read_golden(name):
    vals = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *rest = line.split()
            vals[k] = [float(x) for x in rest]
    return vals


def test_golden_two_keys_hand_worked():
    g = read_golden("softmax_two_keys.txt")
    q = np.asarray(g["q"], np.float32).reshape(2, 1, 2)
    k = np.asarray(g["k"], np.float32).reshape(3, 2)
    v = np.asarray(g["v"], np.float32).reshape(3, 2)
    kc = np.zeros((1, 4, 2), np.float32)
    vc = np.zeros((1, 4, 2), np.float32)
    kc[0, :2], vc[0, :2] = k[:2], v[:2]
    kc[0, 2:], vc[0, 2:] = 99.0, -99.0  # stale rows beyond cache_len must never be read
    out, lse, p = wsref.block_causal_attn(q, kc, vc, 2, k[2:].reshape(1, 1, 2), v[2:].reshape(1, 1, 2),
                                          g["q_block_end"], g["kv_visible"], math.log(g["scale_is_ln"][0]), return_p=True)
    want = np.asarray(g["out_num"]) / np.asarray(g["out_den"])
    np.testing.assert_allclose(out.reshape(-1), want, rtol=0, atol=1e-13)
    np.testing.assert_allclose(lse.reshape(-1), np.log(g["lse_is_ln"]), rtol=0, atol=1e-13)
    np.testing.assert_allclose(p[0, 0], np.asarray(g["p_row0_num"]) / np.asarray(g["p_row0_den"]), atol=1e-14)
    np.testing.assert_allclose(p[0, 1], np.asarray(g["p_row1_num"]) / np.asarray(g["p_row1_den"]), atol=1e-14)


# ----------------------------------------------------------------------------------------------
# definition by brute force / independent formulations
# ----------------------------------------------------------------------------------------------
CASES = [
    # seed, H, d, block sizes, kv_visible, Tc, Ln
    (0, 2, 4, [3, 2], [5, 9], 6, 3),
    (1, 1, 8, [4], [7], 7, 0),
    (2, 3, 2, [1, 1, 1], [1, 2, 3], 0, 3),
    (3, 2, 16, [5, 6], [0, 11], 4, 9),      # first block sees nothing (R11)
    (4, 2, 3, [2, 3, 2], [4, 4, 10], 4, 6),  # seam exactly at a block edge, repeated visibility
]


@pytest.mark.parametrize("case", CASES)
def test_oracle_equals_pure_python_definition(case):
    p = rand_problem(*case)
    out, lse = run(p)
    ref_out, ref_lse = pure_python_attention(p)
    np.testing.assert_allclose(out, ref_out, rtol=0, atol=TOL)
    fin = np.isfinite(ref_lse)
    assert np.array_equal(np.isfinite(lse), fin)
    np.testing.assert_allclose(lse[fin], ref_lse[fin], rtol=0, atol=TOL)


@pytest.mark.parametrize("case", CASES + [(5, 2, 64, [32, 32], [160, 192], 192, 0), (6, 3, 32, [17, 40, 7], [33, 100, 131], 70, 61)])
def test_oracle_equals_dense_mask_twin(case):
    p = rand_problem(*case)
    out, lse, pr = run(p, return_p=True)
    t_out, t_lse, t_p = dense_twin.dense_masked_attn(p["q"], p["k_cache"], p["v_cache"], p["cache_len"], p["k_new"],
                                                     p["v_new"], p["q_block_end"], p["kv_visible"], p["softmax_scale"])
    np.testing.assert_allclose(out, t_out, rtol=0, atol=TOL)
    np.testing.assert_allclose(pr, t_p, rtol=0, atol=TOL)
    fin = np.isfinite(t_lse)
    assert np.array_equal(np.isfinite(lse), fin)
    np.testing.assert_allclose(lse[fin], t_lse[fin], rtol=0, atol=TOL)


@pytest.mark.parametrize("name", ["cfg1", "cfg1_split"])
def test_cfg1_oracle_equals_twin_and_readings_agree(name):
    """BASELINE.json configs[0] under both readings of R2; they must give the same answer."""
    res = {}
    for nm in ("cfg1", "cfg1_split"):
        cfg = wl.CONFIGS[nm]
        x = wl.generate(cfg)
        kc, vc = x["k_cache"].copy(), x["v_cache"].copy()
        if cfg.write_rows:
            wsref.kv_cache_write(kc, vc, x["k_slice"], x["v_slice"], 0, cfg.write_offset)
        kn = x["k_new"][0] if cfg.Ln else None
        vn = x["v_new"][0] if cfg.Ln else None
        args = (x["q"][0], kc, vc, cfg.cache_len, kn, vn, cfg.q_block_end, cfg.kv_visible, cfg.softmax_scale)
        out, lse = wsref.block_causal_attn(*args)
        t_out, t_lse, _ = dense_twin.dense_masked_attn(*args)
        np.testing.assert_allclose(out, t_out, rtol=0, atol=TOL)
        np.testing.assert_allclose(lse, t_lse, rtol=0, atol=TOL)
        res[nm] = (out, lse)
    # the generator draws the slice (cfg1) and the new rows (cfg1_split) at the same point of the stream
    np.testing.assert_allclose(res["cfg1"][0], res["cfg1_split"][0], rtol=0, atol=TOL)
    np.testing.assert_allclose(res["cfg1"][1], res["cfg1_split"][1], rtol=0, atol=TOL)


def test_oracle_equals_torch_sdpa_fp64():
    torch = pytest.importorskip("torch")
    p = rand_problem(7, 3, 16, [9, 14, 5], [20, 37, 50], 25, 25)
    out, _ = run(p)
    K = np.concatenate([p["k_cache"][:, :25], np.transpose(p["k_new"], (1, 0, 2))], axis=1)
    V = np.concatenate([p["v_cache"][:, :25], np.transpose(p["v_new"], (1, 0, 2))], axis=1)
    allowed = np.zeros((28, 50), bool)
    prev = 0
    for e, v in zip(p["q_block_end"], p["kv_visible"]):
        allowed[prev:e, :v] = True
        prev = e
    tq = torch.from_numpy(np.transpose(p["q"], (1, 0, 2)).astype(np.float64))[None]
    o = torch.nn.functional.scaled_dot_product_attention(tq, torch.from_numpy(K.astype(np.float64))[None],
                                                         torch.from_numpy(V.astype(np.float64))[None],
                                                         attn_mask=torch.from_numpy(allowed), scale=p["softmax_scale"])
    np.testing.assert_allclose(out, np.transpose(o[0].numpy(), (1, 0, 2)), rtol=0, atol=1e-12)


def test_rows_entry_point_matches_full():
    p = rand_problem(8, 3, 8, [6, 7], [9, 20], 11, 9)
    out, lse = run(p)
    rows = np.asarray([0, 5, 6, 12, 3], np.int32)
    heads = np.asarray([2, 0, 1, 2, 1], np.int32)
    o, l = wsref.block_causal_attn_rows(p["q"], p["k_cache"], p["v_cache"], p["cache_len"], p["k_new"], p["v_new"],
                                        p["q_block_end"], p["kv_visible"], p["softmax_scale"], rows, heads)
    for s, (r, h) in enumerate(zip(rows, heads)):
        np.testing.assert_array_equal(o[s], out[r, h])
        assert l[s] == lse[h, r]


# ----------------------------------------------------------------------------------------------
# closed forms
# ----------------------------------------------------------------------------------------------
def test_equal_keys_give_mean_of_visible_values():
    p = rand_problem(10, 2, 8, [3, 4, 2], [5, 11, 17], 9, 8)
    p["k_cache"][:] = 0.25
    p["k_new"][:] = 0.25
    out, lse = run(p)
    V = np.concatenate([p["v_cache"][:, :9], np.transpose(p["v_new"], (1, 0, 2))], axis=1).astype(np.float64)
    prev = 0
    for e, n in zip(p["q_block_end"], p["kv_visible"]):
        for i in range(prev, e):
            for h in range(2):
                np.testing.assert_allclose(out[i, h], V[h, :n].mean(axis=0), rtol=0, atol=1e-13)
                s = p["softmax_scale"] * 0.25 * float(p["q"][i, h].astype(np.float64).sum())
                assert abs(lse[h, i] - (s + math.log(n))) < 1e-12
        prev = e


def test_zero_query_gives_mean_and_one_key_gives_v0():
    p = rand_problem(11, 2, 4, [2, 2], [1, 6], 3, 3)
    p["q"][:] = 0
    out, lse = run(p)
    V = np.concatenate([p["v_cache"][:, :3], np.transpose(p["v_new"], (1, 0, 2))], axis=1).astype(np.float64)
    for h in range(2):
        for i in (0, 1):
            np.testing.assert_allclose(out[i, h], V[h, 0], atol=1e-15)  # one visible key -> v_0
            assert abs(lse[h, i]) < 1e-15
        for i in (2, 3):
            np.testing.assert_allclose(out[i, h], V[h, :6].mean(axis=0), atol=1e-14)
            assert abs(lse[h, i] - math.log(6)) < 1e-14


def test_one_hot_keys_select_value_row():
    d, n, beta = 8, 8, 60.0
    rng = np.random.default_rng(12)
    kc = np.zeros((1, n, d), np.float32)
    kc[0, np.arange(n), np.arange(n)] = 1.0
    vc = rng.standard_normal((1, n, d)).astype(np.float32)
    q = np.zeros((n, 1, d), np.float32)
    q[np.arange(n), 0, np.arange(n)] = beta
    out, _ = wsref.block_causal_attn(q, kc, vc, n, None, None, [n], [n], 1.0)
    bound = (n - 1) * math.exp(-beta) * np.abs(vc).max() * 2
    assert np.max(np.abs(out[:, 0] - vc[0].astype(np.float64))) <= bound


# ----------------------------------------------------------------------------------------------
# invariants
# ----------------------------------------------------------------------------------------------
def test_row_sums_and_unit_values():
    p = rand_problem(20, 2, 8, [5, 5], [12, 20], 10, 10)
    _, _, pr = run(p, return_p=True)
    np.testing.assert_allclose(pr.sum(axis=-1), 1.0, atol=1e-14)
    assert np.all(pr[:, :5, 12:] == 0) and np.all(pr[:, :, :] >= 0)
    p["v_cache"][:] = 1
    p["v_new"][:] = 1
    out, _ = run(p)
    np.testing.assert_allclose(out, 1.0, atol=1e-14)


def test_permuting_keys_within_visible_prefix_of_all_blocks():
    """Keys [0, kv_visible[0]) are visible to every block: a joint permutation of (k_j, v_j) there
    changes nothing; the same for keys seen only by later blocks, permuted among themselves."""
    p = rand_problem(21, 2, 8, [4, 4], [7, 16], 9, 7)
    out, lse = run(p)
    rng = np.random.default_rng(0)
    K = np.concatenate([p["k_cache"][:, :9], np.transpose(p["k_new"], (1, 0, 2))], axis=1)
    V = np.concatenate([p["v_cache"][:, :9], np.transpose(p["v_new"], (1, 0, 2))], axis=1)
    perm = np.concatenate([rng.permutation(7), 7 + rng.permutation(9)])
    K2, V2 = K[:, perm], V[:, perm]
    q2 = dict(p)
    q2["k_cache"], q2["v_cache"] = np.ascontiguousarray(K2[:, :9]), np.ascontiguousarray(V2[:, :9])
    q2["k_new"] = np.ascontiguousarray(np.transpose(K2[:, 9:], (1, 0, 2)))
    q2["v_new"] = np.ascontiguousarray(np.transpose(V2[:, 9:], (1, 0, 2)))
    out2, lse2 = run(q2)
    np.testing.assert_allclose(out2, out, atol=1e-13)
    np.testing.assert_allclose(lse2, lse, atol=1e-13)


def test_key_shift_v_linearity_and_scale_tradeoff():
    p = rand_problem(22, 2, 8, [3, 5], [6, 14], 8, 6)
    out, lse = run(p)
    # adding one vector delta to every key shifts all logits of a row equally -> same O
    delta = np.linspace(-1, 1, 8).astype(np.float32) * 0.5
    s = dict(p)
    s["k_cache"] = (p["k_cache"].astype(np.float64) + delta).astype(np.float32)
    s["k_new"] = (p["k_new"].astype(np.float64) + delta).astype(np.float32)
    out_s, _ = run(s)
    np.testing.assert_allclose(out_s, out, atol=5e-6)  # float32 re-rounding of shifted keys
    # linear in V
    # (BF16-valued V so that 2 v + 1 is exact in float32)
    v0 = dict(p, v_cache=wl.bf16_round(p["v_cache"]), v_new=wl.bf16_round(p["v_new"]))
    out0, lse0 = run(v0)
    a = dict(v0)
    a["v_cache"], a["v_new"] = v0["v_cache"] * 2 + 1, v0["v_new"] * 2 + 1
    out_a, lse_a = run(a)
    np.testing.assert_allclose(out_a, out0 * 2 + 1, atol=1e-12)
    np.testing.assert_allclose(lse_a, lse0, atol=0)
    # Q * alpha with scale / alpha (alpha a power of two: exact)
    b = dict(p)
    b["q"], b["softmax_scale"] = p["q"] * 4, p["softmax_scale"] / 4
    out_b, lse_b = run(b)
    np.testing.assert_allclose(out_b, out, atol=1e-13)
    np.testing.assert_allclose(lse_b, lse, atol=1e-13)


def test_merge_identity_and_single_vs_two_source():
    """Attention over A u B = LSE-weighted merge of attention over A and over B; and moving rows
    from the 'new' source into the cache (same timeline) changes nothing."""
    p = rand_problem(23, 2, 8, [6], [15], 9, 6)
    out, lse = run(p)
    a = dict(p, k_new=None, v_new=None, kv_visible=np.asarray([9], np.int32))
    out_a, lse_a = run(a)
    kcb = np.ascontiguousarray(np.transpose(p["k_new"], (1, 0, 2)))
    vcb = np.ascontiguousarray(np.transpose(p["v_new"], (1, 0, 2)))
    b = dict(p, k_cache=kcb, v_cache=vcb, cache_len=6, k_new=None, v_new=None, kv_visible=np.asarray([6], np.int32))
    out_b, lse_b = run(b)
    la, lb = lse_a.T[:, :, None], lse_b.T[:, :, None]
    m = np.maximum(la, lb)
    wa, wb = np.exp(la - m), np.exp(lb - m)
    merged = (wa * out_a + wb * out_b) / (wa + wb)
    np.testing.assert_allclose(merged, out, atol=1e-13)
    np.testing.assert_allclose((m + np.log(wa + wb))[:, :, 0].T, lse, atol=1e-13)
    # single source: everything in the cache
    K = np.concatenate([p["k_cache"][:, :9], kcb], axis=1)
    V = np.concatenate([p["v_cache"][:, :9], vcb], axis=1)
    c = dict(p, k_cache=np.ascontiguousarray(K), v_cache=np.ascontiguousarray(V), cache_len=15, k_new=None, v_new=None)
    out_c, lse_c = run(c)
    np.testing.assert_array_equal(out_c, out)
    np.testing.assert_array_equal(lse_c, lse)


def test_block_causal_equals_independent_prefix_calls():
    p = rand_problem(24, 2, 8, [3, 4, 5], [4, 9, 17], 10, 7)
    out, lse = run(p)
    prev = 0
    for e, n in zip(p["q_block_end"], p["kv_visible"]):
        sub = dict(p, q=np.ascontiguousarray(p["q"][prev:e]), q_block_end=np.asarray([e - prev], np.int32),
                   kv_visible=np.asarray([n], np.int32))
        o, l = run(sub)
        np.testing.assert_array_equal(o, out[prev:e])
        np.testing.assert_array_equal(l, lse[:, prev:e])
        prev = e


def test_heads_are_independent_so_relayout_commutes_with_attention():
    """What ws_block_causal_attn_seq_layout relies on: attention acts on each head separately,
    so seq->head, attention on the rank's heads, head->seq equals slicing those heads out of attention on all heads."""
    P, g0 = 2, 1
    p = rand_problem(41, 4, 8, [5, 6], [9, 20], 12, 11)          # H = 4 heads in the token-major tensors
    H, Hp = 4, 2
    full, full_lse = run(p)                                       # all heads
    def pack(a):
        o = np.empty((1, a.shape[0], Hp, a.shape[2]), a.dtype)
        wsref.seq_to_head(o, a, P, g0, 1)
        return o[0]
    sub = dict(p, q=pack(p["q"]), k_new=pack(p["k_new"]), v_new=pack(p["v_new"]),
               k_cache=np.ascontiguousarray(p["k_cache"][g0 * Hp:(g0 + 1) * Hp]),
               v_cache=np.ascontiguousarray(p["v_cache"][g0 * Hp:(g0 + 1) * Hp]))
    o, l = run(sub)
    back = np.full(full.shape, -7.0)
    wsref.head_to_seq(back, o[None], P, g0, 1)
    np.testing.assert_array_equal(back[:, g0 * Hp:(g0 + 1) * Hp], full[:, g0 * Hp:(g0 + 1) * Hp])
    np.testing.assert_array_equal(l, full_lse[g0 * Hp:(g0 + 1) * Hp])
    assert np.all(back[:, :g0 * Hp] == -7.0)                      # other ranks' heads untouched


def test_spike_key_at_every_boundary():
    """A key with a +40 logit at index kv_visible[b]-1 must dominate block b; at index kv_visible[b]
    it must have no effect on block b.  Also at the cache/new seam."""
    base = rand_problem(25, 1, 8, [3, 3, 3], [5, 12, 19], 8, 12)
    ref, _ = run(base)

    def with_spike(j):
        p = dict(base)
        p["k_cache"], p["v_cache"] = base["k_cache"].copy(), base["v_cache"].copy()
        p["k_new"], p["v_new"] = base["k_new"].copy(), base["v_new"].copy()
        # all queries equal so the spike logit is the same for every row
        p["q"] = np.ones_like(base["q"])
        big = np.full(8, 40.0 / (8 * p["softmax_scale"]), np.float32)
        val = np.full(8, 1000.0, np.float32)
        if j < 8:
            p["k_cache"][0, j], p["v_cache"][0, j] = big, val
        else:
            p["k_new"][j - 8, 0], p["v_new"][j - 8, 0] = big, val
        return p

    flat = dict(base, q=np.ones_like(base["q"]))
    ref_flat, _ = run(flat)
    for b, n in enumerate([5, 12, 19]):
        rows = slice(3 * b, 3 * b + 3)
        o, _ = run(with_spike(n - 1))
        assert np.all(np.abs(o[rows] - 1000.0) < 1e-6), "last visible key must dominate"
        if n < 19:
            o, _ = run(with_spike(n))
            np.testing.assert_array_equal(o[rows], ref_flat[rows])  # first invisible key: no effect
    for j in (7, 8):  # seam: last cache row / first new row, both visible to blocks 1, 2
        o, _ = run(with_spike(j))
        assert np.all(np.abs(o[3:] - 1000.0) < 1e-6)
        np.testing.assert_array_equal(o[:3], ref_flat[:3])
    assert ref.shape == ref_flat.shape


def test_empty_visible_set_and_bad_args():
    p = rand_problem(26, 2, 4, [2, 2], [0, 3], 3, 0)
    out, lse = run(p)
    assert np.all(out[:2] == 0) and np.all(np.isneginf(lse[:, :2])) and np.all(np.isfinite(out))
    with pytest.raises(ValueError):
        run(dict(p, kv_visible=np.asarray([2, 1], np.int32)))  # decreasing
    with pytest.raises(ValueError):
        run(dict(p, kv_visible=np.asarray([0, 4], np.int32)))  # beyond cache_len + Ln
    with pytest.raises(ValueError):
        run(dict(p, q_block_end=np.asarray([2, 3], np.int32)))  # last != Lq


# ----------------------------------------------------------------------------------------------
# cache write and relayouts: numpy slicing / transpose are the library routines
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [np.uint16, np.float32, np.uint8])
def test_cache_write_matches_numpy_slicing(dtype):
    rng = np.random.default_rng(30)
    H, cap, d, n, Hs, hb, off = 3, 17, 8, 5, 7, 2, 9
    kc = rng.integers(0, 200, (H, cap, d)).astype(dtype)
    vc = rng.integers(0, 200, (H, cap, d)).astype(dtype)
    ks = (np.arange(n * Hs * d).reshape(n, Hs, d) % 251).astype(dtype)  # unique-ish ids
    vs = ((np.arange(n * Hs * d).reshape(n, Hs, d) * 7 + 3) % 241).astype(dtype)
    want_k, want_v = kc.copy(), vc.copy()
    want_k[:, off:off + n] = np.transpose(ks[:, hb:hb + H], (1, 0, 2))
    want_v[:, off:off + n] = np.transpose(vs[:, hb:hb + H], (1, 0, 2))
    wsref.kv_cache_write(kc, vc, ks, vs, hb, off)
    np.testing.assert_array_equal(kc, want_k)
    np.testing.assert_array_equal(vc, want_v)
    with pytest.raises(ValueError):
        wsref.kv_cache_write(kc, vc, ks, vs, hb, cap - n + 1)
    with pytest.raises(ValueError):
        wsref.kv_cache_write(kc, vc, ks, vs, Hs - H + 1, 0)


@pytest.mark.parametrize("P,g0,G", [(4, 1, 1), (4, 0, 4), (1, 0, 1), (2, 1, 1), (4, 2, 2)])
def test_relayouts_match_numpy_transpose_and_round_trip(P, g0, G):
    n_tok, H, d = 11, 8, 4
    Hp = H // P
    src = np.arange(n_tok * H * d, dtype=np.uint16).reshape(n_tok, H, d)  # unique element ids
    dst = np.full((G, n_tok, Hp, d), 0xABCD, np.uint16)
    wsref.seq_to_head(dst, src, P, g0, G)
    want = np.transpose(src.reshape(n_tok, P, Hp, d), (1, 0, 2, 3))[g0:g0 + G]
    np.testing.assert_array_equal(dst, want)
    if P == 1:
        np.testing.assert_array_equal(dst[0], src)  # P = 1 is a plain copy
    back = np.full((n_tok, H, d), 0xEEEE, np.uint16)
    wsref.head_to_seq(back, dst, P, g0, G)
    sel = np.zeros(H, bool)
    sel[g0 * Hp:(g0 + G) * Hp] = True
    np.testing.assert_array_equal(back[:, sel], src[:, sel])
    assert np.all(back[:, ~sel] == 0xEEEE)  # other heads untouched
    again = np.zeros_like(dst)
    wsref.seq_to_head(again, back, P, g0, G)
    np.testing.assert_array_equal(again, dst)
    with pytest.raises(ValueError):
        wsref.seq_to_head(dst, src, 3, 0, 1)  # H % P != 0


def test_bf16_rounding_helper_matches_torch():
    torch = pytest.importorskip("torch")
    x = np.random.default_rng(40).standard_normal(10000).astype(np.float32)
    x[:4] = [1.00390625, 1.01171875, -1.00390625, 3.0e-40]  # exact ties and a subnormal
    want = torch.from_numpy(x).to(torch.bfloat16).to(torch.float32).numpy()
    got = wl.bf16_round(x)
    np.testing.assert_array_equal(got, want)
    np.testing.assert_array_equal(wl.bf16_from_bits(wl.bf16_bits(got)), got)


def test_config_work_figures_match_survey():
    """flops = 4 * Pi * d * H for the five configs."""
    assert wl.CONFIGS["cfg1"].visible_pairs() == 11264
    assert wl.CONFIGS["cfg3"].visible_pairs() == 16833380
    assert abs(wl.CONFIGS["cfg3"].attn_flops() / 1e9 - 344.75) < 0.01
    assert abs(wl.CONFIGS["cfg2"].attn_flops() / 1e9 - 30.44) < 0.01
    assert wl.CONFIGS["cfg4"].visible_pairs() == 68757120
    assert abs(wl.CONFIGS["cfg4"].attn_flops() / 1e9 - 352.04) < 0.01
    assert abs(wl.CONFIGS["cfg5"].attn_flops() / 1e9 - 1321.18) < 0.01
    assert wl.CONFIGS["cfg3"].cache_len == 16384 and wl.CONFIGS["cfg5"].cache_len == 65536


def test_parity_metrics_against_hand_values():
    """wsref.parity_metrics is what every attention parity assert goes through (north_star: max-abs error and
    relative Frobenius error of the GPU result against the oracle).  Hand values, chosen so that dividing by
    the wrong norm, dropping the abs, or squaring once too often/too seldom fails."""
    # got = (3, 4, 0), ref = (0, 0, 5): diff = (3, 4, -5); max|diff| = 5; |diff|_F = sqrt(50); |ref|_F = 5
    ma, rf = wsref.parity_metrics([3.0, 4.0, 0.0], [0.0, 0.0, 5.0])
    assert ma == 5.0 and abs(rf - math.sqrt(2.0)) < 1e-15
    # |got|_F = 5 too, so swap the magnitudes: got = (6, 8), ref = (3, 4): diff = (3, 4); rel = 5 / 5 = 1 (not 5 / 10)
    ma, rf = wsref.parity_metrics([6.0, 8.0], [3.0, 4.0])
    assert ma == 4.0 and abs(rf - 1.0) < 1e-15
    # the largest deviation is negative: abs must be taken before the max
    ma, rf = wsref.parity_metrics([[1.0, -7.0]], [[1.5, 1.0]])
    assert ma == 8.0 and abs(rf - math.sqrt(0.25 + 64.0) / math.sqrt(3.25)) < 1e-15
    # a sign flip of the whole tensor is a relative error of exactly 2
    x = np.array([[1.0, -2.0], [2.0, 4.0]])
    ma, rf = wsref.parity_metrics(-x, x)
    assert ma == 8.0 and abs(rf - 2.0) < 1e-15
    # identical tensors; an all-zero reference falls back to the absolute norm; empty tensors
    assert wsref.parity_metrics(x, x) == (0.0, 0.0)
    ma, rf = wsref.parity_metrics([3.0, 4.0], [0.0, 0.0])
    assert ma == 4.0 and rf == 5.0
    assert wsref.parity_metrics(np.zeros((0, 4)), np.zeros((0, 4))) == (0.0, 0.0)
    # float32 inputs are compared in FP64: a 1e-9 deviation must not vanish
    ma, _ = wsref.parity_metrics(np.float64(1.0) + 1e-9, np.float32(1.0))
    assert abs(ma - 1e-9) < 1e-15
    # several dimensions: the norm runs over the whole tensor, not per row
    got, ref = np.zeros((2, 3, 4)), np.zeros((2, 3, 4))
    ref[0, 0, 0], ref[1, 2, 3], got[1, 2, 3] = 3.0, 4.0, 4.0 + 0.5
    ma, rf = wsref.parity_metrics(got, ref)
    assert ma == 3.0 and abs(rf - math.sqrt(9.0 + 0.25) / 5.0) < 1e-15
