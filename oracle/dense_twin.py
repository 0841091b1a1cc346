"""Brute-force twin of the attention oracle: explicit dense mask, numpy FP64.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rule as oracle/wsref.c).  Written separately from
wsref.c on purpose -- different language, different formulation -- so that the two pin each
other: wsref.c loops over the visible prefix of the key timeline; this file concatenates the
keys, gives every query and every key a *block id*, materialises the whole Lq x Lk additive
mask (0 where key_block <= query_block, -inf elsewhere), and does softmax(S + mask) @ V.

PAPER.md:25 ("coordinated by block-causal attention"), reading R1: a query in block
b attends to every key that belongs to blocks <= b.
"""
from __future__ import annotations

import numpy as np


def block_ids(q_block_end, kv_visible, Lq: int, Lk: int):
    """query_block[i] = first b with i < q_block_end[b];
    key_block[j] = first b with j < kv_visible[b] (n_blocks if no block sees key j)."""
    q_block_end = np.asarray(q_block_end, np.int64)
    kv_visible = np.asarray(kv_visible, np.int64)
    nb = len(q_block_end)
    qb = np.full(Lq, -1, np.int64)
    for i in range(Lq):
        for b in range(nb):
            if i < q_block_end[b]:
                qb[i] = b
                break
    kb = np.full(Lk, nb, np.int64)
    for j in range(Lk):
        for b in range(nb):
            if j < kv_visible[b]:
                kb[j] = b
                break
    return qb, kb


def dense_mask(q_block_end, kv_visible, Lq: int, Lk: int):
    qb, kb = block_ids(q_block_end, kv_visible, Lq, Lk)
    allowed = kb[None, :] <= qb[:, None]
    return np.where(allowed, 0.0, -np.inf)


def dense_masked_attn(q, k_cache, v_cache, cache_len, k_new, v_new, q_block_end, kv_visible, softmax_scale):
    """q [Lq,H,d]; k_cache/v_cache [H,cap,d]; k_new/v_new [Ln,H,d] or None.
    Returns (out [Lq,H,d], lse [H,Lq], p [H,Lq,Lk]) in float64."""
    q = np.asarray(q, np.float64)
    Lq, H, d = q.shape
    kc = np.asarray(k_cache, np.float64)[:, :cache_len, :]
    vc = np.asarray(v_cache, np.float64)[:, :cache_len, :]
    if k_new is not None and len(k_new) > 0:
        kn = np.transpose(np.asarray(k_new, np.float64), (1, 0, 2))  # [H, Ln, d]
        vn = np.transpose(np.asarray(v_new, np.float64), (1, 0, 2))
        K = np.concatenate([kc, kn], axis=1)
        V = np.concatenate([vc, vn], axis=1)
    else:
        K, V = kc, vc
    Lk = K.shape[1]
    mask = dense_mask(q_block_end, kv_visible, Lq, Lk)  # [Lq, Lk]
    out = np.zeros((Lq, H, d), np.float64)
    lse = np.full((H, Lq), -np.inf, np.float64)
    p_all = np.zeros((H, Lq, Lk), np.float64)
    for h in range(H):
        S = softmax_scale * (q[:, h, :] @ K[h].T) + mask  # [Lq, Lk]
        for i in range(Lq):
            row = S[i]
            m = np.max(row) if Lk > 0 else -np.inf
            if not np.isfinite(m):
                continue  # no visible key: O = 0, lse = -inf (R11)
            e = np.exp(row - m)
            l = e.sum()
            p = e / l
            p_all[h, i] = p
            out[i, h] = p @ V[h]
            lse[h, i] = m + np.log(l)
    return out, lse, p_all
