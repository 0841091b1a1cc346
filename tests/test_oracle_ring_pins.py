"""Pins for the ring-buffer K/V-cache oracle (oracle/wsref_ring.c) against things other than itself.  No GPU needed.

SURVEY.md 8(f).4 / DESIGN.md reading R19: the cache keeps the most recent `capacity` rows of the session; session row w
lives in physical row w mod capacity; the attention timeline runs over the window oldest row first."""
import numpy as np
import pytest

from oracle import wsref, wsref_ring as ring


def ids(shape, base=0):
    """float32 tensor whose every element is a distinct integer: any misplaced element shows."""
    return (np.arange(int(np.prod(shape)), dtype=np.float32) + base).reshape(shape)


# ---------------------------------------------------------------------------------------------- state rule
def test_ring_state_matches_a_brute_force_simulation_of_the_session():
    for capacity in (1, 3, 8, 10):
        phys_of = {}                                   # physical row -> session row it holds
        for W in range(0, 4 * capacity + 3):
            start, n = ring.ring_state(W, capacity)
            held = sorted(phys_of.values())
            assert n == len(held) == min(W, capacity)
            assert held == list(range(max(0, W - capacity), W))          # the most recent rows, nothing else
            # timeline order: key j is physical row (start + j) % capacity and holds session row (W - n + j)
            for j in range(n):
                assert phys_of[(start + j) % capacity] == W - n + j
            phys_of[W % capacity] = W                  # write session row W
    assert ring.ring_state(0, 5) == (0, 0) and ring.ring_state(5, 5) == (0, 5) and ring.ring_state(7, 5) == (2, 5)
    with pytest.raises(ValueError):
        ring.ring_state(-1, 5)
    with pytest.raises(ValueError):
        ring.ring_state(3, 0)


# ---------------------------------------------------------------------------------------------- write
@pytest.mark.parametrize("dtype", [np.float32, np.uint16, np.uint8])
def test_ring_write_matches_numpy_modular_indexing(dtype):
    H, cap, d, H_src, hb = 3, 11, 4, 5, 1
    for write_pos, n in [(0, 4), (9, 2), (9, 5), (10, 11), (25, 7), (11, 0), (1000003, 6)]:
        k0, v0 = ids((H, cap, d), 1e4).astype(dtype), ids((H, cap, d), 2e4).astype(dtype)
        ks, vs = ids((n, H_src, d), 3e4).astype(dtype), ids((n, H_src, d), 4e4).astype(dtype)
        k, v = k0.copy(), v0.copy()
        ring.kv_cache_write_ring(k, v, ks, vs, hb, write_pos)
        rows = (write_pos + np.arange(n)) % cap
        wk, wv = k0.copy(), v0.copy()
        wk[:, rows, :] = ks[:, hb:hb + H, :].transpose(1, 0, 2)      # numpy fancy indexing: an independent statement
        wv[:, rows, :] = vs[:, hb:hb + H, :].transpose(1, 0, 2)
        assert np.array_equal(k, wk) and np.array_equal(v, wv)        # whole images: untouched rows stay untouched


def test_ring_write_without_wrap_is_the_linear_write():
    H, cap, d = 2, 16, 8
    ks, vs = ids((5, 4, d), 100), ids((5, 4, d), 900)
    for pos in (0, 3, 11):
        k1, v1 = ids((H, cap, d)), ids((H, cap, d), 5000)
        k2, v2 = k1.copy(), v1.copy()
        ring.kv_cache_write_ring(k1, v1, ks, vs, 2, pos)
        wsref.kv_cache_write(k2, v2, ks, vs, 2, pos)
        assert np.array_equal(k1, k2) and np.array_equal(v1, v2)
    # one full lap later the same physical rows are hit
    k3, v3 = ids((H, cap, d)), ids((H, cap, d), 5000)
    ring.kv_cache_write_ring(k3, v3, ks, vs, 2, 11 + 3 * cap)
    assert np.array_equal(k3, k1) and np.array_equal(v3, v1)


def test_ring_write_rejects_more_rows_than_the_ring_and_bad_heads():
    k, v = np.zeros((2, 4, 8), np.float32), np.zeros((2, 4, 8), np.float32)
    src = np.zeros((5, 2, 8), np.float32)
    with pytest.raises(ValueError):
        ring.kv_cache_write_ring(k, v, src, src, 0, 0)            # 5 rows into a ring of 4
    with pytest.raises(ValueError):
        ring.kv_cache_write_ring(k, v, src[:2], src[:2], 1, 0)    # heads [1, 3) of 2
    with pytest.raises(ValueError):
        ring.kv_cache_write_ring(k, v, src[:2], src[:2], 0, -1)


def test_a_session_of_writes_keeps_exactly_the_most_recent_rows_in_timeline_order():
    rng = np.random.default_rng(7)
    H, cap, d = 2, 13, 4
    k, v = np.full((H, cap, d), -1.0, np.float32), np.full((H, cap, d), -2.0, np.float32)
    all_k, all_v = np.zeros((0, H, d), np.float32), np.zeros((0, H, d), np.float32)
    W = 0
    for step in range(12):
        n = int(rng.integers(0, 8))
        ks, vs = ids((n, H, d), 1000 * step), ids((n, H, d), 1000 * step + 500)
        ring.kv_cache_write_ring(k, v, ks, vs, 0, W)
        W += n
        all_k, all_v = np.concatenate([all_k, ks]), np.concatenate([all_v, vs])
        start, clen = ring.ring_state(W, cap)
        want_k, want_v = all_k[max(0, W - cap):W].transpose(1, 0, 2), all_v[max(0, W - cap):W].transpose(1, 0, 2)
        assert np.array_equal(ring.linearise(k, start, clen), want_k)
        assert np.array_equal(ring.linearise(v, start, clen), want_v)


# ---------------------------------------------------------------------------------------------- linearise
def test_linearise_is_numpy_roll():
    c = ids((3, 10, 4))
    for start in range(10):
        full = ring.linearise(c, start, 10)
        assert np.array_equal(full, np.roll(c, -start, axis=1))
        assert np.array_equal(ring.linearise(c, start, 6), np.roll(c, -start, axis=1)[:, :6])
    assert ring.linearise(c, 0, 0).shape == (3, 0, 4)
    with pytest.raises(ValueError):
        ring.linearise(c, 10, 3)
    with pytest.raises(ValueError):
        ring.linearise(c, 2, 11)


# ---------------------------------------------------------------------------------------------- attention
def rnd(rng, *shape):
    return rng.standard_normal(shape).astype(np.float32)


def test_ring_attention_with_a_fully_visible_cache_equals_attention_on_the_physical_order():
    """Softmax attention does not depend on the order of the visible keys: with every cache row visible to every query
    the ring (timeline) order and the physical order give the same result -- a property the linearisation cannot fake."""
    rng = np.random.default_rng(11)
    H, cap, d, Lq, Ln = 2, 40, 16, 9, 9
    kc, vc, q, kn, vn = rnd(rng, H, cap, d), rnd(rng, H, cap, d), rnd(rng, Lq, H, d), rnd(rng, Ln, H, d), rnd(rng, Ln, H, d)
    qe, kv = [4, 9], [cap + 4, cap + 9]
    want, want_lse = wsref.block_causal_attn(q, kc, vc, cap, kn, vn, qe, kv, 0.25)
    for start in (0, 1, 17, 39):
        got, lse = ring.block_causal_attn_ring(q, kc, vc, start, cap, kn, vn, qe, kv, 0.25)
        assert np.max(np.abs(got - want)) < 1e-12 and np.max(np.abs(lse - want_lse)) < 1e-12


def test_ring_attention_prefix_visibility_follows_the_timeline_not_the_physical_rows():
    """kv_visible cuts the TIMELINE (oldest first).  A spike key (logit +40) is planted on either side of the wrap seam:
    timeline index capacity - ring_start - 1 is the last physical row, the next timeline index is physical row 0."""
    rng = np.random.default_rng(12)
    H, cap, d, Lq = 1, 24, 8, 2
    start = 17
    seam = cap - start                              # timeline index of physical row 0
    q = np.zeros((Lq, H, d), np.float32); q[:, 0, 0] = 1.0
    for spike_j, vis, dominated in [(seam - 1, seam, True), (seam, seam, False), (seam, seam + 1, True),
                                    (cap - 1, cap - 1, False), (cap - 1, cap, True), (0, 1, True)]:
        kc, vc = 0.01 * rnd(rng, H, cap, d), rnd(rng, H, cap, d)
        phys = (start + spike_j) % cap
        kc[0, phys, :] = 0.0; kc[0, phys, 0] = 40.0
        vc[0, phys, :] = 7.0
        out, _ = ring.block_causal_attn_ring(q, kc, vc, start, cap, None, None, [Lq], [vis], 1.0)
        if dominated:
            assert np.max(np.abs(out - 7.0)) < 1e-9, (spike_j, vis)
        else:
            assert np.max(np.abs(out)) < 6.0, (spike_j, vis)       # the spike is outside the visible prefix
    # and the definition itself, spelled out once with numpy for a partially visible window
    kc, vc = rnd(rng, H, cap, d), rnd(rng, H, cap, d)
    vis = 10
    out, lse = ring.block_causal_attn_ring(q, kc, vc, start, cap, None, None, [Lq], [vis], 0.5)
    rows = (start + np.arange(vis)) % cap
    s = 0.5 * (q[:, 0, :].astype(np.float64) @ kc[0, rows, :].astype(np.float64).T)
    p = np.exp(s - s.max(axis=1, keepdims=True)); p /= p.sum(axis=1, keepdims=True)
    assert np.max(np.abs(out[:, 0, :] - p @ vc[0, rows, :].astype(np.float64))) < 1e-12
    assert np.max(np.abs(lse[0] - (np.log(np.exp(s - s.max(axis=1, keepdims=True)).sum(axis=1)) + s.max(axis=1)))) < 1e-12
