"""Host logic of the attention work schedule (ws_attn_schedule), no GPU needed: every KV-tile
iteration of every (head, Q-pair) work item is assigned to exactly one CTA, the loads are balanced, and the
BASELINE.json configs take the schedules DESIGN.md says they take."""
import math

import pytest

import paper_2607_04443_b200 as ws
from paper_2607_04443_b200 import workloads as wl


def expand(plan, H):
    """-> per-CTA list of (item, tile) and per-CTA load."""
    tiles, grid, waves, pool = plan["pair_tiles"], plan["grid"], plan["n_waves"], plan["pool_begin"]
    n_pairs, Tp = len(tiles), sum(tiles)
    prefix = [0]
    for t in tiles:
        prefix.append(prefix[-1] + t)
    work = [[] for _ in range(grid)]
    for c in range(grid):
        for w in range(waves):
            item = w * grid + c
            work[c] += [(item, j) for j in range(tiles[item % n_pairs])]
        for t in range(pool[c], pool[c + 1]):
            head, rem = divmod(t, Tp)
            pair = max(p for p in range(n_pairs) if prefix[p] <= rem and tiles[p] > 0 and rem < prefix[p + 1])
            work[c].append((head * n_pairs + pair, rem - prefix[pair]))
    return work


def tiles_of(kv_vis, cache_len):
    if kv_vis <= 0:
        return 0
    nc = math.ceil(cache_len / 128)
    return math.ceil(kv_vis / 128) if kv_vis <= cache_len else nc + math.ceil((kv_vis - cache_len) / 128)


CASES = [
    # Lq, H, cache_len, Ln, q_block_end, kv_visible, n_sms
    (970, 40, 16384, 970, [970], [17354], 148),                                    # cfg3
    (3680, 10, 16384, 3680, [920, 1840, 2760, 3680], [17304, 18224, 19144, 20064], 148),  # cfg4
    (292, 24, 8192, 292, [292], [8484], 148),                                      # cfg2
    (970, 40, 65536, 970, [970], [66506], 148),                                    # cfg5
    (64, 2, 128, 64, [32, 64], [160, 192], 148),                                   # cfg1 (fewer iterations than SMs)
    (556, 160, 200, 250, [256, 556], [0, 450], 148),                               # whole pairs that see nothing
    (1100, 40, 300, 100, [1100], [400], 148),
    (1536, 30, 1500, 300, [256, 512, 768, 1024, 1280, 1536], [300, 600, 900, 1200, 1500, 1800], 148),
    (700, 7, 1000, 0, [700], [1000], 5),                                           # tiny device
    (300, 3, 0, 300, [100, 300], [0, 300], 132),
]


@pytest.mark.parametrize("case", CASES)
def test_every_iteration_is_assigned_exactly_once_and_loads_are_balanced(case):
    Lq, H, Tc, Ln, qe, kv, sms = case
    plan = ws.attn_schedule(Lq, H, Tc, Ln, qe, kv, sms)
    n_pairs = math.ceil(Lq / 256)
    # tiles per pair follow the last row of the pair
    want = []
    for p in range(n_pairs):
        last = min((p + 1) * 256, Lq) - 1
        b = next(i for i, e in enumerate(qe) if last < e)
        want.append(tiles_of(kv[b], Tc))
    assert plan["pair_tiles"] == want
    T = sum(want) * H
    assert 1 <= plan["grid"] <= sms
    assert plan["pool_begin"] == sorted(plan["pool_begin"])
    work = expand(plan, H)
    flat = [x for w in work for x in w]
    assert len(flat) == T and len(set(flat)) == T, "some iteration is missing or assigned twice"
    assert set(flat) == {(h * n_pairs + p, j) for h in range(H) for p in range(n_pairs) for j in range(want[p])}
    # phase-1 items are whole and phase-2 items are the tail of the item order
    first_pool_item = plan["n_waves"] * plan["grid"]
    for c, w in enumerate(work):
        for item, _ in w[sum(want[(k * plan["grid"] + c) % n_pairs] for k in range(plan["n_waves"])):]:
            assert item >= first_pool_item
    # balance: within 3 % (+1 iteration) of the perfectly even split
    if T:
        loads = [len(w) for w in work]
        assert max(loads) <= math.ceil(T / plan["grid"]) * 1.03 + 1


def test_baseline_configs_take_the_documented_schedules():
    def plan(name):
        c = wl.CONFIGS[name]
        return ws.attn_schedule(c.Lq, c.H, c.cache_len, c.Ln, list(c.q_block_end), list(c.kv_visible), 148)
    p3, p4, p2, p5 = plan("cfg3"), plan("cfg4"), plan("cfg2"), plan("cfg5")
    assert (p3["grid"], p3["n_waves"], p3["pair_tiles"]) == (148, 1, [136] * 4)       # 148 whole items + 12 split ones
    assert p3["pool_begin"][0] == 37 * 4 * 136 and p3["pool_begin"][-1] == 160 * 136
    assert (p5["grid"], p5["n_waves"]) == (148, 1)
    assert p4["n_waves"] == 0 and p4["pool_begin"][-1] == 10 * sum(p4["pair_tiles"])   # unequal items: pure stream-K
    assert p2["n_waves"] == 0 and p2["pair_tiles"] == [67, 67]                         # fewer items than SMs


def test_schedule_rejects_bad_masks():
    with pytest.raises(ws.WsError) as e:
        ws.attn_schedule(100, 2, 50, 0, [100], [51], 148)       # sees more keys than exist
    assert e.value.status == -4
    with pytest.raises(ws.WsError) as e:
        ws.attn_schedule(100, 2, 50, 0, [60, 100], [40, 30], 148)  # kv_visible must not decrease
    assert e.value.status == -1
