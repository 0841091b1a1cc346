"""Pins for the Ulysses-exchange oracle (oracle/wsref_ulysses.c) against things other than itself.  No GPU needed.

SURVEY.md 8(f).2 / DESIGN.md reading R20: exchange #1 (all-to-all, seq -> head), exchange #2 (all-to-all for the sharded
video rows, all-gather for the unsharded audio rows, head -> seq) and the K/V-slice broadcast fused with the cache write.
The multi-process tests carry the two exchanges out for real with torch.distributed (gloo, CPU ranks)."""
import os
import sys

import numpy as np
import pytest

from oracle import wsref, wsref_ulysses as uly

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def ids(shape, base=0):
    return (np.arange(int(np.prod(shape)), dtype=np.float32) + base).reshape(shape)


def make_xs(P, Ls, La, H, d, seed=0, dtype=np.float32):
    """Rank r's X_r [Ls + La, H, d]: distinct ids for the video rows, THE SAME audio rows on every rank (replicated)."""
    audio = ids((La, H, d), 9e6)
    return [np.concatenate([ids((Ls, H, d), 1e5 * (r + 1) + seed), audio]).astype(dtype) for r in range(P)]


# ---------------------------------------------------------------------------------------------- exchange #1
@pytest.mark.parametrize("P,Ls,La,H,d", [(4, 5, 3, 8, 4), (2, 7, 0, 6, 2), (1, 4, 2, 3, 2), (8, 2, 1, 8, 2)])
def test_seq_to_head_is_the_numpy_statement(P, Ls, La, H, d):
    xs = make_xs(P, Ls, La, H, d)
    ys = uly.seq_to_head(xs, Ls)
    Hp = H // P
    video = np.concatenate([x[:Ls] for x in xs])                       # the whole video sequence, token-major [P * Ls, H, d]
    for g in range(P):
        want = np.concatenate([video[:, g * Hp:(g + 1) * Hp], xs[g][Ls:, g * Hp:(g + 1) * Hp]])
        assert ys[g].shape == (P * Ls + La, Hp, d) and np.array_equal(ys[g], want)


@pytest.mark.parametrize("dtype", [np.float32, np.uint16, np.uint8])
def test_exchanges_are_byte_moves_for_any_element_size(dtype):
    xs = make_xs(2, 3, 2, 4, 8, dtype=dtype)
    ys = uly.seq_to_head(xs, 3)
    assert ys[1].dtype == dtype and np.array_equal(ys[1][3:6], xs[1][:3, 2:4])


# ---------------------------------------------------------------------------------------------- exchange #2
@pytest.mark.parametrize("P,Ls,La,Hp,d", [(4, 5, 3, 2, 4), (2, 7, 0, 3, 2), (1, 4, 2, 3, 2)])
def test_head_to_seq_is_the_numpy_statement(P, Ls, La, Hp, d):
    os_ = [ids((P * Ls + La, Hp, d), 1e5 * (g + 1)) for g in range(P)]
    zs = uly.head_to_seq(os_, Ls)
    full = np.concatenate(os_, axis=1)                                 # all heads side by side: [P * Ls + La, H, d]
    for r in range(P):
        want = np.concatenate([full[r * Ls:(r + 1) * Ls], full[P * Ls:]])   # own video shard + every audio row (gather)
        assert zs[r].shape == (Ls + La, P * Hp, d) and np.array_equal(zs[r], want)


def test_exchange_2_after_exchange_1_is_the_identity_on_every_rank():
    P, Ls, La, H, d = 4, 6, 5, 8, 3
    xs = make_xs(P, Ls, La, H, d, seed=7)
    zs = uly.head_to_seq(uly.seq_to_head(xs, Ls), Ls)
    for r in range(P):
        assert np.array_equal(zs[r], xs[r])


def test_bad_arguments():
    with pytest.raises(ValueError):
        uly.seq_to_head([np.zeros((4, 3, 2), np.float32)] * 2, 3)      # 3 heads over 2 ranks


# ---------------------------------------------------------------------------------------------- the pipeline
def test_ulysses_pipeline_equals_single_rank_attention_on_all_heads():
    """exchange #1 -> attention on each rank's Hp heads -> exchange #2 must equal attention on all H heads computed in one
    place, cut into token shards: heads are independent, which is all Ulysses relies on."""
    rng = np.random.default_rng(3)
    P, Ls, La, H, d, Tc = 2, 6, 3, 4, 8, 10
    Hp, L = H // P, P * Ls + La
    audio_q, audio_k, audio_v = (rng.standard_normal((La, H, d)).astype(np.float32) for _ in range(3))
    mk = lambda a: [np.concatenate([rng.standard_normal((Ls, H, d)).astype(np.float32), a]) for _ in range(P)]
    q_r, k_r, v_r = mk(audio_q), mk(audio_k), mk(audio_v)
    kc, vc = rng.standard_normal((H, Tc, d)).astype(np.float32), rng.standard_normal((H, Tc, d)).astype(np.float32)
    qe, kv, scale = [L], [Tc + L], 0.3
    # one place, all heads: the full token-major sequence is the video shards in rank order, then the audio rows
    cat = lambda xs: np.concatenate([x[:Ls] for x in xs] + [xs[0][Ls:]])
    want, _ = wsref.block_causal_attn(cat(q_r), kc, vc, Tc, cat(k_r), cat(v_r), qe, kv, scale)
    # the performer group
    qg, kg, vg = uly.seq_to_head(q_r, Ls), uly.seq_to_head(k_r, Ls), uly.seq_to_head(v_r, Ls)
    og = [wsref.block_causal_attn(qg[g], kc[g * Hp:(g + 1) * Hp], vc[g * Hp:(g + 1) * Hp], Tc, kg[g], vg[g], qe, kv, scale)[0]
          for g in range(P)]
    zs = uly.head_to_seq(og, Ls)
    for r in range(P):
        assert np.max(np.abs(zs[r][:Ls] - want[r * Ls:(r + 1) * Ls])) < 1e-12
        assert np.max(np.abs(zs[r][Ls:] - want[P * Ls:])) < 1e-12


# ---------------------------------------------------------------------------------------------- broadcast write
def test_slice_broadcast_write_is_the_cache_write_of_every_rank():
    P, Hp, cap, d, n, off = 4, 2, 12, 4, 5, 6
    ks, vs = ids((n, P * Hp, d), 100), ids((n, P * Hp, d), 9000)
    kcs = [ids((Hp, cap, d), 1e5 * (g + 1)) for g in range(P)]
    vcs = [ids((Hp, cap, d), 2e5 * (g + 1)) for g in range(P)]
    want_k, want_v = [c.copy() for c in kcs], [c.copy() for c in vcs]
    for g in range(P):
        wsref.kv_cache_write(want_k[g], want_v[g], ks, vs, g * Hp, off)          # a1 on rank g (pinned against numpy elsewhere)
    uly.kv_slice_broadcast_write(kcs, vcs, ks, vs, off)
    for g in range(P):
        assert np.array_equal(kcs[g], want_k[g]) and np.array_equal(vcs[g], want_v[g])
        assert np.array_equal(kcs[g][:, off:off + n], ks[:, g * Hp:(g + 1) * Hp].transpose(1, 0, 2))   # and numpy directly
    with pytest.raises(ValueError):
        uly.kv_slice_broadcast_write(kcs, vcs, ks, vs, cap - n + 1)


# ---------------------------------------------------------------------------------------------- real collectives (gloo)
def _worker(rank, world, port, Ls, La, H, d, q):
    """Rank `rank` of a real process group: exchange #1 as all_to_all_single of the [P, Ls, Hp, d] pack (the G = P layout of
    a2), exchange #2 as all_to_all_single + all_gather of the audio rows; returns (Y_rank, Z_rank)."""
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    P, Hp = world, H // world
    x = torch.from_numpy(make_xs(P, Ls, La, H, d)[rank])
    # exchange #1: send chunk g = this rank's video tokens, heads of group g
    send = x[:Ls].reshape(Ls, P, Hp, d).permute(1, 0, 2, 3).contiguous()           # [P, Ls, Hp, d]
    recv = torch.empty_like(send)
    dist.all_to_all_single(recv, send)                                             # recv[r] = rank r's tokens, my heads
    y = torch.cat([recv.reshape(P * Ls, Hp, d), x[Ls:, rank * Hp:(rank + 1) * Hp]])
    # "attention": any per-head function of the full sequence will do for a data-movement pin
    o = y * 2.0 + 1.0
    # exchange #2: send chunk r = the output rows of rank r's tokens; audio rows are all-gathered
    send2 = o[:P * Ls].reshape(P, Ls, Hp, d).contiguous()
    recv2 = torch.empty_like(send2)
    dist.all_to_all_single(recv2, send2)                                           # recv2[g] = my tokens, heads of group g
    audio = [torch.empty(La, Hp, d) for _ in range(P)]
    dist.all_gather(audio, o[P * Ls:].contiguous())
    z = torch.cat([recv2.permute(1, 0, 2, 3).reshape(Ls, H, d), torch.cat(audio, dim=1)])
    q.put((rank, y.numpy(), z.numpy()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_oracle_exchanges_match_real_gloo_collectives(world):
    import torch.multiprocessing as mp
    Ls, La, H, d = 5, 3, 8, 4
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31000 + (os.getpid() * 7 + world) % 3000
    procs = [ctx.Process(target=_worker, args=(r, world, port, Ls, La, H, d, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=180) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    xs = make_xs(world, Ls, La, H, d)
    ys = uly.seq_to_head(xs, Ls)
    zs = uly.head_to_seq([y * 2.0 + 1.0 for y in ys], Ls)
    for rank, y, z in res:
        assert np.array_equal(y, ys[rank]), f"exchange #1, rank {rank}"
        assert np.array_equal(z, zs[rank]), f"exchange #2, rank {rank}"
