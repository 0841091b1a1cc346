"""The N > 1 path of bench.py is "replicas only" (no data-path collective): what the ranks share is
the barrier, the max-over-ranks time and the summed unit count.  Covered here with gloo, world 2."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    r, w, d = bench.dist_setup(world, backend="gloo")
    assert (r, w) == (rank, world)
    d.barrier()
    ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 40.0, d, "cpu")
    q.put((rank, ms, units))
    d.barrier()
    d.destroy_process_group()


def test_aggregate_over_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units in res:
        assert ms == 15.0      # max over ranks
        assert units == 80.0   # replicas: every rank processed its own 40 units


def test_single_rank_is_identity():
    import bench
    assert bench.aggregate_over_ranks(3.5, 7.0, None, "cpu") == (3.5, 7.0)


def test_reference_arm_non_zero_ranks_do_no_work(monkeypatch, capsys):
    import bench
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(type("A", (), {"steps": 1, "warmup": 0})())
    assert capsys.readouterr().out == ""
