"""CPU test of bench.py's multi-rank path (replicas only): world_size 2 over gloo, barrier + max-over-ranks timing."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    sec = bench.max_over_ranks(1.0 + rank, world, dist, torch, "cpu")      # rank 1 is the slow one
    q.put((rank, sec, bench.aggregate_rate(1000, 5, 2, sec, world)))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_max_over_ranks_and_aggregate_gloo():
    import torch.multiprocessing as mp
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
    for rank, sec, rate in res:
        assert sec == pytest.approx(2.0)                       # every rank sees the slowest rank's time
        assert rate == pytest.approx(2 * 1000 * 5 * 2 / 2.0 / 1e9)


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(0.5, 1, None, None, "cpu") == 0.5
    assert bench.aggregate_rate(21600000, 5, 10, 0.6, 1) == pytest.approx(1.8)
