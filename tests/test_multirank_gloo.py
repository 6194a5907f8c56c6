"""The N > 1 path of bench.py is "replicas only": every rank refines its own copy, the only exchange is the
barrier + max-over-ranks timing + sum of units.  Covered here with a world_size-2 gloo run on CPU."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r pretends its K steps took (10 + 5 r) ms and consumed 1000 (r + 1) units
    ms, per_s, w = bench.aggregate_over_ranks(dist, 10.0 + 5.0 * rank, 1000.0 * (rank + 1))
    dist.barrier()
    q.put((rank, ms, per_s, w))
    dist.destroy_process_group()


def test_replica_aggregation_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, per_s, w in out:
        assert w == 2
        assert ms == pytest.approx(15.0)                    # max over ranks
        assert per_s == pytest.approx(3000.0 / 0.015)       # all ranks' units / max time


def test_single_process_aggregation():
    sys.path.insert(0, ROOT)
    import bench
    ms, per_s, w = bench.aggregate_over_ranks(None, 20.0, 500.0)
    assert (ms, w) == (20.0, 1) and per_s == pytest.approx(25000.0)
