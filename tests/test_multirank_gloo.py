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


# ------------------------------------------------------------------ batch-level sharding of Algorithm 2 (sharded.py)
def _shard_graphs():
    import graphgen as gg
    return {
        "rmat10_dir": gg.rmat(10, seed=2, symmetrize=False),
        "rmat9_sym": gg.rmat(9, seed=1),
        "er": gg.erdos_renyi(1500, 6000, seed=5),
        "grid": gg.grid2d(16),
        "weighted": gg.random_weighted_digraph(300, 2000, 9, max_w=3),
        "hub": gg.from_edge_list(2001, [(0, j) for j in range(1, 2001)] + [(j, j % 7 + 1) for j in range(1, 2001)]),
        "sinks_on_cuts": gg.from_edge_list(40, [(i, (i * 7) % 40) for i in range(0, 40, 3)] + [(i, (i + 1) % 40) for i in range(0, 40, 3)]),
    }


@pytest.mark.parametrize("name", ["rmat10_dir", "rmat9_sym", "er", "grid", "weighted", "hub", "sinks_on_cuts"])
@pytest.mark.parametrize("nb", [2, 5, 16])
def test_sharded_lockstep_equals_cpu_algorithm2(name, nb):
    """The exchange logic of the sharded driver (offsets of Eq. 4, block-map all-gather, per-rank quotient rows, inherited
    batches) with the oracle doing the per-batch work, for 1, 2 and 3 virtual ranks: the colouring equals the CPU Algorithm 2 with
    inherited batches on the same first cuts, bit for bit, whatever the number of ranks."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle
    from sharded_harness import OracleBackend, run_lockstep
    g = _shard_graphs()[name]
    n, rp, ci, wt = g.numpy()
    cap = max(1, -(-g.m // nb))
    want, k_want, outer_want, _ = oracle.rbsc(n, rp, ci, wt, cap, inherit=True)
    for world in (1, 2, 3):
        got, k, outer, ranks = run_lockstep(OracleBackend, n, g.row_ptr, g.col, g.weights, cap, world)
        assert got.numpy().tolist() == want.tolist(), (name, nb, world)
        assert k == k_want and outer == outer_want


def _shard_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from paper_2607_02603_b200.sharded import ShardedRefiner
    from sharded_harness import OracleBackend
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    out = {}
    for name, g in _shard_graphs().items():
        cap = max(1, g.m // 6 + 1)
        r = ShardedRefiner(OracleBackend(), g.n, g.row_ptr, g.col, g.weights, cap, seed=1, rank=rank, world=world)
        colours, k, outer = r.run(dist, "cpu")
        out[name] = (colours.tolist(), k, outer, r.state.n1 - r.state.n0)
    dist.barrier()
    q.put((rank, out))
    dist.destroy_process_group()


def test_sharded_world2_gloo_equals_cpu_algorithm2():
    """Two real ranks over gloo: all-gather of the block counts and all-gather-v of the block-map slices; both ranks end with
    the colouring of the CPU Algorithm 2 (inherited batches), and both really owned a part of the graph."""
    sys.path.insert(0, ROOT)
    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    shared = 0
    for name, g in _shard_graphs().items():
        n, rp, ci, wt = g.numpy()
        want, k_want, outer_want, _ = oracle.rbsc(n, rp, ci, wt, max(1, g.m // 6 + 1), inherit=True)
        for rank in (0, 1):
            colours, k, outer, owned = res[rank][name]
            assert colours == want.tolist() and k == k_want and outer == outer_want, (name, rank)
        shared += res[0][name][3] > 0 and res[1][name][3] > 0
    assert shared >= 4  # the graphs really were split over the two ranks
