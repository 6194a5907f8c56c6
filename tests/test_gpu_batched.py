"""GPU parity tests of the batched path (Algorithm 2) and its step-level pieces."""
import os
import numpy as np
import pytest
import torch

import graphgen as gg
import oracle
from helpers import refines

pytestmark = pytest.mark.gpu
wl = pytest.importorskip("paper_2607_02603_b200")


def dev():
    return torch.device("cuda", 0)


# ------------------------------------------------------------------ B2
@pytest.mark.parametrize("seed", range(6))
def test_inner_labels_match_oracle(seed):
    g = gg.rmat(10, edge_factor=6, seed=seed, symmetrize=bool(seed % 2))
    n, rp, ci, wt = g.numpy()
    nb = 2 + seed
    eb = gg.random_edge_batches(g, nb, seed)
    sink = (torch.arange(n) % nb).to(torch.int32)
    want = oracle.inner_labels(n, rp, eb.numpy(), sink.numpy())
    got = wl.wl_inner_labels(n, g.row_ptr.to(dev()), eb.to(dev()), sink.to(dev())).cpu().numpy()
    assert (got == want).all()
    # disjointness (L145) and the census  sum_k |V_k| + |boundary| = n
    assert sum((got == k).sum() for k in range(nb)) + (got == -1).sum() == n


def test_inner_labels_contiguous_batches_have_few_boundary_nodes():
    g = gg.rmat(11, seed=3)
    n, rp, ci, wt = g.numpy()
    cuts = gg.contiguous_row_batches(g, g.m // 5 + 1)
    eb = torch.bucketize(torch.arange(g.m), cuts[1:-1], right=True).to(torch.int32)
    sink = torch.bucketize(g.row_ptr[:-1], cuts[1:-1], right=True).to(torch.int32)
    got = wl.wl_inner_labels(n, g.row_ptr.to(dev()), eb.to(dev()), sink.to(dev())).cpu().numpy()
    want = oracle.inner_labels(n, rp, eb.numpy(), sink.numpy())
    assert (got == want).all()
    assert (got == -1).sum() <= len(cuts) - 2


# ------------------------------------------------------------------ B6
def _rows_as_dicts(k, qrp, qc, qw):
    return [dict(zip(qc[qrp[b]:qrp[b + 1]].tolist(), qw[qrp[b]:qrp[b + 1]].tolist())) for b in range(k)]


@pytest.mark.parametrize("seed", range(6))
def test_quotient_matches_oracle(seed):
    g = gg.rmat(9, edge_factor=6, seed=seed, symmetrize=bool(seed % 2)) if seed < 4 else gg.random_weighted_digraph(300, 2500, seed, max_w=5)
    n, rp, ci, wt = g.numpy()
    c, counts, _ = oracle.refine(n, rp, ci, wt)
    k, qrp, qc, qw = oracle.quotient(n, rp, ci, wt, c)
    d = g.to(dev())
    grp, gc, gw = wl.wl_quotient(n, d.row_ptr, d.col, d.weights, torch.from_numpy(c).to(dev()), k)
    grp, gc, gw = grp.cpu().numpy(), gc.cpu().numpy(), gw.cpu().numpy()
    assert grp.tolist() == qrp.tolist()  # every (B, B') pair stored once => same row lengths
    assert _rows_as_dicts(k, grp, gc, gw) == _rows_as_dicts(k, qrp, qc, qw)


def test_quotient_of_a_non_coarsest_stable_colouring():
    g = gg.grid2d(12)
    n, rp, ci, wt = g.numpy()
    c = np.arange(n, dtype=np.int32)  # discrete partition: the quotient is the graph itself
    d = g.to(dev())
    grp, gc, gw = wl.wl_quotient(n, d.row_ptr, d.col, None, torch.from_numpy(c).to(dev()), n)
    assert grp.cpu().numpy().tolist() == rp.tolist()
    assert _rows_as_dicts(n, grp.cpu().numpy(), gc.cpu().numpy(), gw.cpu().numpy()) == \
        _rows_as_dicts(n, rp, ci, np.ones(g.m, dtype=np.int64))


# ------------------------------------------------------------------ Algorithm 2
BATCH_GRAPHS = {
    "rmat10_sym": lambda: gg.rmat(10, seed=1),
    "rmat11_dir": lambda: gg.rmat(11, seed=2, symmetrize=False),
    "er": lambda: gg.erdos_renyi(2000, 9000, seed=5),
    "grid": lambda: gg.grid2d(20),
    "weighted": lambda: gg.random_weighted_digraph(400, 3000, 9, max_w=3),
    "hub": lambda: gg.from_edge_list(3001, [(0, j) for j in range(1, 3001)] + [(j, j % 7 + 1) for j in range(1, 3001)]),
    "twins": lambda: gg.from_edge_list(6, [(0, 5), (1, 5), (2, 5), (3, 4), (4, 3)]),
}


@pytest.mark.parametrize("name", list(BATCH_GRAPHS))
@pytest.mark.parametrize("nb", [1, 2, 4, 16])
def test_batched_equals_cpu_algorithm2_and_invariants(name, nb):
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    cap = max(1, -(-g.m // nb))
    coarsest, _, _ = oracle.refine(n, rp, ci, wt)
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, wt, cap)
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb)
    got = res.colors.numpy()
    # bit-exact against the CPU Algorithm 2 that uses the deterministic oracle as RSC on the same edge partition
    assert got.tolist() == want.tolist()
    # the same with every batch uploaded again for its local refinement (no refinement on the staged quotient rows)
    res_nf = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb, flags=wl.WL_FLAG_NO_FUSED_RECUT)
    assert res_nf.colors.numpy().tolist() == want.tolist() and res_nf.stats["outer_iters"] == res.stats["outer_iters"]
    if res.stats["outer_iters"] >= 3 and name != "hub":  # (hub: a row longer than a batch, no fusion)
        assert res.stats["bytes_h2d"] < res_nf.stats["bytes_h2d"]  # one upload pass per later iteration instead of two
    assert res.num_colors == k_want
    assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
    # Theorem 2 (L163), refinement of the coarsest colouring (L165), case (i) (L208)
    assert oracle.is_stable(n, rp, ci, wt, got)
    assert refines(got, coarsest)
    if res.stats["last_num_batches"] == 1:
        assert got.tolist() == coarsest.tolist()


@pytest.mark.parametrize("name", list(BATCH_GRAPHS))
@pytest.mark.parametrize("nb", [2, 4, 16])
def test_batched_inherited_batches_equal_cpu_algorithm2(name, nb):
    """WL_FLAG_INHERIT_BATCHES (reading Q14b): from the second outer iteration on the quotient keeps the batches of its graph
    and is refined while its rows are still on the device.  Bit-exact against the CPU Algorithm 2 with the same rule, plus
    Theorem 2 and L165."""
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    cap = max(1, -(-g.m // nb))
    coarsest, _, _ = oracle.refine(n, rp, ci, wt)
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, wt, cap, inherit=True)
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb,
                               flags=wl.WL_FLAG_INHERIT_BATCHES)
    got = res.colors.numpy()
    assert got.tolist() == want.tolist()
    assert res.num_colors == k_want
    assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
    assert oracle.is_stable(n, rp, ci, wt, got)
    assert refines(got, coarsest)


@pytest.mark.parametrize("name", list(BATCH_GRAPHS))
@pytest.mark.parametrize("nb", [2, 3, 5, 16])
@pytest.mark.parametrize("inherit", [False, True])
def test_batched_aggressive_stop_equals_cpu_algorithm2(name, nb, inherit):
    """WL_FLAG_AGGRESSIVE_STOP (stop as soon as the next iteration would not run with fewer batches), alone and
    with inherited batches: bit-exact against the CPU Algorithm 2 with the same stop rule, same number of outer iterations;
    the result is a stable colouring (Thm 2) that refines the coarsest one and is refined by... the full loop's result is
    coarser or equal (L206)."""
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    cap = max(1, -(-g.m // nb))
    coarsest, _, _ = oracle.refine(n, rp, ci, wt)
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, wt, cap, inherit=inherit, aggressive=True)
    flags = wl.WL_FLAG_AGGRESSIVE_STOP | (wl.WL_FLAG_INHERIT_BATCHES if inherit else 0)
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb, flags=flags)
    got = res.colors.numpy()
    assert got.tolist() == want.tolist() and res.num_colors == k_want
    assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
    assert oracle.is_stable(n, rp, ci, wt, got) and refines(got, coarsest)
    full = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb,
                                flags=flags & ~wl.WL_FLAG_AGGRESSIVE_STOP)
    assert refines(got, full.colors.numpy()) and res.stats["outer_iters"] <= full.stats["outer_iters"]


# ------------------------------------------------------------------ arbitrary (COO) edge partitions, Thm 2
COO_PARTITIONS = {
    "random_edges": lambda g, nb, seed: gg.random_edge_batches(g, nb, seed),          # nearly every node is a boundary node
    "by_source": lambda g, nb, seed: gg.node_hash_edge_batches(g, nb, seed),          # all inner, V_k scattered
    "by_source_flip5": lambda g, nb, seed: gg.node_hash_edge_batches(g, nb, seed, 5),  # some boundary nodes, several iterations
}


@pytest.mark.parametrize("name", list(BATCH_GRAPHS))
@pytest.mark.parametrize("nb", [2, 3, 4])
@pytest.mark.parametrize("part", list(COO_PARTITIONS))
def test_batched_coo_partitions_equal_cpu_algorithm2(name, nb, part):
    """wl_refine_batched over an ARBITRARY edge partition given as COO batches: bit-exact against the CPU Algorithm 2 run on
    the same per-edge batch labels (oracle.rbsc(first_edge_batch=...)), Theorem 2 stability, refinement of the coarsest
    colouring, and invariance under renumbering the batches (L213)."""
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    eb = COO_PARTITIONS[part](g, nb, 7)
    cap = max(1, -(-g.m // nb))
    coarsest, _, _ = oracle.refine(n, rp, ci, wt)
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, wt, cap, first_edge_batch=eb.numpy(), num_first_batches=nb)
    res = wl.wl_refine_batched(n, None, None, None, max_batch_edges=cap, seed=nb, coo_batches=gg.coo_batches(g, eb, nb))
    got = res.colors.numpy()
    assert got.tolist() == want.tolist() and res.num_colors == k_want
    assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
    assert oracle.is_stable(n, rp, ci, wt, got) and refines(got, coarsest)
    # Def. 5 census of the first iteration
    src = gg.edge_sources(g).numpy()
    nbatches_of = np.zeros(n, dtype=np.int64)
    for k in range(nb):
        nbatches_of[np.unique(src[eb.numpy() == k])] += 1
    assert res.stats["boundary_nodes"] == int((nbatches_of >= 2).sum())
    # renumbering the batches (and shuffling the edges inside them) changes nothing
    perm = torch.tensor([(k + 1) % nb for k in range(nb)], dtype=torch.int32)
    batches2 = gg.coo_batches(g, perm[eb.long()], nb)
    batches2 = [(s.flip(0).contiguous(), c.flip(0).contiguous(), None if w is None else w.flip(0).contiguous())
                for s, c, w in batches2]
    # (sinks are inner to batch 0 by reading Q9, so a renumbering may group them with other nodes in iteration 1: the
    # renumbered run is compared with the CPU Algorithm 2 on the renumbered labels, and must be stable all the same)
    res2 = wl.wl_refine_batched(n, None, None, None, max_batch_edges=cap, seed=99, coo_batches=batches2)
    assert oracle.is_stable(n, rp, ci, wt, res2.colors.numpy()) and refines(res2.colors.numpy(), coarsest)
    want2, _, _, _ = oracle.rbsc(n, rp, ci, wt, cap, first_edge_batch=perm[eb.long()].numpy(), num_first_batches=nb)
    assert res2.colors.numpy().tolist() == want2.tolist()


# ------------------------------------------------------------------ initial classes (L94 carried into Algorithm 2, reading Q18)
@pytest.mark.parametrize("name", list(BATCH_GRAPHS))
@pytest.mark.parametrize("nb", [1, 2, 4, 16])
@pytest.mark.parametrize("classes", [2, 5])
def test_batched_with_initial_classes_equals_cpu_algorithm2(name, nb, classes):
    """wl_options.batched_init_colors in every mode of the CSR forms (fused re-cut, uploads twice, inherited batches, aggressive
    stop): bit-exact against the CPU Algorithm 2 started from the same classes; the result is stable (Thm 2), refines the
    classes and the coarsest stable colouring refining them, and equals it when the loop ends on one batch (L208)."""
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    cap = max(1, -(-g.m // nb))
    init = gg.random_partition(n, classes, 100 + nb)
    labels = (init * 3 + 1).to(torch.int32)  # arbitrary non-negative labels, not dense
    coarsest, _, _ = oracle.refine(n, rp, ci, wt, init.numpy())
    for flags, kw in [(0, {}), (wl.WL_FLAG_NO_FUSED_RECUT, {}), (wl.WL_FLAG_INHERIT_BATCHES, {"inherit": True}),
                      (wl.WL_FLAG_AGGRESSIVE_STOP, {"aggressive": True})]:
        want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, wt, cap, init=init.numpy(), **kw)
        res = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb, flags=flags, init_colors=labels)
        got = res.colors.numpy()
        assert got.tolist() == want.tolist() and res.num_colors == k_want
        assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
        assert oracle.is_stable(n, rp, ci, wt, got)
        assert refines(got, init.numpy()) and refines(got, coarsest)
        if res.stats["last_num_batches"] == 1 and not flags & wl.WL_FLAG_AGGRESSIVE_STOP:
            assert got.tolist() == coarsest.tolist()
    # one class = no classes
    one = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb,
                               init_colors=torch.full((n,), 9, dtype=torch.int32))
    none = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=nb)
    assert one.colors.tolist() == none.colors.tolist() and one.stats["outer_iters"] == none.stats["outer_iters"]


@pytest.mark.parametrize("name", ["rmat10_sym", "rmat11_dir", "weighted", "twins"])
@pytest.mark.parametrize("nb", [2, 3])
@pytest.mark.parametrize("part", list(COO_PARTITIONS))
def test_batched_coo_partitions_with_initial_classes(name, nb, part):
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    eb = COO_PARTITIONS[part](g, nb, 7)
    cap = max(1, -(-g.m // nb))
    init = gg.random_partition(n, 3, 5)
    coarsest, _, _ = oracle.refine(n, rp, ci, wt, init.numpy())
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, wt, cap, first_edge_batch=eb.numpy(), num_first_batches=nb,
                                                     init=init.numpy())
    res = wl.wl_refine_batched(n, None, None, None, max_batch_edges=cap, seed=nb, coo_batches=gg.coo_batches(g, eb, nb),
                               init_colors=init.to(torch.int32))
    got = res.colors.numpy()
    assert got.tolist() == want.tolist() and res.num_colors == k_want
    assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
    assert oracle.is_stable(n, rp, ci, wt, got) and refines(got, init.numpy()) and refines(got, coarsest)


@pytest.mark.parametrize("flags", [0, 4096])
def test_batched_with_initial_classes_over_several_tiles(flags):
    """A graph whose batches span several kernel tiles and a ragged tail (n = 2^15 + 77 with isolated tail nodes)."""
    g0 = gg.rmat(15, edge_factor=8, seed=4, symmetrize=False)
    n = g0.n + 77
    row_ptr = torch.cat([g0.row_ptr, g0.row_ptr[-1:].repeat(77)])
    rp, ci = row_ptr.numpy(), g0.col.numpy()
    init = gg.random_partition(n, 6, 11)
    cap = -(-g0.m // 7)
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, None, cap, init=init.numpy(), inherit=bool(flags & 4096))
    res = wl.wl_refine_batched(n, row_ptr, g0.col, None, max_batch_edges=cap, seed=3, flags=flags, init_colors=init)
    assert res.colors.numpy().tolist() == want.tolist() and res.num_colors == k_want
    assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
    assert oracle.is_stable(n, rp, ci, None, res.colors.numpy()) and refines(res.colors.numpy(), init.numpy())


def test_batched_initial_classes_errors_and_limits():
    g = gg.rmat(10, seed=3, symmetrize=False)
    n = g.n
    bad = torch.zeros(n, dtype=torch.int32)
    bad[n // 2] = -1
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=g.m // 3, init_colors=bad)
    assert e.value.code == wl.WL_EINVAL
    # discrete classes: nothing can merge, one outer iteration
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=g.m // 3, init_colors=torch.arange(n, dtype=torch.int32))
    assert res.num_colors == n and res.colors.tolist() == list(range(n)) and res.stats["outer_iters"] == 1
    # the classes count against the device cap (8 bytes per node): a cap that holds the run without them but not with them
    init = gg.random_partition(n, 4, 1).to(torch.int32)
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=g.m // 3, init_colors=init, device_cap_bytes=4 * n - 1)
    assert e.value.code == wl.WL_ENOMEM


def test_batched_coo_errors_and_edge_cases():
    g = gg.rmat(9, seed=2, symmetrize=False)
    n = g.n
    eb = gg.random_edge_batches(g, 3, 1)
    batches = gg.coo_batches(g, eb, 3)
    bad = [(s.clone(), c.clone(), w) for s, c, w in batches]
    bad[1][1][0] = n  # target out of range
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, None, None, None, max_batch_edges=g.m, coo_batches=bad)
    assert e.value.code == wl.WL_EINVAL
    bad = [(s.clone(), c.clone(), w) for s, c, w in batches]
    bad[2][0][-1] = -1  # source out of range
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, None, None, None, max_batch_edges=g.m, coo_batches=bad)
    assert e.value.code == wl.WL_EINVAL
    with pytest.raises(wl.WlError) as e:  # inherited batches are defined for row-contiguous partitions only
        wl.wl_refine_batched(n, None, None, None, max_batch_edges=g.m, coo_batches=batches, flags=wl.WL_FLAG_INHERIT_BATCHES)
    assert e.value.code == wl.WL_EINVAL
    # an empty batch, and a graph without edges
    empty = (torch.empty(0, dtype=torch.int32), torch.empty(0, dtype=torch.int32), None)
    res = wl.wl_refine_batched(n, None, None, None, max_batch_edges=g.m, coo_batches=batches + [empty])
    nn, rp, ci, wt = g.numpy()
    want, _, _, _ = oracle.rbsc(nn, rp, ci, wt, g.m, first_edge_batch=eb.numpy(), num_first_batches=4)
    assert res.colors.numpy().tolist() == want.tolist()
    res = wl.wl_refine_batched(5, None, None, None, max_batch_edges=1, coo_batches=[empty, empty])
    assert res.colors.tolist() == [0] * 5
    # a weighted row whose pieces sum to 2^32 across two batches (Theorem 1's precondition is per ROW, L129)
    s0 = torch.tensor([0, 1], dtype=torch.int32)
    c0 = torch.tensor([1, 0], dtype=torch.int32)
    w0 = torch.tensor([(1 << 31), 1], dtype=torch.int64)
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(2, None, None, None, max_batch_edges=4, coo_batches=[(s0, c0, w0), (s0[:1], c0[:1], w0[:1])])
    assert e.value.code == wl.WL_ERANGE


def test_batched_caller_supplied_slices():
    g = gg.rmat(10, seed=4)
    n, rp, ci, wt = g.numpy()
    cuts = gg.contiguous_row_batches(g, g.m // 3 + 1)
    want, k_want, _, _ = oracle.rbsc(n, rp, ci, wt, g.m // 3 + 1, first_cuts=cuts.numpy())
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=g.m // 3 + 1, cuts=cuts.tolist(), seed=1)
    assert res.colors.numpy().tolist() == want.tolist()


def test_batched_cut_inside_a_long_row():
    # one row of 3000 entries with cap 1000: the hub is a boundary node (Def. 5) in the first iteration
    g = BATCH_GRAPHS["hub"]()
    n, rp, ci, wt = g.numpy()
    want, k_want, outer, nbl = oracle.rbsc(n, rp, ci, wt, 1000)
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=1000, seed=3)
    assert res.colors.numpy().tolist() == want.tolist()
    assert res.stats["boundary_nodes"] >= 1
    assert oracle.is_stable(n, rp, ci, wt, res.colors.numpy())


def test_batched_with_caller_host_workspace_and_long_hub_rows():
    """The pinned host scratch of the quotients supplied by the caller (later quotients are written in place), on a graph
    whose hub rows exceed kQuotLongRow (quot_insert_long_kernel) and are cut by batch borders; a workspace that is too
    small is ignored (the library pins its own)."""
    edges = [(h, j) for h in (0, 1, 2) for j in range(3, 9003)] + [(j, j + 1) for j in range(3, 9002)] + \
            [(j, 0) for j in range(100, 4700)]
    g = gg.from_edge_list(9003, edges)
    n, rp, ci, wt = g.numpy()
    cap = 5000
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rp, ci, wt, cap)
    rp_p, col_p = g.row_ptr.pin_memory(), g.col.pin_memory()
    hws = torch.empty(wl.wl_refine_batched_host_bytes(n, g.m), dtype=torch.uint8).pin_memory()
    small = torch.empty(64, dtype=torch.uint8).pin_memory()
    for ws in (hws, small, None):
        res = wl.wl_refine_batched(n, rp_p, col_p, None, max_batch_edges=cap, seed=9, host_workspace=ws)
        assert res.colors.numpy().tolist() == want.tolist()
        assert res.stats["outer_iters"] == outer_want and res.stats["last_num_batches"] == nbl_want
    assert oracle.is_stable(n, rp, ci, wt, res.colors.numpy())


def test_batched_validation_reaches_cut_rows_and_host_offsets():
    """S0 in the batched path: a bad target inside a row that is CUT by a batch border (a boundary node: refine_core never
    sees that row, the quotient pass maps it through the block map), malformed host offsets, and a weighted cut row whose
    sum reaches 2^32 (Theorem 1's precondition, L129) must come back as WL_EINVAL / WL_ERANGE, never as a CUDA fault."""
    g = BATCH_GRAPHS["hub"]()  # row 0 has 3000 entries; cap 1000 cuts it twice
    n, m = g.n, g.m
    for pos, val in ((1500, n + 5), (2999, -4), (10, n)):
        bad = g.col.clone()
        bad[pos] = val
        with pytest.raises(wl.WlError) as e:
            wl.wl_refine_batched(n, g.row_ptr, bad, None, max_batch_edges=1000, seed=1)
        assert e.value.code == wl.WL_EINVAL
    for mutate in (lambda rp: rp.__setitem__(5, int(rp[6]) + 1), lambda rp: rp.__setitem__(0, 1)):
        rp2 = g.row_ptr.clone()
        mutate(rp2)
        with pytest.raises(wl.WlError) as e:
            wl.wl_refine_batched(n, rp2, g.col, None, max_batch_edges=1000, seed=1)
        assert e.value.code == wl.WL_EINVAL
    w = torch.ones(m, dtype=torch.int64)
    w[:3000] = 1 << 21  # 3000 * 2^21 > 2^32 on the cut row
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, g.row_ptr, g.col, w, max_batch_edges=1000, seed=1)
    assert e.value.code == wl.WL_ERANGE
    w[:3000] = 1 << 20  # 3000 * 2^20 < 2^32: fine, and equal to the CPU Algorithm 2
    nn, rp, ci, _ = g.numpy()
    want, _, _, _ = oracle.rbsc(nn, rp, ci, w.numpy().astype(np.uint32), 1000)
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, w, max_batch_edges=1000, seed=1)
    assert res.colors.numpy().tolist() == want.tolist()


@pytest.mark.parametrize("name", ["rmat11_dir", "weighted", "hub", "grid"])
@pytest.mark.parametrize("flags", [0, 4096])
@pytest.mark.parametrize("extra", [False, True])
def test_batched_consume_input_overwrites_the_column_array(name, flags, extra):
    """WL_FLAG_CONSUME_INPUT: the first quotient is written over the caller's column (and weight) array; the scratch holds no
    column array.  Same colouring as without the flag (bit-exact against the CPU Algorithm 2); the input array is clobbered."""
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    cap = max(1, -(-g.m // 5))
    want, k_want, outer_want, _ = oracle.rbsc(n, rp, ci, wt, cap, inherit=bool(flags))
    col = g.col.clone().pin_memory()
    w = None if g.weights is None else g.weights.clone()
    w32 = None if w is None else (w & 0xFFFFFFFF).to(torch.uint32).pin_memory()
    # extra: room for the overflow lists of the one-byte weights behind the arrays (else the library pins them itself)
    hws_bytes = wl.wl_refine_batched_host_bytes_consume(n, g.m, w is not None)
    assert hws_bytes < wl.wl_refine_batched_host_bytes(n, g.m)
    hws = torch.empty(hws_bytes + (wl.wl_refine_batched_host_overflow_bytes(g.m) if extra else 0), dtype=torch.uint8).pin_memory()
    res = wl.wl_refine_batched(n, g.row_ptr.pin_memory(), col, w32, max_batch_edges=cap, seed=3,
                               flags=flags | wl.WL_FLAG_CONSUME_INPUT, host_workspace=hws)
    assert res.colors.numpy().tolist() == want.tolist() and res.stats["outer_iters"] == outer_want
    if outer_want >= 2 and k_want < n:
        assert not torch.equal(col, g.col)  # the quotient really went over the input
    # the same from initial classes
    init = gg.random_partition(n, 3, 4)
    want_i, _, outer_i, _ = oracle.rbsc(n, rp, ci, wt, cap, inherit=bool(flags), init=init.numpy())
    col.copy_(g.col)
    if w32 is not None:
        w32.copy_((w & 0xFFFFFFFF).to(torch.uint32))
    res = wl.wl_refine_batched(n, g.row_ptr.pin_memory(), col, w32, max_batch_edges=cap, seed=3,
                               flags=flags | wl.WL_FLAG_CONSUME_INPUT, host_workspace=hws, init_colors=init)
    assert res.colors.numpy().tolist() == want_i.tolist() and res.stats["outer_iters"] == outer_i


def _heavy_multigraph():
    # duplicate CSR entries add (Q10): six classes of ten twin nodes, each twin points 254 + c times to each of the five sinks of
    # its class -> quotient weights 254, 255, 256, ... and their multiples: the escape value of the compressed weights and its
    # neighbours, nearly every entry in the overflow lists; several outer iterations are needed to merge the twins across batches
    edges = []
    for c in range(6):
        for l in range(10):
            for r in range(5):
                edges += [(c * 10 + l, 60 + c * 5 + r)] * (254 + c)
    edges += [(60, 61)] * 3
    return gg.from_edge_list(90, edges)


@pytest.mark.parametrize("flags", [0, 4096, 1 << 29, (1 << 29) | 4096])
@pytest.mark.parametrize("nb", [3, 7, 20])
def test_batched_compressed_weights_with_heavy_entries(flags, nb):
    """Quotient weights travel as one byte + overflow lists (unweighted inputs).  A multigraph whose quotient weights are all
    >= 255 (and some exactly 254 / 255 / 256 / 300k), with inherited and re-cut batches, and with the device-side overflow list
    shrunk to 2 entries so that the fallback to uint32 weights runs: bit-exact against the CPU Algorithm 2 every time."""
    for g in (_heavy_multigraph(), BATCH_GRAPHS["hub"](), BATCH_GRAPHS["rmat10_sym"]()):
        n, rp, ci, wt = g.numpy()
        cap = max(1, -(-g.m // nb))
        want, k_want, outer_want, _ = oracle.rbsc(n, rp, ci, wt, cap, inherit=bool(flags & 4096))
        res = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=5, flags=flags)
        assert res.colors.numpy().tolist() == want.tolist() and res.stats["outer_iters"] == outer_want
        assert oracle.is_stable(n, rp, ci, wt, res.colors.numpy())
        # the same with the overflow lists inside a caller's host workspace (room behind its arrays), and a workspace that is
        # one byte short of holding them (the library then pins the lists itself)
        need = wl.wl_refine_batched_host_bytes(n, g.m)
        for hws_bytes in (need, need + wl.wl_refine_batched_host_overflow_bytes(g.m), need - 1):
            hws = torch.empty(hws_bytes, dtype=torch.uint8).pin_memory()
            res = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=5, flags=flags, host_workspace=hws)
            assert res.colors.numpy().tolist() == want.tolist() and res.stats["outer_iters"] == outer_want
        # and from initial classes
        init = gg.random_partition(n, 3, nb)
        want_i, _, outer_i, _ = oracle.rbsc(n, rp, ci, wt, cap, inherit=bool(flags & 4096), init=init.numpy())
        res = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=5, flags=flags, init_colors=init)
        assert res.colors.numpy().tolist() == want_i.tolist() and res.stats["outer_iters"] == outer_i


@pytest.mark.parametrize("flags", [0, 4096, 2048])
def test_batched_with_a_caller_device_arena(flags):
    """wl_options.device_workspace: every device buffer of the call is cut from the caller's arena (no cudaMalloc / cudaFree:
    the driver's free-memory count does not move during the call); a small or misaligned arena only means that some buffers
    are allocated as before.  Same colouring either way."""
    g = gg.rmat(13, seed=5, symmetrize=False)
    n = g.n
    cap = -(-g.m // 6)
    want = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=1, flags=flags)
    hws = torch.empty(wl.wl_refine_batched_host_bytes(n, g.m), dtype=torch.uint8, pin_memory=True)
    out = torch.empty(n, dtype=torch.int32, pin_memory=True)
    arena = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=1, flags=flags, device_workspace=arena,
                         host_workspace=hws, out=out)  # (first call: module loading and the library's pinned scalars)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    lows = []
    for seed in (1, 2):
        got = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=seed, flags=flags, device_workspace=arena,
                                   host_workspace=hws, out=out)
        lows.append(torch.cuda.mem_get_info()[0])
        assert got.colors.tolist() == want.colors.tolist() and got.stats["outer_iters"] == want.stats["outer_iters"]
    assert lows == [free0, free0]
    for small in (arena[:1 << 20], arena[3:(1 << 22) + 3], arena[:100]):
        got = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=3, flags=flags, device_workspace=small)
        assert got.colors.tolist() == want.colors.tolist()
    # the cap is still the cap
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=1, flags=flags, device_workspace=arena,
                             device_cap_bytes=4 * n)
    assert e.value.code == wl.WL_ENOMEM
    # the other forms and options draw from the arena too: COO batches, initial classes, caller-supplied slices
    if flags == 0:
        eb = gg.random_edge_batches(g, 3, 7)
        coo = gg.coo_batches(g, eb, 3)
        a = wl.wl_refine_batched(n, None, None, None, max_batch_edges=cap, seed=1, coo_batches=coo)
        b = wl.wl_refine_batched(n, None, None, None, max_batch_edges=cap, seed=1, coo_batches=coo, device_workspace=arena)
        assert a.colors.tolist() == b.colors.tolist() and a.stats["outer_iters"] == b.stats["outer_iters"]
    init = gg.random_partition(n, 4, 2)
    a = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=1, flags=flags, init_colors=init)
    b = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=1, flags=flags, init_colors=init,
                             device_workspace=arena)
    assert a.colors.tolist() == b.colors.tolist() and a.stats["outer_iters"] == b.stats["outer_iters"]


def test_batched_device_cap_is_checked_for_every_allocation():
    """A cap that admits the buffers of the local-refinement pass but not those of the quotient pass must give WL_ENOMEM
    (a failed allocation used to be overwritten by the next successful one)."""
    g = gg.rmat(12, seed=5, symmetrize=False)
    cap_edges = g.m // 4 + 1
    ok = wl.wl_refine_batched(g.n, g.row_ptr, g.col, None, max_batch_edges=cap_edges, seed=1)
    assert ok.stats["outer_iters"] >= 2
    # bisect the smallest cap that works; every smaller cap must fail cleanly with WL_ENOMEM, never with a CUDA error
    lo, hi = 4096, 1 << 30
    while hi - lo > 4096:
        mid = (lo + hi) // 2
        try:
            r = wl.wl_refine_batched(g.n, g.row_ptr, g.col, None, max_batch_edges=cap_edges, seed=1, device_cap_bytes=mid)
            assert r.colors.tolist() == ok.colors.tolist()
            hi = mid
        except wl.WlError as e:
            assert e.code == wl.WL_ENOMEM
            lo = mid
    assert hi < (1 << 30)


def test_batched_batch_cap_derived_from_device_cap():
    """max_batch_edges <= 0: M_b comes from the device cap (the shape of configs[4]: a cap forces the batching).  The run must
    stay under the cap (every allocation is checked), use several batches, and give a stable refinement of the coarsest
    colouring; without a cap the request is invalid."""
    g = gg.rmat(14, seed=6, symmetrize=False)
    n, rp, ci, wt = g.numpy()
    coarsest, _, _ = oracle.refine(n, rp, ci)
    for cap in (6 << 20, 12 << 20):
        res = wl.wl_refine_batched(n, g.row_ptr, g.col, None, device_cap_bytes=cap, seed=2)
        got = res.colors.numpy()
        assert oracle.is_stable(n, rp, ci, None, got) and refines(got, coarsest)
        assert res.stats["outer_iters"] >= 2  # more than one batch: the graph did not fit the cap
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, g.row_ptr, g.col, None, seed=2)
    assert e.value.code == wl.WL_EINVAL
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(n, g.row_ptr, g.col, None, device_cap_bytes=1 << 16, seed=2)
    assert e.value.code == wl.WL_ENOMEM


@pytest.mark.parametrize("flags", [0, 4096])
def test_batched_composed_map_on_the_host_under_a_tight_cap(flags):
    """When the composed map of the original nodes (4 B per node) would take more than an eighth of the device cap it stays in
    out_colors and passes through the device in tiles: same colouring as the uncapped run, stable, refines the coarsest."""
    g = gg.rmat(17, seed=4, symmetrize=False)
    n, rp, ci, wt = g.numpy()
    cap = 32 * n - 1
    free = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=8000, seed=1, flags=flags)
    tight = wl.wl_refine_batched(n, g.row_ptr, g.col, None, max_batch_edges=8000, seed=2, flags=flags, device_cap_bytes=cap)
    assert torch.equal(free.colors, tight.colors) and tight.stats["outer_iters"] == free.stats["outer_iters"] >= 3
    got = tight.colors.numpy()
    coarsest, _, _ = oracle.refine(n, rp, ci)
    assert oracle.is_stable(n, rp, ci, None, got) and refines(got, coarsest)


def test_batched_device_cap_and_limits():
    g = gg.rmat(10, seed=1)
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_batched(g.n, g.row_ptr, g.col, None, max_batch_edges=g.m // 4, device_cap_bytes=4096)
    assert e.value.code == wl.WL_ENOMEM
    res = wl.wl_refine_batched(g.n, g.row_ptr, g.col, None, max_batch_edges=g.m // 4, max_outer_iters=1, allow_limit=True)
    n, rp, ci, wt = g.numpy()
    assert oracle.is_stable(n, rp, ci, wt, res.colors.numpy())  # every outer iteration ends on a stable colouring


@pytest.mark.parametrize("name", ["rmat11_dir", "weighted", "hub"])
def test_batched_with_edge_balanced_local_rsc(name):
    """Local RSC through the edge-balanced kernel: batch slices start at arbitrary entry positions (shifted column pointer,
    unaligned origin) and targets outside V_k are implicit singletons."""
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    cap = max(1, g.m // 3 + 1)
    want, k_want, _, _ = oracle.rbsc(n, rp, ci, wt, cap)
    res = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=5, flags=wl.WL_FLAG_EDGE_BALANCED)
    assert res.colors.numpy().tolist() == want.tolist() and res.num_colors == k_want


def test_batched_seed_independence():
    g = gg.rmat(10, seed=6, symmetrize=False)
    a = wl.wl_refine_batched(g.n, g.row_ptr, g.col, None, max_batch_edges=g.m // 5, seed=1).colors
    b = wl.wl_refine_batched(g.n, g.row_ptr, g.col, None, max_batch_edges=g.m // 5, seed=2).colors
    assert torch.equal(a, b)


# ------------------------------------------------------------------ batch-level sharding over ranks (sharded.py)
@pytest.mark.parametrize("name", list(BATCH_GRAPHS))
@pytest.mark.parametrize("nb", [2, 5, 16])
def test_sharded_driver_with_cuda_backend_equals_cpu_algorithm2(name, nb):
    """The sharded driver with the CUDA backend (wl_refine_inner / wl_quotient_rows per batch on device buffers), 1 to 3 virtual
    ranks played in lock step on this one GPU (the collectives are host-level; the ranks never wait on each other inside a
    kernel): bit-exact against the CPU Algorithm 2 with inherited batches and against wl_refine_batched(INHERIT)."""
    import os
    import sys
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from sharded_harness import run_lockstep
    from paper_2607_02603_b200.sharded import CudaBackend
    g = BATCH_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    cap = max(1, -(-g.m // nb))
    want, k_want, outer_want, _ = oracle.rbsc(n, rp, ci, wt, cap, inherit=True)
    single = wl.wl_refine_batched(n, g.row_ptr, g.col, g.weights, max_batch_edges=cap, seed=1, flags=wl.WL_FLAG_INHERIT_BATCHES)
    assert single.colors.numpy().tolist() == want.tolist()
    for world in (1, 2, 3):
        got, k, outer, ranks = run_lockstep(lambda: CudaBackend(dev()), n, g.row_ptr, g.col, g.weights, cap, world, seed=world)
        assert got.numpy().tolist() == want.tolist(), (name, nb, world)
        assert k == k_want and outer == outer_want


def test_refine_batched_sharded_single_process_entry_point():
    from paper_2607_02603_b200.sharded import refine_batched_sharded
    g = gg.rmat(12, seed=8, symmetrize=False)
    n, rp, ci, wt = g.numpy()
    cap = g.m // 7 + 1
    want, k_want, outer_want, _ = oracle.rbsc(n, rp, ci, wt, cap, inherit=True)
    colours, k, outer = refine_batched_sharded(n, g.row_ptr, g.col, None, max_batch_edges=cap, seed=4, device=dev())
    assert colours.numpy().tolist() == want.tolist() and k == k_want and outer == outer_want


@pytest.mark.parametrize("seed", range(5))
def test_per_batch_device_calls_match_the_definitions(seed):
    """wl_refine_inner (B3 + B4 of one batch: inner nodes one block, every outside target an implicit singleton, ids in
    first-occurrence order) and wl_quotient_rows (Def. 4 for the representatives among a node range) against the oracle-made
    backend of the sharded tests, on a node range in the middle of a graph."""
    import os
    import sys
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from sharded_harness import OracleBackend
    g = gg.rmat(10, edge_factor=6, seed=seed, symmetrize=bool(seed % 2)) if seed < 4 else gg.random_weighted_digraph(600, 5000, seed, max_w=4)
    n = g.n
    lo, hi = n // 5, n // 5 + n // 2
    a, b = int(g.row_ptr[lo]), int(g.row_ptr[hi])
    rp = (g.row_ptr[lo:hi + 1] - a).contiguous()
    col = g.col[a:b].contiguous()
    wt = None if g.weights is None else g.weights[a:b].contiguous()
    ob = OracleBackend()
    want_c, want_f, want_k = ob.refine_inner(rp, 0, col, wt, lo, n, 0, 0)
    c, f, k = wl.wl_refine_inner(rp.to(dev()), col.to(dev()), None if wt is None else wt.to(dev()), lo, n, seed=seed)
    assert k == want_k and c.cpu().tolist() == want_c.tolist() and f.cpu().tolist() == want_f.tolist()
    # a block map of the whole graph: the inner range keeps its local blocks, everybody else is a singleton
    block_of = torch.empty(n, dtype=torch.int32)
    block_of[:lo] = torch.arange(lo, dtype=torch.int32)
    block_of[lo:hi] = want_c + lo
    block_of[hi:] = torch.arange(n - hi, dtype=torch.int32) + lo + k
    ob.set_block_map(block_of)
    h_rp, _, h_col, h_wt = ob.host_buffers(k, col.numel())
    qm = ob.quotient_rows(rp, 0, col, wt, lo, want_f, lo, k, h_rp[1:], h_col, h_wt, 0)
    h_rp[0] = 0
    wr, wc, ww = h_rp[:k + 1], h_col[:qm], torch.from_numpy(h_wt[:qm].numpy().view(np.uint32).astype(np.int64))
    qr, qc, qw = wl.wl_quotient_rows(rp.to(dev()), col.to(dev()), None if wt is None else wt.to(dev()), lo, block_of.to(dev()),
                                     f, lo, k)
    assert qr.cpu().tolist() == wr.tolist()
    assert _rows_as_dicts(k, qr.cpu().numpy(), qc.cpu().numpy(), qw.cpu().numpy()) == _rows_as_dicts(k, wr.numpy(), wc.numpy(), ww.numpy())
    with pytest.raises(wl.WlError) as e:  # the range does not fit the node count
        wl.wl_refine_inner(rp.to(dev()), col.to(dev()), None, n, n, seed=1)
    assert e.value.code == wl.WL_EINVAL


def _sharded_cuda_worker(rank, world, port, q):
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    import torch.distributed as dist
    from paper_2607_02603_b200.sharded import refine_batched_sharded
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    out = {}
    for name in ("rmat11_dir", "weighted", "hub"):
        g = BATCH_GRAPHS[name]()
        cap = max(1, g.m // 6 + 1)
        colours, k, outer = refine_batched_sharded(g.n, g.row_ptr.pin_memory(), g.col.pin_memory(),
                                                   None if g.weights is None else g.weights.pin_memory(), max_batch_edges=cap,
                                                   seed=3 + rank, dist=dist, device=torch.device("cuda", 0))
        out[name] = (colours.tolist(), k, outer)
    dist.barrier()
    q.put((rank, out))
    dist.destroy_process_group()


def test_sharded_two_processes_with_cuda_backend_over_gloo():
    """The real loop of the sharded driver (run(): all-gather of the block counts, all-gather-v of the block-map slices that
    live on the GPU) with the CUDA backend in TWO processes; both use this one GPU and talk over gloo (host-level collectives
    only: no kernel of one rank ever waits for the other).  Both ranks must end with the colouring of the CPU Algorithm 2."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 32500 + os.getpid() % 2000
    procs = [ctx.Process(target=_sharded_cuda_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=600) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for name in ("rmat11_dir", "weighted", "hub"):
        g = BATCH_GRAPHS[name]()
        n, rp, ci, wt = g.numpy()
        want, k_want, outer_want, _ = oracle.rbsc(n, rp, ci, wt, max(1, g.m // 6 + 1), inherit=True)
        for rank in (0, 1):
            colours, k, outer = res[rank][name]
            assert colours == want.tolist() and k == k_want and outer == outer_want, (name, rank)
