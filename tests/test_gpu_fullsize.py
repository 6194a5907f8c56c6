"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times.
C1: element by element against the oracle.  C2 (2048^2 grid, 1024 rounds): the closed-form orbit colouring.
C3 (R-MAT scale 22): element by element against the oracle (finishes in ~10 s on the box's host cores).
C4 (R-MAT scale 27): the oracle cannot finish; properties that hold at any size + sampled blocks checked one by one
with the oracle's signature builder (stability, Def. 1) + the trajectory's structure."""
import numpy as np
import pytest
import torch

import graphgen as gg
import oracle

pytestmark = pytest.mark.gpu
wl = pytest.importorskip("paper_2607_02603_b200")


def dev():
    return torch.device("cuda", 0)


def test_c1_er_equals_oracle():
    g = gg.erdos_renyi()
    n, rp, ci, wt = g.numpy()
    want, counts, rounds = oracle.refine(n, rp, ci)
    d = g.to(dev())
    mism = 0
    for seed in range(100):
        res = wl.wl_refine(n, d.row_ptr, d.col, seed=seed)
        if res.colors.cpu().numpy().tolist() != want.tolist() or res.round_colors != counts:
            mism += 1
    # Theorem 1: error probability <= 1e-9 per run; expected mismatches over 100 seeds: 0
    assert mism == 0


def test_c2_grid_2048_closed_form():
    s = 2048
    g = gg.grid2d(s, device=dev())
    res = wl.wl_refine(g.n, g.row_ptr, g.col, seed=11)
    assert res.rounds == 1024 and res.num_colors == 524800  # tests/golden/grid_closed_form.txt
    assert torch.equal(res.colors.cpu(), gg.grid2d_orbit_colors(s))


def test_c3_rmat22_equals_oracle():
    g = gg.rmat(22, seed=1, device=dev())
    n, rp, ci, wt = g.numpy()
    want, counts, rounds = oracle.refine(n, rp, ci)
    assert oracle.is_stable(n, rp, ci, None, want)
    for seed, flags in ((1, 0), (2, 2)):
        res = wl.wl_refine(g.n, g.row_ptr, g.col, seed=seed, flags=flags)
        assert res.round_colors == counts and res.rounds == rounds
        assert (res.colors.cpu().numpy() == want).all()
    # the host-buffer entry point at the same size
    res = wl.wl_refine_host(n, g.row_ptr.cpu().pin_memory(), g.col.cpu().pin_memory(), seed=3)
    assert (res.colors.numpy() == want).all()


def test_c4_rmat27_properties_and_sampled_stability():
    g = gg.rmat(27, seed=2, device=dev(), chunk=1 << 28)
    torch.cuda.empty_cache()
    n, m = g.n, g.m
    assert n == 1 << 27 and m > (1 << 31)  # 64-bit offsets are exercised
    res = wl.wl_refine(n, g.row_ptr, g.col, seed=2027)
    res2 = wl.wl_refine(n, g.row_ptr, g.col, seed=5, flags=wl.WL_FLAG_NO_PRUNE)
    c = res.colors
    # (1) seed and pruning independence of the whole result, (2) same trajectory
    assert torch.equal(c, res2.colors) and res.round_colors == res2.round_colors
    # (3) monotone trajectory that ends with a confirming round; canonical first-occurrence ids
    rc = res.round_colors
    assert all(a <= b for a, b in zip(rc, rc[1:])) and rc[-1] == rc[-2] == res.num_colors
    assert int(c.max()) + 1 == res.num_colors and int(c[0]) == 0
    first_seen = torch.zeros(res.num_colors, dtype=torch.bool, device=dev())
    # canonical: the running maximum of the ids grows by at most one per node
    cm = torch.cummax(c.to(torch.int64), 0).values
    assert bool(((cm[1:] - cm[:-1]) <= 1).all())
    del first_seen, cm
    # (4) round 1 separates exactly the out-degrees (round-1 closed form z = outdeg * w0)
    deg = g.row_ptr[1:] - g.row_ptr[:-1]
    assert rc[0] == int(torch.unique(deg).numel())
    # (5) nodes of one block have equal degree (necessary for stability), checked on ALL nodes:
    #     max and min degree per block coincide
    k = res.num_colors
    dmax = torch.zeros(k, dtype=torch.int64, device=dev()).scatter_reduce_(0, c.to(torch.int64), deg, "amax", include_self=False)
    dmin = torch.zeros(k, dtype=torch.int64, device=dev()).scatter_reduce_(0, c.to(torch.int64), deg, "amin", include_self=False)
    assert bool((dmax == dmin).all())
    del dmax, dmin
    # (6) Def. 1 on sampled non-singleton blocks, one by one with the oracle: build the subgraph made of the rows of the
    #     sampled nodes (targets renamed to their colours' representatives is not needed: is_stable only reads colours of targets)
    sizes = torch.bincount(c.to(torch.int64), minlength=k)
    multi = torch.nonzero((sizes >= 2) & (sizes <= 64)).flatten()
    pick = multi[torch.randperm(multi.numel(), device=dev(), generator=torch.Generator(device=dev()).manual_seed(0))[:300]]
    member = torch.isin(c.to(torch.int64), pick)
    nodes = torch.nonzero(member).flatten()
    assert nodes.numel() >= 600
    # rows of the sampled nodes with targets replaced by their colour (what Def. 1 sums over)
    a, b = g.row_ptr[nodes], g.row_ptr[nodes + 1]
    lens = (b - a)
    starts = torch.repeat_interleave(a, lens)
    offs = torch.arange(int(lens.sum()), device=dev()) - torch.repeat_interleave(torch.cumsum(lens, 0) - lens, lens)
    tgt_col = c[g.col[starts + offs].to(torch.int64)]
    # tiny CSR: node t = sampled node t, targets = colour ids (as node ids of a graph whose colouring is the identity on them)
    kk = int(tgt_col.max()) + 1 if tgt_col.numel() else 1
    nn = nodes.numel()
    sub_rp = torch.zeros(nn + 1, dtype=torch.int64)
    sub_rp[1:] = torch.cumsum(lens.cpu(), 0)
    # colouring of the auxiliary graph: sampled nodes keep their block id (offset past the target ids), targets are discrete
    sub_n = nn + kk
    rp_full = torch.cat([sub_rp, torch.full((kk,), int(sub_rp[-1]), dtype=torch.int64)])
    col_full = (tgt_col.cpu().to(torch.int64) + nn).to(torch.int32)
    colours = torch.cat([c[nodes].cpu().to(torch.int64) + kk + nn, torch.arange(kk) + nn]).to(torch.int64)
    colours = gg.canonical_first_occurrence(colours)
    assert oracle.is_stable(sub_n, rp_full.numpy(), col_full.numpy(), None, colours.numpy())
    # sanity of the checker itself on this data: moving one sampled node into another sampled block must break it
    bad = colours.clone()
    other = int(torch.nonzero(colours[:nn] != colours[0])[0])
    if lens[0] != lens[other]:
        bad[0] = colours[other]
        assert not oracle.is_stable(sub_n, rp_full.numpy(), col_full.numpy(), None, bad.numpy())


def test_c5_shape_batched_rmat20_directed():
    """The shape of configs[4] at a size the oracle finishes: directed R-MAT scale 20 (1.05 M nodes, ~16 M edges) in pinned
    host memory, 16 batches, caller-supplied pinned scratch.  Theorem 2 (stable on the original graph), L165 (refines the
    coarsest colouring), seed independence, and bit-exact agreement with the CPU Algorithm 2 on the same edge partition."""
    from helpers import refines
    g = gg.rmat(20, seed=3, symmetrize=False, device=dev())
    n, m = g.n, g.m
    rp, col = g.row_ptr.cpu().pin_memory(), g.col.cpu().pin_memory()
    hws = torch.empty(wl.wl_refine_batched_host_bytes(n, m), dtype=torch.uint8).pin_memory()
    cap = m // 16 + 1
    res = wl.wl_refine_batched(n, rp, col, None, max_batch_edges=cap, seed=1, host_workspace=hws, device_cap_bytes=2 << 30)
    res2 = wl.wl_refine_batched(n, rp, col, None, max_batch_edges=cap, seed=77, host_workspace=hws)
    assert res.stats["outer_iters"] >= 2 and res.stats["bytes_h2d"] > 2 * 4 * m
    assert torch.equal(res.colors, res2.colors)
    got = res.colors.numpy()
    rpn, cin = rp.numpy(), col.numpy()
    assert oracle.is_stable(n, rpn, cin, None, got)
    coarsest, _, _ = oracle.refine(n, rpn, cin)
    assert refines(got, coarsest) and res.num_colors >= int(coarsest.max()) + 1
    want, k_want, outer_want, nbl_want = oracle.rbsc(n, rpn, cin, None, cap)
    assert res.num_colors == k_want and res.stats["outer_iters"] == outer_want
    assert (got == want).all()
