"""Test-only helpers that are independent of BOTH the oracle and the CUDA path: dense numpy
restatements of the paper's definitions, used to pin the oracle."""
import itertools

import numpy as np


def dense_adj(n, rp, ci, wt=None):
    """A in N_0^{n x n}; duplicate entries add."""
    A = np.zeros((n, n), dtype=np.int64)
    for i in range(n):
        for e in range(rp[i], rp[i + 1]):
            A[i, ci[e]] += 1 if wt is None else int(wt[e])
    return A


def indicator(colors):
    colors = np.asarray(colors)
    k = int(colors.max()) + 1 if colors.size else 0
    S = np.zeros((colors.size, k), dtype=np.int64)
    S[np.arange(colors.size), colors] = 1
    return S


def stable_dense(A, colors):
    """Def. 1 (L47-L49) literally: rows of A.S are equal inside every block."""
    AS = A @ indicator(colors)
    colors = np.asarray(colors)
    for b in np.unique(colors):
        rows = AS[colors == b]
        if not (rows == rows[0]).all():
            return False
    return True


def set_partitions(n):
    """All set partitions of range(n) as restricted-growth strings."""
    def rec(prefix, mx):
        if len(prefix) == n:
            yield tuple(prefix)
            return
        for v in range(mx + 2):
            yield from rec(prefix + [v], max(mx, v))
    if n == 0:
        yield ()
        return
    yield from rec([0], 0)


def refines(fine, coarse):
    """every block of `fine` lies inside one block of `coarse` (Def. 2)."""
    fine, coarse = np.asarray(fine), np.asarray(coarse)
    m = {}
    for f, c in zip(fine.tolist(), coarse.tolist()):
        if m.setdefault(f, c) != c:
            return False
    return True


def brute_force_coarsest(A, init):
    """Def. 3 (L57) + L94 by exhaustion: among all partitions that refine `init` and are stable, the one with
    the fewest blocks; asserts it is unique and that every other stable refinement of init refines it."""
    n = A.shape[0]
    stable = [p for p in set_partitions(n) if refines(p, init) and stable_dense(A, p)]
    assert stable, "the discrete partition is always stable"
    kmin = min(max(p) + 1 for p in stable)
    best = [p for p in stable if max(p) + 1 == kmin]
    assert len(best) == 1
    for p in stable:
        assert refines(p, best[0])
    return np.array(best[0], dtype=np.int32)  # restricted growth string == first-occurrence numbering


def same_partition(a, b):
    return refines(a, b) and refines(b, a)


def classify(got, want):
    """Reading Q12: RSC separates two nodes only if their z differ, and equal signatures force equal z, so
    every RSC partition is coarser than or equal to the exact one.  A randomized collision can therefore only show up as
    "coarser": the exact colouring `want` strictly refines `got`.  Anything else ("other") is a bug, never a collision."""
    if same_partition(got, want):
        return "equal"
    return "coarser" if refines(want, got) else "other"


def split_pairs(prev, cur):
    """N_r of DESIGN.md's union bound: sum over the blocks B of `prev` of C(s_B, 2), s_B = number of blocks of `cur` inside B
    (the pairs of sub-blocks whose z must differ for the round to be computed exactly)."""
    prev, cur = np.asarray(prev, dtype=np.int64), np.asarray(cur, dtype=np.int64)
    pairs = np.unique(np.stack([prev, cur], 1), axis=0)
    s = np.bincount(pairs[:, 0])
    return int((s * (s - 1) // 2).sum())


def sampled_block_stability(row_ptr, col, colors, k, dev, n_blocks=300, max_block=64, max_row=20000, seed=0, min_row=0):
    """Def. 1 on sampled non-singleton blocks of a colouring too large for a full check: the rows of every
    member of the sampled blocks are cut out (row_ptr / col may live on the host or on `dev`), their targets are replaced by
    the targets' colours, and oracle.is_stable runs on that auxiliary graph (sampled nodes keep their block, the target
    colours are discrete).  Also checks, on ALL nodes, that the members of a block have equal out-degree (necessary for
    stability).  min_row: only blocks whose members have at least that many entries (most non-singleton blocks of an R-MAT
    graph are twins with a single out-edge; a second sample with min_row > 1 looks at the others).  Returns (blocks checked, nodes checked, entries checked, verdict, verdict of a planted violation or None)."""
    import torch
    import graphgen as gg
    import oracle
    n = colors.numel()
    c = colors.to(dev)
    c64 = c.to(torch.int64)
    sizes = torch.bincount(c64, minlength=k)
    rpd = row_ptr.to(dev)
    deg = rpd[1:] - rpd[:-1]
    del rpd
    dmax = torch.zeros(k, dtype=torch.int64, device=dev).scatter_reduce_(0, c64, deg, "amax", include_self=False)
    dmin = torch.zeros(k, dtype=torch.int64, device=dev).scatter_reduce_(0, c64, deg, "amin", include_self=False)
    degrees_equal = bool((dmax == dmin).all())
    multi = torch.nonzero((sizes >= 2) & (sizes <= max_block) & (dmax <= max_row) & (dmax >= min_row)).flatten()
    del dmin, sizes
    gen = torch.Generator(device=dev).manual_seed(seed)
    pick = multi[torch.randperm(multi.numel(), device=dev, generator=gen)[:n_blocks]]
    lut = torch.zeros(k, dtype=torch.bool, device=dev)
    lut[pick] = True
    nodes = torch.nonzero(lut[c64]).flatten()
    del lut, c64, dmax
    nn = nodes.numel()
    if nn == 0:  # no block of the asked shape exists
        return {"blocks": 0, "nodes": 0, "entries": 0, "stable": True, "degrees_equal_on_all_nodes": degrees_equal,
                "planted_violation_passes": None, "candidate_blocks": 0}
    n_candidates = int(multi.numel())
    nodes_rp = nodes.to(row_ptr.device)
    a, b = row_ptr[nodes_rp], row_ptr[nodes_rp + 1]
    lens = (b - a)
    total = int(lens.sum())
    starts = torch.repeat_interleave(a, lens)
    offs = torch.arange(total, device=a.device) - torch.repeat_interleave(torch.cumsum(lens, 0) - lens, lens)
    targets = col[(starts + offs).to(col.device)].to(dev).to(torch.int64)
    tgt_col = c[targets].to(torch.int64)
    sub_rp = torch.zeros(nn + 1, dtype=torch.int64)
    sub_rp[1:] = torch.cumsum(lens.cpu(), 0)
    # nodes of the auxiliary graph: the sampled nodes, then one node per distinct target colour (compressed: the colour ids of
    # a billion-node graph plus the sample would not fit int32 node ids)
    uniq, inv = torch.unique(tgt_col.cpu(), return_inverse=True)
    kk2 = uniq.numel()
    sub_n = nn + kk2
    rp_full = torch.cat([sub_rp, torch.full((kk2,), int(sub_rp[-1]), dtype=torch.int64)])
    col_small = (inv + nn).to(torch.int32)
    colours = torch.cat([c[nodes].cpu().to(torch.int64) + (nn + kk2), torch.arange(kk2) + nn]).to(torch.int64)
    colours = gg.canonical_first_occurrence(colours)
    ok = bool(oracle.is_stable(sub_n, rp_full.numpy(), col_small.numpy(), None, colours.numpy()))
    # the checker must notice a node moved into a block whose members see other colours: take the first sampled node of
    # another block whose row (as a sorted list of target colours) differs from node 0's
    planted = None
    rows_np, col_np = sub_rp.numpy(), col_small.numpy()
    sig0 = sorted(col_np[rows_np[0]:rows_np[1]].tolist())
    for t in torch.nonzero(colours[:nn] != colours[0]).flatten()[:2000].tolist():
        if sorted(col_np[rows_np[t]:rows_np[t + 1]].tolist()) != sig0:
            bad = colours.clone()
            bad[0] = colours[t]
            planted = bool(oracle.is_stable(sub_n, rp_full.numpy(), col_small.numpy(), None, bad.numpy()))
            break
    return {"blocks": int(pick.numel()), "nodes": nn, "entries": total, "stable": ok, "degrees_equal_on_all_nodes": degrees_equal,
            "planted_violation_passes": planted, "candidate_blocks": n_candidates}
