"""GPU parity tests: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle on the same
seeded inputs.  Integer / index work: bit exact (partitions compared after canonical first-occurrence relabelling)."""
import numpy as np
import pytest
import torch

import graphgen as gg
import oracle

pytestmark = pytest.mark.gpu

wl = pytest.importorskip("paper_2607_02603_b200")


def dev():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch.device("cuda", 0)


def dgraph(g):
    d = g.to(dev())
    return d.n, d.row_ptr, d.col, d.weights


def u64(t):
    return t.cpu().numpy().view(np.uint64)


def oracle_w(key, colors):
    return np.array([oracle.weight(key, int(c)) for c in colors], dtype=np.uint64)


GRAPHS = {
    "er_c1": lambda: gg.erdos_renyi(),
    "er_small": lambda: gg.erdos_renyi(300, 900, seed=3),
    "grid_33": lambda: gg.grid2d(33),
    "grid_64": lambda: gg.grid2d(64),
    "rmat12_sym": lambda: gg.rmat(12, seed=1),
    "rmat13_dir": lambda: gg.rmat(13, seed=2, symmetrize=False),
    "path_101": lambda: gg.path_graph(101),
    "dpath_40": lambda: gg.directed_path(40),
    "star_1000": lambda: gg.star_graph(1000),
    "hub_20000": lambda: gg.from_edge_list(20001, [(0, j) for j in range(1, 20001)] + [(5, 7), (9, 7)]),
    # two twin hubs (degree 10000 > the hub-chunk threshold) that stay in one block over many rounds, plus a directed
    # path among their targets so that refinement takes a few hundred rounds with the hubs still active
    "twin_hubs": lambda: gg.from_edge_list(10302, [(h, j) for h in (0, 1) for j in range(2, 10002)]
                                           + [(j, j + 1) for j in range(10002, 10301)] + [(2, 10002), (3, 10002)]),
    "k_5_7": lambda: gg.complete_bipartite(5, 7),
    "circ": lambda: gg.circulant(50, (1, 4, 9)),
    "empty_edges": lambda: gg.from_edge_list(17, []),
    "one_node": lambda: gg.from_edge_list(1, []),
    "self_loops": lambda: gg.from_edge_list(4, [(0, 0), (1, 1), (2, 3)]),
    # duplicate CSR entries add (Q10); many sinks, twins and repeated targets: the finality pruning (R5) sees blocks whose
    # members reach the same final colours through different nodes
    "multigraph": lambda: gg.from_edge_list(400, [((7 * t) % 130, 130 + (t * t) % 270) for t in range(1500)] +
                                            [(t % 130, (3 * t) % 130) for t in range(260)]),
    "weighted": lambda: gg.random_weighted_digraph(500, 3000, 5, max_w=4),
    "weighted_big_w": lambda: gg.random_weighted_digraph(200, 2000, 6, max_w=1 << 20),
}


# ------------------------------------------------------------------ S1+S2
@pytest.mark.parametrize("name", list(GRAPHS))
@pytest.mark.parametrize("flags", [0, 4, 32, 128, 128 | 32])
def test_spmv_bit_exact(name, flags):
    g = GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    colors = gg.random_partition(n, max(1, min(n // 3, 60000)), 11).numpy()
    key = wl.wl_round_key(123, 0, 2)
    assert key == oracle.round_key(123, 0, 2)
    want = oracle.spmv_u64(n, rp, ci, wt, oracle_w(key, colors))
    dn, drp, dci, dwt = dgraph(g)
    y = wl.wl_spmv_round(dn, drp, dci, dwt, torch.from_numpy(colors).to(dev()), key, flags=flags)
    assert (u64(y) == want).all()


@pytest.mark.parametrize("shift", [1, 2, 3])
@pytest.mark.parametrize("name", ["rmat12_sym", "hub_20000", "weighted", "empty_rows_mix"])
def test_spmv_edge_balanced_unaligned_columns(name, shift):
    """A column array that starts 4, 8 or 12 bytes past a 16-byte boundary (a slice of a larger buffer, as the batched
    path passes them) must give the same sums; graphs with runs of empty rows and rows crossing chunk borders."""
    if name == "empty_rows_mix":  # runs of empty rows at the start, in the middle and at the end; rows crossing 2048-entry chunks
        edges = [(i, (7 * i + j) % 9000) for i in range(100, 4000) for j in range(i % 5)] + \
                [(5000, j) for j in range(0, 9000, 2)] + [(8000 + i, i) for i in range(50)]
        g = gg.from_edge_list(9000, edges)
    else:
        g = GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    colors = gg.random_partition(n, max(1, n // 4), 5).numpy()
    key = wl.wl_round_key(77, 3, 9)
    want = oracle.spmv_u64(n, rp, ci, wt, oracle_w(key, colors))
    dn, drp, dci, dwt = dgraph(g)
    pad = torch.zeros(shift, dtype=torch.int32, device=dev())
    dci2 = torch.cat([pad, dci])[shift:]
    assert dci2.data_ptr() % 16 == 4 * shift
    y = wl.wl_spmv_round(dn, drp, dci2, dwt, torch.from_numpy(colors).to(dev()), key, flags=wl.WL_FLAG_EDGE_BALANCED)
    assert (u64(y) == want).all()


@pytest.mark.parametrize("name", ["weighted", "weighted_big_w", "rmat12_sym", "hub_20000", "twin_hubs", "multigraph"])
@pytest.mark.parametrize("narrow", [False, True])
def test_spmv_active_row_list_bit_exact(name, narrow):
    """Step-level S1+S2 with an ACTIVE ROW LIST (the kernels of the pruned rounds: rows != NULL), weighted and unweighted,
    32-bit and 16-bit colour ids, hub rows inside and outside the list: the listed entries of y equal the oracle's u64 SpMV,
    every other entry keeps the value it had."""
    g = GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    colors = gg.random_partition(n, max(1, min(n // 3, 60000)), 17).numpy()
    key = wl.wl_round_key(5, 2, 3)
    want = oracle.spmv_u64(n, rp, ci, wt, oracle_w(key, colors))
    dn, drp, dci, dwt = dgraph(g)
    for frac, sd in ((2, 1), (7, 2)):
        pick = torch.nonzero(gg.hash_u32(sd, torch.arange(n, dtype=torch.int64)) % frac == 0).flatten().to(torch.int32)
        if name in ("hub_20000", "twin_hubs") and sd == 2:
            pick = pick[pick != 0]  # the hub row (node 0) stays outside the list: its y must not be touched
        marker = 0x0123456789ABCDEF
        y = torch.full((n,), marker, dtype=torch.int64, device=dev())
        wl.wl_spmv_rows(dn, drp, dci, dwt, torch.from_numpy(colors).to(dev()), key, pick.to(dev()), y,
                        flags=wl.WL_FLAG_NARROW_COLORS if narrow else 0)
        got = u64(y)
        listed = np.zeros(n, dtype=bool)
        listed[pick.numpy()] = True
        assert (got[listed] == want[listed]).all()
        assert (got[~listed] == np.uint64(marker)).all()


@pytest.mark.parametrize("name", ["rmat12_sym", "rmat13_dir", "weighted", "grid_33", "twin_hubs", "multigraph", "er_c1"])
@pytest.mark.parametrize("flags", [0, 2, 1024, 512, 64, 256])
def test_refine_with_init_equals_oracle(name, flags):
    """Arbitrary initial partition (L94): sparse, non-dense labels, the output aliasing the init array.  Colours and the
    per-round colour counts equal the oracle's over the flag matrix (pruning, finality, worklist regime, per-round sync)."""
    g = GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    dn, drp, dci, dwt = dgraph(g)
    for k0, seed in ((2, 1), (7, 2), (max(2, n // 5), 3)):
        init = gg.random_partition(n, k0, seed)
        want, counts, rounds = oracle.refine(n, rp, ci, wt, init.numpy())
        labels = (init.to(torch.int64) * 1000003 % 2147483000).to(torch.int32).to(dev())  # sparse non-dense labels
        assert torch.unique(labels).numel() == torch.unique(init).numel()
        res = wl.wl_refine(dn, drp, dci, dwt, labels, seed=seed * 31, flags=flags, out=labels)  # out aliases init
        assert res.round_colors == counts and res.rounds == rounds
        assert res.colors.cpu().numpy().tolist() == want.tolist()
        assert res.colors.data_ptr() == labels.data_ptr()


def test_spmv_uniform_gives_degrees_times_w0():
    g = gg.rmat(12, seed=4)
    n, rp, ci, wt = g.numpy()
    key = wl.wl_round_key(9, 0, 1)
    dn, drp, dci, dwt = dgraph(g)
    y = wl.wl_spmv_round(dn, drp, dci, dwt, torch.zeros(n, dtype=torch.int32, device=dev()), key)
    assert (u64(y) == np.diff(rp).astype(np.uint64) * np.uint64(oracle.weight(key, 0))).all()


# ------------------------------------------------------------------ S3+S4
def _same_partition(a, b):
    return oracle.canonical(a).tolist() == oracle.canonical(b).tolist()


@pytest.mark.parametrize("case", ["all_equal", "all_distinct", "equal_y_across_colours", "same_colour_distinct_y", "random"])
def test_relabel_matches_cpu_sort(case):
    n = 5000
    rng = np.random.default_rng(3)
    if case == "all_equal":
        c, y = np.zeros(n, np.int32), np.full(n, 77, np.uint64)
    elif case == "all_distinct":
        c, y = np.zeros(n, np.int32), rng.permutation(n).astype(np.uint64)
    elif case == "equal_y_across_colours":
        c, y = (np.arange(n) % 7).astype(np.int32), np.full(n, 5, np.uint64)
    elif case == "same_colour_distinct_y":
        c, y = (np.arange(n) % 3).astype(np.int32), (np.arange(n) % 11).astype(np.uint64) << np.uint64(40)
    else:
        c, y = rng.integers(0, 50, n).astype(np.int32), rng.integers(0, 4, n).astype(np.uint64) * np.uint64(0x9E3779B97F4A7C15)
    c = oracle.canonical(c)
    k = int(c.max()) + 1
    new, k2 = wl.wl_relabel(torch.from_numpy(c).to(dev()), k, torch.from_numpy(y.view(np.int64)).to(dev()))
    new = new.cpu().numpy()
    # CPU: dense ids of lexicographically sorted exact pairs
    pairs = np.stack([c.astype(np.uint64), y], 1)
    _, inv = np.unique(pairs, axis=0, return_inverse=True)
    assert k2 == inv.max() + 1
    assert sorted(np.unique(new).tolist()) == list(range(k2))  # dense
    assert _same_partition(new, inv)
    # refinement of the old partition (L153)
    assert len({(a, b) for a, b in zip(new.tolist(), c.tolist())}) == k2


# ------------------------------------------------------------------ S6
@pytest.mark.parametrize("n", [1, 2, 31, 2048, 2049, 100_003])
def test_canonicalize(n):
    rng = np.random.default_rng(n)
    c = rng.integers(0, max(1, n // 2), n).astype(np.int32)
    out, k = wl.wl_canonicalize(torch.from_numpy(c).to(dev()))
    assert out.cpu().numpy().tolist() == oracle.canonical(c).tolist()
    assert k == np.unique(c).size


# ------------------------------------------------------------------ whole Algorithm 1
# 256 = WL_FLAG_NO_DEEP, 512 = WL_FLAG_DEEP_EARLY (worklist regime from round 2 on: every graph goes through it),
# 1024 = WL_FLAG_NO_FINAL (no finality pruning), 32768 = WL_FLAG_DEEP_CLUSTER (every worklist window as one cluster launch)
@pytest.mark.parametrize("name", list(GRAPHS))
# 16384 = WL_FLAG_TAG_TABLE (the shared-memory hot-id table in every 16-bit round)
@pytest.mark.parametrize("flags", [0, 2, 4, 64, 128, 128 | 2, 256, 512, 512 | 64, 512 | 2, 1024, 1024 | 256,
                                   16384, 16384 | 2, 16384 | 512, 512 | 32768, 32768 | 2])
def test_refine_equals_oracle(name, flags):
    g = GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    want, counts, rounds = oracle.refine(n, rp, ci, wt)
    dn, drp, dci, dwt = dgraph(g)
    for seed in (0, 1, 2):
        res = wl.wl_refine(dn, drp, dci, dwt, seed=seed, flags=flags)
        assert res.round_colors == counts and res.rounds == rounds  # same trajectory
        assert res.num_colors == counts[-1]
        assert res.colors.cpu().numpy().tolist() == want.tolist()


@pytest.mark.parametrize("flags", [0, 512])
@pytest.mark.parametrize("seed", range(20))
def test_refine_many_seeds_rmat(seed, flags):
    g = gg.rmat(10, edge_factor=8, seed=seed, symmetrize=bool(seed % 2))
    n, rp, ci, wt = g.numpy()
    init = None if seed % 3 == 0 else gg.random_partition(n, 1 + seed, seed)
    want, counts, rounds = oracle.refine(n, rp, ci, wt, None if init is None else init.numpy())
    dn, drp, dci, dwt = dgraph(g)
    res = wl.wl_refine(dn, drp, dci, dwt, None if init is None else (init * 3 + 5).to(dev()), seed=seed * 977, flags=flags)
    assert res.round_colors == counts
    assert res.colors.cpu().numpy().tolist() == want.tolist()


DEEP_GRAPHS = {
    "path_3001": lambda: gg.path_graph(3001),
    "dpath_700": lambda: gg.directed_path(700),
    "grid_97": lambda: gg.grid2d(97),
    "btree_11": lambda: gg.from_edge_list(2 ** 11 - 1, [(i, 2 * i + 1) for i in range(2 ** 10 - 1)] +
                                          [(i, 2 * i + 2) for i in range(2 ** 10 - 1)]),
    "btree_11_up": lambda: gg.from_edge_list(2 ** 11 - 1, [(2 * i + 1, i) for i in range(2 ** 10 - 1)] +
                                             [(2 * i + 2, i) for i in range(2 ** 10 - 1)]),
    "weighted_chain": lambda: gg.from_edge_list(400, [(i, i + 1) for i in range(399)] + [(i + 1, i) for i in range(399)],
                                                weights=[1 + (i % 3) for i in range(399)] * 2),
    "comb": lambda: gg.from_edge_list(600, [(i, i + 1) for i in range(299)] + [(i + 1, i) for i in range(299)] +
                                      [(i, 300 + i) for i in range(300)] + [(300 + i, i) for i in range(300)]),
}


@pytest.mark.parametrize("name", list(DEEP_GRAPHS))
@pytest.mark.parametrize("flags", [0, 64, 256, 512, 32768, 512 | 32768])
def test_refine_deep_rounds_equal_oracle(name, flags):
    """Graphs that need tens to thousands of rounds: the worklist regime (rounds > 6, wl_deep.cuh) must give the oracle's
    colouring AND its per-round colour counts, with and without run-ahead windows, and the same as the plain loop (256)."""
    g = DEEP_GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    want, counts, rounds = oracle.refine(n, rp, ci, wt)
    dn, drp, dci, dwt = dgraph(g)
    for seed in (0, 7):
        res = wl.wl_refine(dn, drp, dci, dwt, seed=seed, flags=flags)
        assert res.rounds == rounds and res.round_colors == counts
        assert res.colors.cpu().numpy().tolist() == want.tolist()


@pytest.mark.parametrize("scale,sym", [(16, True), (17, False)])
def test_hot_id_table_rounds_equal_plain_rounds(scale, sym):
    """The 16-bit rounds through the shared-memory hot-id table (persistent kernel, ticketed row groups, tag hits and misses,
    hub rows beside it) against the plain row kernel and the oracle, on graphs large enough for many tickets per CTA."""
    g = gg.rmat(scale, seed=5, symmetrize=sym)
    n, rp, ci, wt = g.numpy()
    want, counts, rounds = oracle.refine(n, rp, ci)
    dn, drp, dci, dwt = dgraph(g)
    for flags in (wl.WL_FLAG_TAG_TABLE, wl.WL_FLAG_TAG_TABLE | wl.WL_FLAG_NO_PRUNE, 0):
        res = wl.wl_refine(dn, drp, dci, None, seed=3, flags=flags)
        assert res.round_colors == counts and res.colors.cpu().numpy().tolist() == want.tolist()


def test_refine_weighted_equals_multigraph():
    g1 = gg.from_edge_list(4, [(0, 1), (0, 1), (2, 1), (3, 3)])
    g2 = gg.from_edge_list(4, [(0, 1), (2, 1), (3, 3)], weights=[2, 1, 1])
    r1 = wl.wl_refine(*dgraph(g1), seed=1)
    r2 = wl.wl_refine(*dgraph(g2), seed=1)
    assert r1.colors.tolist() == r2.colors.tolist() == oracle.refine(*g1.numpy())[0].tolist()


def test_grid_256_closed_form():
    s = 256
    g = gg.grid2d(s)
    res = wl.wl_refine(*dgraph(g), seed=5)
    h = s // 2
    assert res.rounds == h and res.num_colors == h * (h + 1) // 2
    assert torch.equal(res.colors.cpu(), gg.grid2d_orbit_colors(s))


def test_refine_host_entry_point():
    g = gg.erdos_renyi(2000, 9000, seed=7)
    n, rp, ci, wt = g.numpy()
    want, counts, _ = oracle.refine(n, rp, ci)
    res = wl.wl_refine_host(n, g.row_ptr.pin_memory(), g.col.pin_memory(), seed=3)
    assert res.colors.numpy().tolist() == want.tolist() and res.round_colors == counts
    assert res.stats["bytes_h2d"] == 8 * (n + 1) + 4 * g.m and res.stats["bytes_d2h"] == 4 * n


@pytest.mark.parametrize("name", list(GRAPHS))
@pytest.mark.parametrize("pieces", [0, 2, 5, 32])
def test_refine_host_column_pieces_equal_oracle(name, pieces):
    """wl_refine_host uploads the columns in pieces of whole rows and runs the first pass over them piece by piece behind the
    copies (ColumnFeed): same colouring and trajectory as the oracle for any number of pieces, for weighted graphs, empty graphs,
    hub rows, with and without an initial partition, from pinned and from pageable host memory."""
    g = GRAPHS[name]()
    n, rp, ci, wt = g.numpy()
    want, counts, _ = oracle.refine(n, rp, ci, wt)
    w = None if g.weights is None else g.weights
    pin = (lambda t: t.pin_memory()) if pieces != 5 else (lambda t: t)  # pieces == 5: pageable memory
    res = wl.wl_refine_host(n, pin(g.row_ptr), pin(g.col), None if w is None else pin(w), seed=13, pieces=pieces)
    assert res.colors.numpy().tolist() == want.tolist() and res.round_colors == counts
    if n >= 4:
        init = gg.random_partition(n, 3, 2)
        want2, counts2, _ = oracle.refine(n, rp, ci, wt, init.numpy())
        res = wl.wl_refine_host(n, pin(g.row_ptr), pin(g.col), None if w is None else pin(w), pin(init), seed=14, pieces=pieces)
        assert res.colors.numpy().tolist() == want2.tolist() and res.round_colors == counts2


def test_refine_host_with_caller_device_workspace():
    """wl_options.device_workspace: the call uploads into and works in the caller's device arena (no cudaMalloc / cudaFree inside
    the call); too small an arena is WL_ENOMEM; same colouring, also when the arena is reused by the next call."""
    g = GRAPHS["rmat12_sym"]()
    n, rp, ci, wt = g.numpy()
    want, counts, _ = oracle.refine(n, rp, ci, wt)
    need = wl.wl_refine_host_device_bytes(n, g.m)
    assert need >= wl.wl_refine_workspace_bytes(n, g.m) + 8 * (n + 1) + 4 * g.m + 4 * n
    arena = torch.full((need,), 0xAB, dtype=torch.uint8, device=dev())
    for seed in (1, 2):
        res = wl.wl_refine_host(n, g.row_ptr.pin_memory(), g.col.pin_memory(), seed=seed, device_workspace=arena, pieces=3)
        assert res.colors.numpy().tolist() == want.tolist() and res.round_colors == counts
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine_host(n, g.row_ptr.pin_memory(), g.col.pin_memory(), seed=1, device_workspace=arena[: need - 256])
    assert e.value.code == wl.WL_ENOMEM
    gw = GRAPHS["weighted"]()
    assert wl.wl_refine_host_device_bytes(gw.n, gw.m, True, True) > wl.wl_refine_host_device_bytes(gw.n, gw.m)


@pytest.mark.parametrize("pieces", [1, 4])
def test_refine_host_rejects_malformed_input_in_any_piece(pieces):
    """S0 through the host entry point: a bad target in the first / last piece, decreasing offsets and a wrong last offset come
    back as WL_EINVAL (the piece borders are read from the unvalidated offsets: the copies must stay inside the arrays)."""
    g = gg.rmat(10, seed=4)
    n, m = g.n, g.m
    for pos, val in ((3, n), (m - 2, -1), (m // 2, n + 7)):
        bad = g.col.clone()
        bad[pos] = val
        with pytest.raises(wl.WlError) as e:
            wl.wl_refine_host(n, g.row_ptr.pin_memory(), bad.pin_memory(), seed=1, pieces=pieces)
        assert e.value.code == wl.WL_EINVAL
    for i, v in ((n // 2, 10 * m), (n // 3, -5), (n, m - 1)):
        rp2 = g.row_ptr.clone()
        rp2[i] = v
        with pytest.raises(wl.WlError) as e:
            wl.wl_refine_host(n, rp2.pin_memory(), g.col.pin_memory(), seed=1, pieces=pieces)
        assert e.value.code == wl.WL_EINVAL


# ------------------------------------------------------------------ error behaviour
def test_refine_host_entry_point_deep_rounds():
    """wl_refine_host on a graph that needs 128 rounds: the engine allocates the worklist regime's workspace itself once the
    loop gets to round 7 (kFlagLazyDeep) and must give the closed-form colouring and round count."""
    s = 256
    g = gg.grid2d(s)
    res = wl.wl_refine_host(g.n, g.row_ptr.pin_memory(), g.col.pin_memory(), seed=4)
    h = s // 2
    assert res.rounds == h and res.num_colors == h * (h + 1) // 2
    assert torch.equal(res.colors, gg.grid2d_orbit_colors(s))
    assert res.stats["kernel_launches"] < 600  # two launches per round after the switch, not four


def test_error_codes():
    g = gg.erdos_renyi(100, 300, seed=1)
    n, rp, ci, wt = dgraph(g)
    bad = ci.clone()
    bad[5] = n
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine(n, rp, bad)
    assert e.value.code == wl.WL_EINVAL
    for flags in (wl.WL_FLAG_EDGE_BALANCED, wl.WL_FLAG_NO_PRUNE):
        bad2 = ci.clone()
        bad2[-1] = -7
        with pytest.raises(wl.WlError) as e:
            wl.wl_refine(n, rp, bad2, flags=flags)
        assert e.value.code == wl.WL_EINVAL
    bad_rp = rp.clone()
    bad_rp[3] = bad_rp[4] + 1
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine(n, bad_rp, ci)
    assert e.value.code == wl.WL_EINVAL
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine(n, rp, ci, workspace=torch.empty(1024, dtype=torch.uint8, device=dev()))
    assert e.value.code == wl.WL_ENOMEM
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine(n, rp, ci, init_colors=torch.full((n,), -3, dtype=torch.int32, device=dev()))
    assert e.value.code == wl.WL_EINVAL
    res = wl.wl_refine(n, rp, ci, max_rounds=1, allow_max_rounds=True)
    assert res.status == wl.WL_EMAXROUNDS
    big = gg.from_edge_list(2, [(0, 1), (0, 1)], weights=[(1 << 32) - 1, 5])
    with pytest.raises(wl.WlError) as e:
        wl.wl_refine(*dgraph(big))
    assert e.value.code == wl.WL_ERANGE
