"""Pins for the CPU oracle against things that are NOT the oracle: brute force over all set partitions,
closed forms, dense numpy restatements of the paper's definitions, and the counting results of
Lemma 1 / Lemma 2 / Theorem 1."""
import math
import os
from math import isqrt

import numpy as np
import pytest
import torch

import graphgen as gg
import oracle
from helpers import (brute_force_coarsest, dense_adj, indicator, refines, same_partition, stable_dense)

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _np(g):
    return g.numpy()


# ------------------------------------------------------------------ canonical
def test_canonical_hand_cases():
    assert oracle.canonical([5, 5, 2, 9, 2]).tolist() == [0, 0, 1, 2, 1]
    assert oracle.canonical([]).tolist() == []
    assert oracle.canonical([7]).tolist() == [0]
    assert oracle.canonical([3, 2, 1, 0]).tolist() == [0, 1, 2, 3]


# ------------------------------------------------------------------ refine: brute force
@pytest.mark.parametrize("seed", range(60))
def test_refine_equals_brute_force_small(seed):
    n = 2 + seed % 6  # 2..7 nodes
    m = 1 + (seed * 7) % (2 * n + 3)
    g = gg.random_weighted_digraph(n, m, seed, max_w=3)
    _, rp, ci, wt = _np(g)
    init = gg.random_partition(n, 1 + seed % 3, seed).numpy()
    A = dense_adj(n, rp, ci, wt)
    want = brute_force_coarsest(A, init)
    got, counts, rounds = oracle.refine(n, rp, ci, wt, init)
    assert got.tolist() == want.tolist()
    assert counts[-1] == want.max() + 1
    # unweighted reading of the same structure (a_ij = multiplicity)
    A1 = dense_adj(n, rp, ci, None)
    want1 = brute_force_coarsest(A1, init)
    got1, _, _ = oracle.refine(n, rp, ci, None, init)
    assert got1.tolist() == want1.tolist()


def test_refine_brute_force_8_nodes():
    g = gg.random_weighted_digraph(8, 14, 1234, max_w=2)
    _, rp, ci, wt = _np(g)
    init = np.zeros(8, dtype=np.int32)
    want = brute_force_coarsest(dense_adj(8, rp, ci, wt), init)
    got, _, _ = oracle.refine(8, rp, ci, wt, init)
    assert got.tolist() == want.tolist()


# ------------------------------------------------------------------ refine: closed forms
@pytest.mark.parametrize("n,offs", [(7, (1,)), (12, (1, 3)), (20, (1, 2, 5)), (9, (2,))])
def test_regular_graph_one_colour(n, offs):
    _, rp, ci, wt = _np(gg.circulant(n, offs))
    c, counts, rounds = oracle.refine(n, rp, ci)
    assert counts[-1] == 1 and rounds == 1 and (c == 0).all()


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 10, 11, 64, 101])
def test_path_ceil_half(n):
    _, rp, ci, wt = _np(gg.path_graph(n))
    c, counts, _ = oracle.refine(n, rp, ci)
    assert counts[-1] == (n + 1) // 2
    # the classes are the distance-to-nearest-end levels
    want = oracle.canonical(np.minimum(np.arange(n), n - 1 - np.arange(n)))
    assert c.tolist() == want.tolist()


@pytest.mark.parametrize("k", [2, 3, 10, 100])
def test_star_two_colours(k):
    _, rp, ci, wt = _np(gg.star_graph(k))
    c, counts, _ = oracle.refine(k + 1, rp, ci)
    assert counts[-1] == 2 and c.tolist() == [0] + [1] * k


@pytest.mark.parametrize("a,b", [(2, 3), (1, 4), (5, 7)])
def test_complete_bipartite_two_colours(a, b):
    _, rp, ci, wt = _np(gg.complete_bipartite(a, b))
    c, counts, _ = oracle.refine(a + b, rp, ci)
    assert c.tolist() == [0] * a + [1] * b


@pytest.mark.parametrize("n", [1, 2, 5, 17])
def test_directed_path_discrete_in_n_rounds(n):
    _, rp, ci, wt = _np(gg.directed_path(n))
    c, counts, rounds = oracle.refine(n, rp, ci)
    assert counts[-1] == n and rounds == n  # one new class per round, the last round confirms (n=1: 1 round)
    assert sorted(c.tolist()) == list(range(n))


@pytest.mark.parametrize("n", [1, 3, 8])
def test_directed_cycle_one_colour(n):
    _, rp, ci, wt = _np(gg.directed_cycle(n))
    c, counts, _ = oracle.refine(n, rp, ci)
    assert counts[-1] == 1


def test_grid_closed_form_matches_golden():
    """s x s grid: h(h+1)/2 colours in h rounds, h = ceil(s/2); classes = dihedral orbits."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "grid_closed_form.txt")) if l.strip() and l[0] != "#"]
    for s, colours, rounds in ((int(a), int(b), int(c)) for a, b, c in rows):
        h = (s + 1) // 2
        assert colours == h * (h + 1) // 2 and rounds == h  # the fixture itself is the closed form
        if s > 40:
            continue
        _, rp, ci, wt = _np(gg.grid2d(s))
        c, counts, r = oracle.refine(s * s, rp, ci)
        assert counts[-1] == colours and r == rounds
        assert c.tolist() == gg.grid2d_orbit_colors(s).tolist()


def test_direction_matters_out_edges_only():
    """Rows are sources (L43, L49): in 0->1, 0->2 node 0 differs from the sinks; sinks are equal."""
    g = gg.from_edge_list(3, [(0, 1), (0, 2)])
    _, rp, ci, wt = _np(g)
    c, _, _ = oracle.refine(3, rp, ci)
    assert c.tolist() == [0, 1, 1]
    # in-edges do not count: 1->0, 2->0 gives {0} and {1,2} too, but a lone in-degree difference does not split
    g = gg.from_edge_list(4, [(0, 2), (1, 2), (1, 3), (0, 3), (2, 0)])  # 3 is a sink, 2 is not
    _, rp, ci, wt = _np(g)
    c, _, _ = oracle.refine(4, rp, ci)
    assert c[0] == c[1] and c[2] != c[3]


def test_multi_edges_add_and_weights_equivalent():
    """a_ij in N_0: a duplicate CSR entry equals one entry of weight 2 (L43)."""
    g1 = gg.from_edge_list(4, [(0, 1), (0, 1), (2, 1), (3, 3)])
    g2 = gg.from_edge_list(4, [(0, 1), (2, 1), (3, 3)], weights=[2, 1, 1])
    c1, _, _ = oracle.refine(*_np(g1))
    c2, _, _ = oracle.refine(*_np(g2))
    assert c1.tolist() == c2.tolist()
    A = dense_adj(*_np(g1))
    assert c1.tolist() == brute_force_coarsest(A, np.zeros(4, dtype=np.int32)).tolist()


@pytest.mark.parametrize("seed", range(8))
def test_renumbering_invariance(seed):
    g = gg.rmat(8, edge_factor=4, seed=seed, symmetrize=bool(seed % 2))
    n, rp, ci, wt = _np(g)
    c, counts, rounds = oracle.refine(n, rp, ci)
    perm = gg.random_permutation(n, seed)
    gp = gg.permute_graph(g, perm)
    cp, countsp, roundsp = oracle.refine(*_np(gp))
    assert counts == countsp and rounds == roundsp
    assert same_partition(c, cp[perm.numpy()])


@pytest.mark.parametrize("seed", range(6))
def test_refine_result_is_stable_and_coarsest_property(seed):
    """Stability by the dense definition, and merging any two blocks breaks stability or the init constraint
    (a necessary condition of coarseness that is cheap at this size)."""
    g = gg.rmat(6, edge_factor=3, seed=seed, symmetrize=False)
    n, rp, ci, wt = _np(g)
    init = gg.random_partition(n, 2, seed).numpy()
    c, counts, _ = oracle.refine(n, rp, ci, None, init)
    A = dense_adj(n, rp, ci)
    assert stable_dense(A, c) and refines(c, init)
    k = counts[-1]
    # iterate merges to a fixed point from a merged pair: no stable coarsening may exist
    for a in range(min(k, 12)):
        for b in range(a + 1, min(k, 12)):
            merged = np.where(c == b, a, c)
            if not refines(merged, init):
                continue
            assert not stable_dense(A, oracle.canonical(merged))


# ------------------------------------------------------------------ is_stable
@pytest.mark.parametrize("seed", range(30))
def test_is_stable_matches_dense_definition(seed):
    n = 3 + seed % 6
    g = gg.random_weighted_digraph(n, 2 * n, seed + 100, max_w=2)
    _, rp, ci, wt = _np(g)
    A = dense_adj(n, rp, ci, wt)
    for k in (1, 2, 3, n):
        col = gg.random_partition(n, k, seed * 13 + k).numpy()
        assert oracle.is_stable(n, rp, ci, wt, col) == stable_dense(A, col)
    assert oracle.is_stable(n, rp, ci, wt, np.arange(n, dtype=np.int32))  # discrete partition is stable


# ------------------------------------------------------------------ inner labels (Def. 5)
@pytest.mark.parametrize("seed", range(20))
def test_inner_labels_brute_force(seed):
    n, nb = 9, 1 + seed % 4
    g = gg.random_weighted_digraph(n, 3 + seed, seed + 7)
    _, rp, ci, wt = _np(g)
    eb = gg.random_edge_batches(g, nb, seed).numpy()
    sink = np.zeros(n, dtype=np.int32)
    lab = oracle.inner_labels(n, rp, eb, sink)
    E = [(i, int(ci[e]), e) for i in range(n) for e in range(rp[i], rp[i + 1])]
    Vk = []
    for k in range(nb):
        Ek = {e for (_, _, e) in E if eb[e] == k}
        # V_k = { i | no edge (i, j) in E \ E_k }   (L141)
        Vk.append({i for i in range(n) if not any(s == i and e not in Ek for (s, _, e) in E)})
    for i in range(n):
        has_out = rp[i] < rp[i + 1]
        member = [k for k in range(nb) if i in Vk[k]]
        if has_out:
            assert len(member) <= 1  # pairwise disjoint (L145)
            assert lab[i] == (member[0] if member else -1)
        else:
            assert member == list(range(nb)) and lab[i] == 0  # vacuous case, reading Q9


# ------------------------------------------------------------------ quotient (Def. 4)
@pytest.mark.parametrize("seed", range(12))
def test_quotient_dense_identity(seed):
    g = gg.rmat(5, edge_factor=3, seed=seed, symmetrize=bool(seed % 2))
    n, rp, ci, wt = _np(g)
    c, _, _ = oracle.refine(n, rp, ci)
    k, qrp, qc, qw = oracle.quotient(n, rp, ci, None, c)
    A = dense_adj(n, rp, ci)
    Aq = dense_adj(k, qrp, qc, qw)
    S = indicator(c)
    assert (A @ S == S @ Aq).all()  # A S = S A' characterises the quotient of a stable colouring (Eq. 1)
    assert (Aq.sum(1) == (S.T @ A.sum(1)) // S.sum(0)).all()  # row sums preserved (L447)
    for b in range(k):  # sorted, merged, no zeros
        cols = qc[qrp[b]:qrp[b + 1]]
        assert (np.diff(cols) > 0).all() and (qw[qrp[b]:qrp[b + 1]] > 0).all()
    # fixed point: the coarsest colouring of the quotient of the coarsest colouring is discrete (L67, L204)
    cq, _, _ = oracle.refine(k, qrp, qc, qw)
    assert sorted(cq.tolist()) == list(range(k))


# ------------------------------------------------------------------ Algorithm 2
@pytest.mark.parametrize("seed", range(16))
def test_rbsc_invariants(seed):
    g = gg.rmat(6 + seed % 2, edge_factor=3, seed=seed, symmetrize=bool(seed % 2))
    n, rp, ci, wt = _np(g)
    coarsest, _, _ = oracle.refine(n, rp, ci)
    A = dense_adj(n, rp, ci)
    m = g.m
    for nb in (1, 2, 4):
        cap = -(-m // nb)
        c, k, outer, nb_last = oracle.rbsc(n, rp, ci, None, cap)
        assert stable_dense(A, c)            # Theorem 2 (L163)
        assert refines(c, coarsest)          # L165, L211
        if nb_last == 1:
            assert c.tolist() == coarsest.tolist()   # case (i), L208
    # arbitrary partition (L163) + independence of batch numbering (L213)
    eb = gg.random_edge_batches(g, 3, seed).numpy()
    c1, k1, _, _ = oracle.rbsc(n, rp, ci, None, -(-m // 3), first_edge_batch=eb, num_first_batches=3)
    eb2 = np.array([2, 0, 1], dtype=np.int32)[eb]
    c2, k2, _, _ = oracle.rbsc(n, rp, ci, None, -(-m // 3), first_edge_batch=eb2, num_first_batches=3)
    assert stable_dense(A, c1) and refines(c1, coarsest)
    assert c1.tolist() == c2.tolist()


@pytest.mark.parametrize("seed", range(12))
def test_rbsc_inherited_batches_invariants(seed):
    """Reading Q14b (the quotient keeps the batches of its graph): still Algorithm 2 on SOME edge partition per iteration, so
    Theorem 2 (stability), L165 (refines the coarsest colouring) and case (i) (one batch = the coarsest colouring) must
    hold; the first outer iteration is the same as without the rule, so the result can only be coarser or equal when both
    stop after it."""
    g = gg.rmat(6 + seed % 2, edge_factor=3, seed=seed, symmetrize=bool(seed % 2)) if seed < 8 else \
        gg.random_weighted_digraph(60, 240, seed, max_w=3)
    n, rp, ci, wt = _np(g)
    coarsest, _, _ = oracle.refine(n, rp, ci, wt)
    A = dense_adj(n, rp, ci, wt)
    for nb in (1, 2, 3, 5):
        cap = -(-g.m // nb)
        c, k, outer, nb_last = oracle.rbsc(n, rp, ci, wt, cap, inherit=True)
        assert stable_dense(A, c)
        assert refines(c, coarsest)
        if nb == 1:
            assert c.tolist() == coarsest.tolist() and outer == 1
        c1, _, _, _ = oracle.rbsc(n, rp, ci, wt, cap, max_outer=1)
        ci1, _, _, _ = oracle.rbsc(n, rp, ci, wt, cap, max_outer=1, inherit=True)
        assert c1.tolist() == ci1.tolist()  # the rule only changes iterations >= 2
        assert refines(c1, c)               # every outer iteration coarsens (L206)


def _num_greedy_batches(n, rp, cap):
    """N_b of the library's default partition, restated on a plain offset list (Q13)."""
    import torch
    g = gg.Graph(n=n, row_ptr=torch.as_tensor(np.asarray(rp), dtype=torch.int64),
                 col=torch.zeros(int(rp[-1]), dtype=torch.int32), weights=None, name="q")
    return max(1, len(gg.contiguous_row_batches(g, cap)) - 1)


@pytest.mark.parametrize("seed", range(14))
def test_rbsc_aggressive_stop_is_the_plain_loop_cut_where_the_rule_says(seed):
    """"the outer loop of Algorithm 2 stops as soon as the number of batches in the next iteration would not
    decrease".  Pin: run the PLAIN loop limited to t = 1, 2, ... iterations, build the quotient of each result with
    oracle.quotient, count the batches the default partition gives it (independent restatement in graphgen); the first t
    whose successor would not run with fewer batches (or where the plain loop ends anyway) must be where the aggressive run
    stops, with the same colouring.  Plus Theorem 2, L165 and L206 (the plain result is coarser or equal)."""
    g = gg.rmat(6 + seed % 3, edge_factor=2 + seed % 4, seed=seed, symmetrize=bool(seed % 2)) if seed < 10 else \
        gg.random_weighted_digraph(50 + seed, 260, seed, max_w=2)
    n, rp, ci, wt = _np(g)
    A = dense_adj(n, rp, ci, wt)
    coarsest, _, _ = oracle.refine(n, rp, ci, wt)
    stopped_early = 0
    for nb in (2, 3, 5, 9):
        cap = max(1, -(-g.m // nb))
        full, _, outer_full, _ = oracle.rbsc(n, rp, ci, wt, cap)
        got, k, outer, nbl = oracle.rbsc(n, rp, ci, wt, cap, aggressive=True)
        assert stable_dense(A, got) and refines(got, coarsest) and refines(got, full)
        # walk the plain loop
        nb_t = _num_greedy_batches(n, rp, cap)
        expect_t = None
        for t in range(1, outer_full + 1):
            c_t, k_t, o_t, nbl_t = oracle.rbsc(n, rp, ci, wt, cap, max_outer=t)
            assert nbl_t == nb_t
            if t == outer_full:
                expect_t = t
                break
            _, qrp, qc, qw = oracle.quotient(n, rp, ci, wt, c_t)
            nb_next = _num_greedy_batches(k_t, qrp, cap)
            if nb_next >= nb_t:
                expect_t = t
                break
            nb_t = nb_next
        assert outer == expect_t and nbl == nb_t
        assert got.tolist() == c_t.tolist()
        stopped_early += outer < outer_full
    if seed in (0, 1, 2, 3):
        assert stopped_early >= 1  # the rule really cuts the loop short on these graphs (42 of the 56 cases do)


def test_rbsc_aggressive_stop_hand_case():
    """A directed path 0 -> 1 -> ... -> 9 with one edge per batch: iteration 1 leaves everything discrete except nothing to
    merge, the quotient is the graph itself, so the next iteration would run with the same 9 batches: the aggressive rule
    stops after ONE iteration where the plain rule also stops (|V| unchanged); with twin leaves split over two batches
    (test above) the quotient shrinks to fewer batches and both rules go on."""
    g = gg.directed_path(10)
    n, rp, ci, wt = _np(g)
    c, k, outer, nbl = oracle.rbsc(n, rp, ci, None, 1, aggressive=True)
    assert outer == 1 and k == 10
    # two stars whose leaves are spread over many single-edge batches: iteration 1 merges nothing (every leaf is inner to its
    # own batch, alone), the quotient keeps all edges -> same N_b -> the aggressive rule stops, the plain rule too (|V| = n)
    g = gg.from_edge_list(7, [(1, 0), (2, 0), (3, 0), (4, 6), (5, 6)])
    n, rp, ci, wt = _np(g)
    ca, ka, oa, _ = oracle.rbsc(n, rp, ci, None, 2, aggressive=True)
    cp, kp, op, _ = oracle.rbsc(n, rp, ci, None, 2)
    assert oa <= op and refines(ca, cp)


def test_rbsc_single_batch_is_refine():
    g = gg.erdos_renyi(300, 900, seed=3)
    n, rp, ci, wt = _np(g)
    c, k, outer, nbl = oracle.rbsc(n, rp, ci, None, g.m)
    assert outer == 1 and nbl == 1
    assert c.tolist() == oracle.refine(n, rp, ci)[0].tolist()


def test_rbsc_twin_leaves_merge_only_if_same_batch():
    """Hand case: nodes 0 and 1 both point to node 2 only.  With both edges in one batch they merge;
    split across two batches they are inner to different batches and stay apart in outer iteration 1,
    and the quotient iteration (one batch when m' <= M_b) merges them."""
    g = gg.from_edge_list(3, [(0, 2), (1, 2)])
    n, rp, ci, wt = _np(g)
    c, k, outer, nbl = oracle.rbsc(n, rp, ci, None, 2)
    assert c.tolist() == [0, 0, 1] and outer == 1
    c, k, outer, nbl = oracle.rbsc(n, rp, ci, None, 1, max_outer=1)
    assert c.tolist() == [0, 1, 2]
    c, k, outer, nbl = oracle.rbsc(n, rp, ci, None, 1)
    assert k == 3 and outer == 1  # |V| unchanged after the first contraction: fixed point (L209), finer than coarsest


@pytest.mark.parametrize("seed", range(12))
def test_rbsc_with_init_classes_invariants(seed):
    """Reading Q18 (Algorithm 2 from initial classes, L94 + Eq. 3): the result is a stable colouring (Thm 2) that refines the
    classes, is refined by nothing coarser than the coarsest stable colouring refining them (computed by oracle.refine with the
    same init, itself pinned by brute force), equals it when the loop ends on one batch (case (i), L208), does not depend on how
    the classes are named, and with one class is Algorithm 2 as written."""
    g = gg.rmat(6 + seed % 2, edge_factor=3, seed=seed, symmetrize=bool(seed % 2)) if seed < 8 else \
        gg.random_weighted_digraph(60, 240, seed, max_w=3)
    n, rp, ci, wt = _np(g)
    A = dense_adj(n, rp, ci, wt)
    init = gg.random_partition(n, 2 + seed % 4, seed).numpy()
    coarsest, _, _ = oracle.refine(n, rp, ci, wt, init)
    plain, _, _ = oracle.refine(n, rp, ci, wt)
    renamed = (init.max() - init) * 7 + 3  # another naming of the same classes, not dense, other order
    eb = gg.random_edge_batches(g, 3, seed).numpy()
    for inherit in (False, True):
        for nb in (1, 2, 3, 5):
            cap = -(-g.m // nb)
            c, k, outer, nb_last = oracle.rbsc(n, rp, ci, wt, cap, inherit=inherit, init=init)
            assert stable_dense(A, c)
            assert refines(c, init)
            assert refines(c, coarsest)
            if nb_last == 1:
                assert c.tolist() == coarsest.tolist()
            assert oracle.rbsc(n, rp, ci, wt, cap, inherit=inherit, init=renamed)[0].tolist() == c.tolist()
            one = oracle.rbsc(n, rp, ci, wt, cap, inherit=inherit, init=np.full(n, 5, dtype=np.int32))
            none = oracle.rbsc(n, rp, ci, wt, cap, inherit=inherit)
            assert (one[0].tolist(), one[1:]) == (none[0].tolist(), none[1:])
    c, k, _, _ = oracle.rbsc(n, rp, ci, wt, -(-g.m // 3), first_edge_batch=eb, num_first_batches=3, init=init)
    assert stable_dense(A, c) and refines(c, init) and refines(c, coarsest)
    # the classes matter on these inputs: the coarsest colouring without them does not refine them
    if not refines(plain, init):
        assert not same_partition(coarsest, plain)
    # discrete classes stay discrete
    c, k, outer, _ = oracle.rbsc(n, rp, ci, wt, -(-g.m // 2), init=np.arange(n, dtype=np.int32))
    assert k == n and c.tolist() == list(range(n))


def test_rbsc_with_init_classes_hand_case():
    """Twin leaves 0, 1 -> 2 (one batch: they merge).  Put them in different classes and they must stay apart; put node 2 alone
    in a class and nothing changes."""
    g = gg.from_edge_list(3, [(0, 2), (1, 2)])
    n, rp, ci, wt = _np(g)
    assert oracle.rbsc(n, rp, ci, None, 2)[0].tolist() == [0, 0, 1]
    assert oracle.rbsc(n, rp, ci, None, 2, init=[0, 1, 0])[0].tolist() == [0, 1, 2]
    assert oracle.rbsc(n, rp, ci, None, 2, init=[4, 4, 9])[0].tolist() == [0, 0, 1]
    # two batches: apart after the first iteration either way, merged by the quotient iteration only if the classes allow it
    g = gg.from_edge_list(4, [(0, 2), (1, 2), (3, 2)])
    n, rp, ci, wt = _np(g)
    assert oracle.rbsc(n, rp, ci, None, 2, init=[0, 0, 0, 0])[0].tolist() == oracle.refine(n, rp, ci)[0].tolist()
    assert oracle.refine(n, rp, ci)[0].tolist() == [0, 0, 1, 0]
    got = oracle.rbsc(n, rp, ci, None, 2, init=[0, 0, 0, 1])[0].tolist()  # batches {0->2, 1->2}, {3->2}; sink 2 inner to the second
    assert got == oracle.refine(n, rp, ci, None, [0, 0, 0, 1])[0].tolist() == [0, 0, 1, 2]
    # classes that split the only mergeable pair of the first batch: |V| unchanged after the first contraction, the loop ends
    # (L209) on a colouring finer than the coarsest one [0, 1, 2, 0]
    c, k, outer, _ = oracle.rbsc(n, rp, ci, None, 2, init=[0, 1, 0, 0])
    assert c.tolist() == [0, 1, 2, 3] and outer == 1
    assert oracle.refine(n, rp, ci, None, [0, 1, 0, 0])[0].tolist() == [0, 1, 2, 0]


# ------------------------------------------------------------------ weights / SpMV / Algorithm 1
def test_mix_constants_are_the_documented_ones():
    def frac_sqrt(p):
        return isqrt(p << 128) & ((1 << 64) - 1)
    m1, m2 = frac_sqrt(2) | 1, frac_sqrt(3) | 1
    golden = ((isqrt(5 << 128) - (1 << 64)) >> 1) | 1
    M = (1 << 64) - 1

    def mix(x):
        x ^= x >> 32
        x = (x * m1) & M
        x ^= x >> 29
        x = (x * m2) & M
        x ^= x >> 32
        return x
    for seed, stream, rnd, c in [(0, 0, 1, 0), (1, 2, 3, 4), (M, 5, 77, 2 ** 32 + 9), (12345, 1 << 40, 1000, 99)]:
        key = mix((mix((mix((seed + golden) & M) + stream) & M) + rnd) & M)
        assert oracle.round_key(seed, stream, rnd) == key
        assert oracle.weight(key, c) == mix((c + key) & M)


def test_weight_is_a_bijection():
    """Invert mix step by step: odd multipliers have inverses mod 2^64, xor-shifts are involutive up to iteration."""
    M = (1 << 64) - 1
    m1 = (isqrt(2 << 128) & M) | 1
    m2 = (isqrt(3 << 128) & M) | 1
    i1, i2 = pow(m1, -1, 1 << 64), pow(m2, -1, 1 << 64)

    def unxs(y, s):
        x = y
        for _ in range(64 // s + 1):
            x = y ^ (x >> s)
        return x
    key = oracle.round_key(42, 0, 3)
    for c in list(range(50)) + [2 ** 32 - 1, 2 ** 32, 2 ** 40 + 17]:
        w = oracle.weight(key, c)
        x = unxs(w, 32)
        x = (x * i2) & M
        x = unxs(x, 29)
        x = (x * i1) & M
        x = unxs(x, 32)
        assert (x - key) & M == c
    ws = {oracle.weight(key, c) for c in range(20000)}
    assert len(ws) == 20000  # Alg. 1 line 4: |H| distinct values


@pytest.mark.parametrize("seed", range(6))
def test_spmv_u64_equals_numpy_dense(seed):
    g = gg.random_weighted_digraph(40, 300, seed, max_w=1000)
    n, rp, ci, wt = _np(g)
    rng = np.random.default_rng(seed)
    w = rng.integers(0, 1 << 64, size=n, dtype=np.uint64)
    A = dense_adj(n, rp, ci, wt).astype(np.uint64)
    with np.errstate(over="ignore"):
        want = (A * w[None, :]).sum(axis=1, dtype=np.uint64)
    assert (oracle.spmv_u64(n, rp, ci, wt, w) == want).all()
    assert (oracle.spmv_u64(n, rp, ci, wt, w, qbits=16) == (want & np.uint64(0xFFFF))).all()
    ones = np.ones(n, dtype=np.uint64)
    assert (oracle.spmv_u64(n, rp, ci, None, ones) == np.diff(rp).astype(np.uint64)).all()  # w = 1 gives out-degrees


@pytest.mark.parametrize("seed", range(10))
def test_rsc_equals_refine_with_same_trajectory(seed):
    g = gg.rmat(9, edge_factor=6, seed=seed, symmetrize=bool(seed % 2))
    n, rp, ci, wt = _np(g)
    init = None if seed % 3 else gg.random_partition(n, 3, seed).numpy()
    c, counts, rounds = oracle.refine(n, rp, ci, None, init)
    c2, counts2, rounds2, z1 = oracle.rsc(n, rp, ci, None, init, seed=seed, z_round=1)
    assert c.tolist() == c2.tolist() and counts == counts2 and rounds == rounds2
    if init is None:  # round 1 from a uniform start: z_i = outdeg(i) * w_0
        w0 = oracle.weight(oracle.round_key(seed, 0, 1), 0)
        assert (z1 == (np.diff(rp).astype(np.uint64) * np.uint64(w0))).all()


@pytest.mark.parametrize("t,q", [(12, 16), (8, 12)])
def test_reduced_ring_miss_rate_is_lemma1_tight(t, q):
    """Lemma 1 (L418): a_1 x = 0 mod 2^q with gcd(a_1, 2^q) = 2^t has 2^t roots, so one node of out-degree 2^t
    among sinks misses its only split with probability exactly 2^{t-q} (w_0 uniform).  Count over seeds."""
    d = 1 << t
    g = gg.from_edge_list(d + 1, [(0, j) for j in range(1, d + 1)])
    n, rp, ci, wt = _np(g)
    trials = 3000
    miss = 0
    for seed in range(trials):
        c, counts, rounds, _ = oracle.rsc(n, rp, ci, seed=seed, qbits=q)
        assert counts[-1] in (1, 2)
        miss += counts[-1] == 1
    p = 2.0 ** (t - q)
    sd = math.sqrt(trials * p * (1 - p))
    assert abs(miss - trials * p) < 5 * sd, (miss, trials * p)


def test_lemma1_root_count_brute_force():
    """|{x in (Z/2^q)^k : a.x = 0}| = 2^t (2^q)^{k-1} with 2^t = gcd(a_1..a_k, 2^q) (L418), by enumeration."""
    q, k = 4, 2
    r = 1 << q
    for a in [(1, 0), (2, 4), (4, 8), (6, 2), (8, 8), (3, 5), (12, 4)]:
        gcd = math.gcd(math.gcd(a[0], a[1]), r)
        roots = sum((a[0] * x + a[1] * y) % r == 0 for x in range(r) for y in range(r))
        assert roots == gcd * r ** (k - 1)


def test_theorem1_numeric_bounds_golden():
    """Numbers the paper prints: 2^{-q/2} <= 1e-9 and 2^{q/2}/(0.6 2^q) <= 1e-9 at q = 64 (L402-L406);
    birthday ratio >= 0.60 (L430) for k = sqrt(r) via the exact log-sum bound of L436-L443."""
    vals = dict(l.split()[:2] for l in open(os.path.join(GOLDEN, "theorem1_bounds.txt")) if l.strip() and l[0] != "#")
    q = int(vals["q"])
    eps = float(vals["eps"])
    assert 2.0 ** (-q / 2) <= eps
    assert 2.0 ** (q / 2) / (float(vals["birthday_lower"]) * 2.0 ** q) <= eps
    r = 2.0 ** q
    k = 2.0 ** (q / 2)
    assert math.exp(-(k * (k - 1) / 2) / r / (1 - 2.0 ** (-q / 2))) >= float(vals["birthday_lower"])


def test_generator_hash_pinned_by_python_ints():
    c = torch.tensor([0, 1, 2, 12345678901234, -5, 2 ** 62], dtype=torch.int64)
    assert gg.hash_u32(7, c).tolist() == [gg.hash_u32_int(7, int(x)) for x in c.tolist()]
    def frac_sqrt(p):
        return isqrt(p << 128) & ((1 << 64) - 1)
    assert (gg._K1, gg._K2, gg._K3) == (frac_sqrt(5) | 1, frac_sqrt(7) | 1, frac_sqrt(11) | 1)


def test_config1_shape():
    g = gg.erdos_renyi()
    n, rp, ci, wt = _np(g)
    assert (n, g.m) == (10_000, 50_000)
    src = np.repeat(np.arange(n), np.diff(rp))
    assert (src != ci).all() and np.unique(src.astype(np.int64) * n + ci).size == 50_000
    c, counts, rounds = oracle.refine(n, rp, ci)
    assert rounds <= 8 and counts[-1] > 9000
    assert oracle.is_stable(n, rp, ci, None, c)
