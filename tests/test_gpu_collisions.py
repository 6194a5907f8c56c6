"""Collisions of the randomized refinement on the CUDA path, counted (Theorem 1, proof L396-L414; Lemma 1).

At q = 64 a collision is never seen; Algorithm 1's precision parameter q (wl_options.ring_bits) makes them frequent enough to
measure.  What is pinned here:
  * Lemma 1 is tight on the GPU: one hub of out-degree 2^t among sinks misses its only split with probability 2^{t-q}, seed by
    seed the same event as in the CPU Algorithm 1 (oracle.rsc) because round 1 uses the same w(0);
  * reading Q12: every mismatch is "GPU strictly coarser than the exact colouring", never anything else;
  * plain Algorithm 1 on the GPU (WL_FLAG_NO_DEEP | WL_FLAG_NO_FINAL) misses as rarely as the CPU Algorithm 1: a collision in a
    round that is not the last one is repaired by the fresh weights of the next (the paper's argument, L408-L414);
  * the default build (R4 fixed key from round 7, R5 final blocks) turns mid-run collisions into permanent
    ones: its miss rate is measured next to the union bound  sum_r N_r 2^{-q} / 0.6  that DESIGN.md states for it.
"""
import math

import numpy as np
import pytest
import torch

import graphgen as gg
import oracle
from helpers import classify, split_pairs

pytestmark = pytest.mark.gpu
wl = pytest.importorskip("paper_2607_02603_b200")

PLAIN = 256 | 1024  # WL_FLAG_NO_DEEP | WL_FLAG_NO_FINAL: Algorithm 1 with fresh weights in every round (+ exact pruning R1)


def dev():
    return torch.device("cuda", 0)


@pytest.mark.parametrize("t,q", [(12, 16), (8, 12)])
@pytest.mark.parametrize("flags", [0, PLAIN | 2])
def test_lemma1_miss_rate_on_the_gpu(t, q, flags):
    d = 1 << t
    g = gg.from_edge_list(d + 1, [(0, j) for j in range(1, d + 1)])
    n, rp, ci, wt = g.numpy()
    dg = g.to(dev())
    ws = torch.empty(wl.wl_refine_deep_workspace_bytes(n, g.m), dtype=torch.uint8, device=dev())
    trials, miss = 3000, 0
    for seed in range(trials):
        res = wl.wl_refine(n, dg.row_ptr, dg.col, seed=seed, flags=flags, ring_bits=q, workspace=ws)
        assert res.num_colors in (1, 2)
        _, counts, _, _ = oracle.rsc(n, rp, ci, seed=seed, qbits=q)
        assert res.num_colors == counts[-1]  # the same event seed by seed: z_hub = 2^t w(0) mod 2^q == 0
        miss += res.num_colors == 1
    p = 2.0 ** (t - q)
    assert abs(miss - trials * p) < 5 * math.sqrt(trials * p * (1 - p)), (miss, trials * p)


def _trajectory_pairs(n, rp, ci, wt):
    """sum over rounds of N_r (helpers.split_pairs) along the exact trajectory, from the oracle run one round at a time."""
    prev = np.zeros(n, dtype=np.int32)
    total = []
    while True:
        cur, counts, _ = oracle.refine(n, rp, ci, wt, init=prev, max_rounds=1, allow_unconverged=True)
        if int(cur.max()) == int(prev.max()):
            return total
        total.append(split_pairs(prev, cur))
        prev = cur


CASES = {
    # name: (graph, q, seeds)
    "er_2000": (lambda: gg.erdos_renyi(2000, 9000, seed=5), 18, 600),
    "rmat11_sym": (lambda: gg.rmat(11, edge_factor=8, seed=3), 18, 600),
    "path_301": (lambda: gg.path_graph(301), 12, 600),
    "grid_33": (lambda: gg.grid2d(33), 10, 600),
    "grid_33_q16": (lambda: gg.grid2d(33), 16, 600),
}


@pytest.mark.parametrize("name", list(CASES))
def test_collisions_only_coarsen_and_cost_of_r4_r5(name):
    make, q, seeds = CASES[name]
    g = make()
    n, rp, ci, wt = g.numpy()
    want, counts, rounds = oracle.refine(n, rp, ci, wt)
    N = _trajectory_pairs(n, rp, ci, wt)
    dg = g.to(dev())
    ws = torch.empty(wl.wl_refine_deep_workspace_bytes(n, g.m), dtype=torch.uint8, device=dev())
    tally = {}
    for label, flags in (("plain", PLAIN), ("default", 0), ("deep_early", 512)):
        t = {"equal": 0, "coarser": 0, "other": 0}
        for seed in range(seeds):
            res = wl.wl_refine(n, dg.row_ptr, dg.col, seed=seed, flags=flags, ring_bits=q, workspace=ws)
            t[classify(res.colors.cpu().numpy(), want)] += 1
        tally[label] = t
        assert t["other"] == 0, (name, label, t)  # Q12: a collision can only under-refine
    cpu = {"equal": 0, "coarser": 0, "other": 0}
    for seed in range(seeds):
        c, _, _, _ = oracle.rsc(n, rp, ci, wt, seed=10_000 + seed, qbits=q)
        cpu[classify(c, want)] += 1
    assert cpu["other"] == 0
    # plain Algorithm 1: GPU and CPU miss at the same rate (different colour ids, hence different weights: same law, not the
    # same events); 5 sigma of a two-sample Poisson comparison
    a, b = tally["plain"]["coarser"], cpu["coarser"]
    assert abs(a - b) <= 5 * math.sqrt(a + b + 1), (name, tally, cpu)
    # the default build may miss more often (R4/R5), but never beyond the union bound over every split event of every round
    bound = min(1.0, sum(N) * 2.0 ** (1 - q) / 0.6)  # t <= 1 for the coefficient differences of these graphs
    for label in ("default", "deep_early"):
        m = tally[label]["coarser"]
        assert m <= seeds * bound + 5 * math.sqrt(seeds * bound + 1), (name, label, tally, sum(N), bound)
    print(f"\n[collisions] {name}: q={q} seeds={seeds} pairs per round={N} union bound={bound:.3g} gpu={tally} cpu_alg1={cpu}")


def test_full_ring_never_mismatches_c1_many_seeds():
    """q = 64 (the product): 200 seeds on C1, every result classified; expected and required: all equal."""
    g = gg.erdos_renyi()
    n, rp, ci, wt = g.numpy()
    want, counts, _ = oracle.refine(n, rp, ci)
    dg = g.to(dev())
    t = {"equal": 0, "coarser": 0, "other": 0}
    for seed in range(200):
        res = wl.wl_refine(n, dg.row_ptr, dg.col, seed=seed)
        t[classify(res.colors.cpu().numpy(), want)] += 1
    assert t == {"equal": 200, "coarser": 0, "other": 0}
