"""Batch-level multi-GPU driver of Algorithm 2 (RBSC): one process per GPU, the batches of every outer
iteration spread over the ranks, `torch.distributed` for the exchange.

The paper runs the per-batch loop of Algorithm 2 (lines 7-11) "embarrassingly parallel ... scheduled concurrently across GPUs"
(L213) with a host merge (L239).  Here every rank owns a contiguous run of batches = a contiguous node range of the current
graph.  Per outer iteration:

  local pass   every rank refines its batches (wl_refine_inner: B3 + B4 + ids in first-occurrence order inside the batch) and
               numbers its blocks 0 .. T_r - 1 in node order (boundary nodes between two inner ranges become singletons);
  exchange 1   all-gather of the block counts T_r  ->  id offset O_r of every rank (Eq. 4: global id = offset + local id);
  exchange 2   all-gather-v of the block-map slices: every rank holds the block map of the whole graph (4 bytes per node), the
               gather table of its quotient pass;
  quotient     every rank builds the quotient rows of ITS blocks from ITS rows (wl_quotient_rows, Def. 4): the next graph is
               again spread by contiguous node ranges, no edge ever moves between ranks.

The edge partition of later iterations is the inherited one (reading Q14b, WL_FLAG_INHERIT_BATCHES of the single-GPU
path): batch j of the quotient = the blocks whose representative row is complete once batch j of the graph has been read, so a
rank keeps the rows it produced.  The result equals wl_refine_batched(..., WL_FLAG_INHERIT_BATCHES) on the same first cuts.

No data-path arithmetic lives here: the per-batch work is done by a backend (CudaBackend = the C-ABI kernels; the CPU tests
plug in a backend made of the oracle to check the exchange logic with world size 2 on gloo).
"""
from __future__ import annotations

from bisect import bisect_left, bisect_right
from dataclasses import dataclass
from typing import List, Optional

import torch


# ---------------------------------------------------------------------------------------------------------------------
# host logic shared by every backend (no arithmetic of the method)
# ---------------------------------------------------------------------------------------------------------------------
def greedy_cuts(row_ptr: torch.Tensor, cap: int) -> List[int]:
    """Default edge partition (reading Q13): consecutive runs of at most `cap` entries of the CSR edge array, cut on the
    largest row boundary that fits, inside a row only when the row alone exceeds the cap."""
    rp = row_ptr.tolist() if row_ptr.numel() < (1 << 22) else None
    m = int(row_ptr[-1])
    cuts = [0]
    while cuts[-1] < m:
        start, limit = cuts[-1], cuts[-1] + cap
        if limit >= m:
            cuts.append(m)
            break
        if rp is not None:
            r = bisect_right(rp, limit) - 1
            b = rp[r]
        else:
            r = int(torch.searchsorted(row_ptr, torch.tensor(limit), right=True)) - 1
            b = int(row_ptr[r])
        cuts.append(b if b > start else limit)
    if len(cuts) == 1:
        cuts.append(m)
    return cuts


def split_batches_over_ranks(row_ptr: torch.Tensor, cuts: List[int], world: int) -> List[int]:
    """Batch index borders k_0 = 0 <= k_1 <= ... <= k_world = N_b such that rank r owns the batches [k_r, k_{r+1}) and every
    border falls on the start of a NON-EMPTY row (a row cut by a batch border stays inside one rank, and so does a run of
    edgeless nodes that sits on a cut: reading Q14b groups those with the batch that ends there).  Shares are as even as such
    cuts allow; a rank may own nothing."""
    nb = len(cuts) - 1
    rp = row_ptr
    n = rp.numel() - 1
    aligned = [0]
    for k in range(1, nb):
        i = int(torch.searchsorted(rp, torch.tensor(cuts[k]), right=False))  # first node whose row starts at or after the cut
        if i < n and int(rp[i]) == cuts[k] and int(rp[i + 1]) > cuts[k]:
            aligned.append(k)
    aligned.append(nb)
    borders = [0]
    for r in range(1, world):
        want = r * nb / world
        best = min(aligned, key=lambda k: (abs(k - want), k))
        borders.append(max(best, borders[-1]))
    borders.append(nb)
    return borders


@dataclass
class Batch:
    """One batch of the rank's part of the current graph, in GLOBAL node ids and rank-relative edge positions."""
    r0: int          # inner nodes [r0, r1)
    r1: int
    done: int        # nodes [.., done) have their whole row at or before the end of this batch (Q14b grouping)
    index: int       # global batch index (weight stream id)


class ShardState:
    """The part of the current graph one rank owns: the rows of the nodes [n0, n1) as a host CSR (offsets relative to the
    rank's first entry, global target ids) and its batches."""

    def __init__(self, n_total: int, n0: int, n1: int, row_ptr: torch.Tensor, col: torch.Tensor,
                 weights: Optional[torch.Tensor], batches: List[Batch]):
        self.n_total, self.n0, self.n1 = n_total, n0, n1
        self.row_ptr, self.col, self.weights, self.batches = row_ptr, col, weights, batches


def first_iteration_state(n: int, row_ptr: torch.Tensor, col: torch.Tensor, weights: Optional[torch.Tensor], cuts: List[int],
                          rank: int, world: int) -> ShardState:
    """Rank `rank`'s part of the input graph for the edge partition `cuts` (Alg. 2 line 5): its batches, the inner node range of
    each (Def. 5 for row-contiguous batches: the nodes whose row position lies in the batch, minus a last row that crosses its
    end; the last batch owns the trailing edgeless nodes, Q9) and the Q14b grouping of the nodes."""
    rp = row_ptr
    nb = len(cuts) - 1
    borders = split_batches_over_ranks(rp, cuts, world)
    k0, k1 = borders[rank], borders[rank + 1]
    rpl = rp.tolist()

    def inner_range(c0, c1, last):
        a = bisect_left(rpl, c0, 0, n)
        b = n if last else bisect_left(rpl, c1, 0, n)
        if b > a and rpl[b] > c1:
            b -= 1
        return a, max(a, b)

    def node_of_edge_border(c):  # first node whose row starts at or after edge position c
        return bisect_left(rpl, c, 0, n)

    n0 = 0 if k0 == 0 else node_of_edge_border(cuts[k0])
    n1 = n if k1 == nb else node_of_edge_border(cuts[k1])
    if k0 == k1:
        n0 = n1 = (n if k0 == nb else node_of_edge_border(cuts[k0]))
    batches = []
    for k in range(k0, k1):
        a, b = inner_range(cuts[k], cuts[k + 1], k == nb - 1)
        done = n if k == nb - 1 else bisect_right(rpl, cuts[k + 1], 1, n + 1) - 1  # nodes i with rp[i + 1] <= c1
        batches.append(Batch(a, b, min(max(done, b), n1), k))
    e0, e1 = int(rp[n0]), int(rp[n1])
    return ShardState(n, n0, n1, (rp[n0:n1 + 1] - e0).contiguous(), col[e0:e1].contiguous(),
                      None if weights is None else weights[e0:e1].contiguous(), batches)


# ---------------------------------------------------------------------------------------------------------------------
# backends: the per-batch work
# ---------------------------------------------------------------------------------------------------------------------
class CudaBackend:
    """The product path: every step runs in the CUDA kernels behind the C ABI (no CPU fallback)."""

    def __init__(self, device, flags: int = 0, ring_bits: int = 0):
        from . import binding
        self.b, self.device, self.flags, self.ring_bits = binding, torch.device(device), flags, ring_bits

    def _dev(self, t, dtype=None):
        if t is None:
            return None
        t = t.to(self.device, non_blocking=True)
        return t if dtype is None else t.to(dtype)

    def refine_inner(self, row_ptr, col, weights, lo, n_targets, seed, stream_id):
        c, f, k = self.b.wl_refine_inner(self._dev(row_ptr), self._dev(col), self._dev(weights), lo, n_targets, seed,
                                         stream_id=stream_id, flags=self.flags, ring_bits=self.ring_bits)
        return c.cpu(), f.cpu(), k

    def set_block_map(self, block_of: torch.Tensor):
        self.block_of = block_of.to(self.device)

    def quotient_rows(self, row_ptr, col, weights, lo, is_first, first_block, num_blocks):
        q_rp, q_col, q_wt = self.b.wl_quotient_rows(self._dev(row_ptr), self._dev(col), self._dev(weights), lo, self.block_of,
                                                    self._dev(is_first), first_block, num_blocks)
        return q_rp.cpu(), q_col.cpu(), q_wt.cpu()


# ---------------------------------------------------------------------------------------------------------------------
# the driver
# ---------------------------------------------------------------------------------------------------------------------
class ShardedRefiner:
    """One rank of the sharded Algorithm 2.  `step_*` methods are the phases of an outer iteration; `run` strings them
    together with torch.distributed collectives (or none for a single rank)."""

    def __init__(self, backend, n: int, row_ptr, col, weights, max_batch_edges: int, seed: int = 0, rank: int = 0,
                 world: int = 1, cuts: Optional[List[int]] = None):
        self.backend, self.seed, self.rank, self.world = backend, seed, rank, world
        self.n0_total = n
        cuts = greedy_cuts(row_ptr, max_batch_edges) if cuts is None else list(cuts)
        self.nb_total = len(cuts) - 1
        self.state = first_iteration_state(n, row_ptr, col, weights, cuts, rank, world)
        self.map0: Optional[torch.Tensor] = None  # original node -> node of the current graph
        self.outer = 0
        self.boundary_first = 0

    # -- phase 1: local refinement of the own batches, block ids 0 .. T - 1 in node order ---------------------------------
    def step_local(self):
        s = self.state
        self.outer += 1
        nloc = s.n1 - s.n0
        self.h_local = torch.empty(nloc, dtype=torch.int32)
        self.first_local = torch.zeros(nloc, dtype=torch.uint8)
        base, nxt, boundary = 0, s.n0, 0

        def gap(g0, g1):
            nonlocal base, boundary
            if g1 > g0:
                self.h_local[g0 - s.n0:g1 - s.n0] = torch.arange(base, base + g1 - g0, dtype=torch.int32)
                self.first_local[g0 - s.n0:g1 - s.n0] = 1
                base += g1 - g0
                boundary += g1 - g0

        for bt in s.batches:
            gap(nxt, bt.r0)
            nxt = max(nxt, bt.r1)
            if bt.r1 == bt.r0:
                continue
            a, b = int(s.row_ptr[bt.r0 - s.n0]), int(s.row_ptr[bt.r1 - s.n0])
            rp = (s.row_ptr[bt.r0 - s.n0:bt.r1 - s.n0 + 1] - a).contiguous()
            c, f, k = self.backend.refine_inner(rp, s.col[a:b].contiguous(),
                                                None if s.weights is None else s.weights[a:b].contiguous(), bt.r0, s.n_total,
                                                self.seed, (self.outer << 32) | bt.index)
            self.h_local[bt.r0 - s.n0:bt.r1 - s.n0] = c + base
            self.first_local[bt.r0 - s.n0:bt.r1 - s.n0] = f
            base += k
        gap(nxt, s.n1)
        if self.outer == 1:
            self.boundary_first = boundary
        self.t_local = base
        return base

    # -- phase 2: offsets (Eq. 4) and the global block map ----------------------------------------------------------------
    def step_offsets(self, counts: List[int]):
        self.offset = sum(counts[:self.rank])
        self.k_total = sum(counts)
        self.counts = counts
        return self.h_local + self.offset

    def step_block_map(self, block_of: torch.Tensor):
        """block_of: int32 over all nodes of the current graph (the concatenation of every rank's slice)."""
        self.block_of = block_of
        self.map0 = block_of.clone() if self.map0 is None else block_of[self.map0.long()]
        self.backend.set_block_map(block_of)
        s = self.state
        return self.nb_total == 1 or self.k_total == s.n_total  # Alg. 2 line 15 (L200, Q15)

    # -- phase 3: quotient rows of the own blocks; the next graph stays sharded by node range -----------------------------
    def step_quotient(self):
        s = self.state
        q_rp, q_col, q_wt, batches = [torch.zeros(1, dtype=torch.int64)], [], [], []
        node, block, edges = s.n0, self.offset, 0
        cum_first = torch.cumsum(self.first_local.to(torch.int64), 0)
        for j, bt in enumerate(s.batches):
            done = bt.done if j + 1 < len(s.batches) else s.n1
            if done <= node:
                continue
            nblk = int(cum_first[done - s.n0 - 1]) - (int(cum_first[node - s.n0 - 1]) if node > s.n0 else 0)
            a, b = int(s.row_ptr[node - s.n0]), int(s.row_ptr[done - s.n0])
            if nblk > 0:
                rp = (s.row_ptr[node - s.n0:done - s.n0 + 1] - a).contiguous()
                r, c, w = self.backend.quotient_rows(rp, s.col[a:b].contiguous(),
                                                     None if s.weights is None else s.weights[a:b].contiguous(), node,
                                                     self.first_local[node - s.n0:done - s.n0].contiguous(), block, nblk)
                q_rp.append(r[1:] + edges)
                q_col.append(c)
                q_wt.append(w)
                batches.append(Batch(block, block + nblk, block + nblk, len(batches)))
                edges += int(r[-1])
                block += nblk
            node = done
        self.next_rows = (torch.cat(q_rp), torch.cat(q_col) if q_col else torch.zeros(0, dtype=torch.int32),
                          torch.cat(q_wt) if q_wt else torch.zeros(0, dtype=torch.int64), batches)
        return len(batches)

    def step_advance(self, batch_counts: List[int]):
        """batch_counts: number of (non-empty) batches every rank produced; renumbers the batches globally and moves on."""
        rp, col, wt, batches = self.next_rows
        first_index = sum(batch_counts[:self.rank])
        for i, bt in enumerate(batches):
            bt.index = first_index + i
        self.nb_total = sum(batch_counts)
        self.state = ShardState(self.k_total, self.offset, self.offset + self.t_local, rp, col, wt, batches)

    # -- the loop with torch.distributed --------------------------------------------------------------------------------
    def run(self, dist=None, comm_device="cpu", max_outer_iters: int = 1 << 30):
        """Returns (colours of the original nodes int32[n] (canonical), number of colours, outer iterations)."""
        def gather_ints(v):
            if dist is None or self.world == 1:
                return [v]
            t = torch.tensor([v], dtype=torch.int64, device=comm_device)
            out = [torch.zeros_like(t) for _ in range(self.world)]
            dist.all_gather(out, t)
            return [int(x.item()) for x in out]

        def gather_v(local: torch.Tensor, counts: List[int]):
            if dist is None or self.world == 1:
                return local
            mx = max(max(counts), 1)
            pad = torch.zeros(mx, dtype=local.dtype, device=comm_device)
            pad[:local.numel()] = local.to(comm_device)
            out = [torch.zeros_like(pad) for _ in range(self.world)]
            dist.all_gather(out, pad)
            return torch.cat([o[:c] for o, c in zip(out, counts)]).cpu()

        while True:
            t = self.step_local()
            counts = gather_ints(t)
            mine = self.step_offsets(counts)
            sizes = gather_ints(self.state.n1 - self.state.n0)
            stop = self.step_block_map(gather_v(mine, sizes))
            if stop or self.outer >= max_outer_iters:
                break
            nbat = self.step_quotient()
            self.step_advance(gather_ints(nbat))
        return self.map0, self.k_total, self.outer


def refine_batched_sharded(n, row_ptr, col, weights=None, *, max_batch_edges: int, seed: int = 0, cuts=None, dist=None,
                           device=None, flags: int = 0, max_outer_iters: int = 1 << 30):
    """Algorithm 2 with the batches of every outer iteration spread over the ranks of `dist` (torch.distributed, already
    initialised; None = one process).  Every rank passes the same host CSR and gets the same colouring back."""
    rank = dist.get_rank() if dist is not None else 0
    world = dist.get_world_size() if dist is not None else 1
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device())
    backend = CudaBackend(device, flags=flags)
    comm_device = device if (dist is not None and dist.get_backend() == "nccl") else "cpu"
    r = ShardedRefiner(backend, n, row_ptr, col, weights, max_batch_edges, seed, rank, world, cuts)
    return r.run(dist, comm_device, max_outer_iters)
