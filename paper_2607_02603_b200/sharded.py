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

Where the data lives.  The rank's part of the current graph stays in HOST memory (pinned for the CUDA backend): it exceeds the
device by assumption (L135).  Iteration 1 reads the caller's arrays; every quotient is written into ONE region of the backend's
host workspace and every later quotient overwrites its predecessor in place (its rows come out in the order of its graph's rows
and never hold more entries, Def. 4, so the write position never passes what has already been uploaded).  Everything that is
per NODE (local block ids, first-node flags, the block map of the whole graph, the composed map of the original nodes) lives on
the backend's array device (the GPU for CudaBackend, where NCCL wants it anyway).  The CUDA backend uploads batch j + 1 on a
copy stream while batch j is being refined, and returns quotient rows on a third stream: one host synchronisation per batch
(the C call reports a count), none for the copies.
"""
from __future__ import annotations

from bisect import bisect_left, bisect_right
from dataclasses import dataclass
from typing import List, Optional

import torch


# ---------------------------------------------------------------------------------------------------------------------
# host logic shared by every backend (no arithmetic of the method)
# ---------------------------------------------------------------------------------------------------------------------
def _at(t: torch.Tensor, i: int) -> int:
    return int(t[i])


def greedy_cuts(row_ptr: torch.Tensor, cap: int) -> List[int]:
    """Default edge partition (reading Q13): consecutive runs of at most `cap` entries of the CSR edge array, cut on the
    largest row boundary that fits, inside a row only when the row alone exceeds the cap."""
    m = _at(row_ptr, -1)
    cuts = [0]
    while cuts[-1] < m:
        start, limit = cuts[-1], cuts[-1] + cap
        if limit >= m:
            cuts.append(m)
            break
        r = int(torch.searchsorted(row_ptr, torch.tensor(limit), right=True)) - 1
        b = _at(row_ptr, r)
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
    if nb > 1:
        c = torch.tensor(cuts[1:nb], dtype=torch.int64)
        first = torch.searchsorted(rp, c, right=False)  # first node whose row starts at or after the cut
        ok = first < n
        fi = torch.clamp(first, max=n - 1)
        ok &= (rp[fi] == c) & (rp[fi + 1] > c)
        aligned += [k + 1 for k in torch.nonzero(ok).flatten().tolist()]
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
    """The part of the current graph one rank owns: the rows of the nodes [n0, n1) as a host CSR and its batches.  row_ptr holds
    the offsets of those rows into col / weights PLUS `rp_base` (iteration 1: views of the caller's arrays, rp_base = the
    rank's first entry; later: the rank's own quotient, rp_base = 0), global target ids."""

    def __init__(self, n_total: int, n0: int, n1: int, row_ptr: torch.Tensor, col: torch.Tensor,
                 weights: Optional[torch.Tensor], batches: List[Batch], rp_base: int = 0):
        self.n_total, self.n0, self.n1 = n_total, n0, n1
        self.row_ptr, self.col, self.weights, self.batches, self.rp_base = row_ptr, col, weights, batches, rp_base

    def entry(self, node: int) -> int:
        """offset of the row of global node `node` (n0 <= node <= n1) into col / weights"""
        return _at(self.row_ptr, node - self.n0) - self.rp_base


def first_iteration_state(n: int, row_ptr: torch.Tensor, col: torch.Tensor, weights: Optional[torch.Tensor], cuts: List[int],
                          rank: int, world: int) -> ShardState:
    """Rank `rank`'s part of the input graph for the edge partition `cuts` (Alg. 2 line 5): its batches, the inner node range of
    each (Def. 5 for row-contiguous batches: the nodes whose row position lies in the batch, minus a last row that crosses its
    end; the last batch owns the trailing edgeless nodes, Q9) and the Q14b grouping of the nodes.  Nothing is copied: the
    state holds views of the caller's arrays."""
    rp = row_ptr
    nb = len(cuts) - 1
    borders = split_batches_over_ranks(rp, cuts, world)
    k0, k1 = borders[rank], borders[rank + 1]
    c = torch.tensor(cuts, dtype=torch.int64)
    # bisect_left over the offsets of the n nodes: first node whose row starts at or after an edge position
    left = torch.searchsorted(rp[:n], c, right=False)
    # number of nodes i with rp[i + 1] <= position
    ends_before = torch.searchsorted(rp[1:], c, right=True)
    left_l, ends_l = left.tolist(), ends_before.tolist()
    rp_at_left = rp[torch.clamp(left, max=n)].tolist()

    def inner_range(k):
        a = left_l[k]
        last = k == nb - 1
        b = n if last else left_l[k + 1]
        if b > a and not last and rp_at_left[k + 1] > cuts[k + 1]:
            b -= 1
        if b > a and last and _at(rp, b) > cuts[k + 1]:
            b -= 1
        return a, max(a, b)

    n0 = 0 if k0 == 0 else left_l[k0]
    n1 = n if k1 == nb else left_l[k1]
    if k0 == k1:
        n0 = n1 = (n if k0 == nb else left_l[k0])
    batches = []
    for k in range(k0, k1):
        a, b = inner_range(k)
        done = n if k == nb - 1 else ends_l[k + 1]
        batches.append(Batch(a, b, min(max(done, b), n1), k))
    e0, e1 = _at(rp, n0), _at(rp, n1)
    return ShardState(n, n0, n1, rp[n0:n1 + 1], col[e0:e1], None if weights is None else weights[e0:e1], batches, rp_base=e0)


# ---------------------------------------------------------------------------------------------------------------------
# backends: the per-batch work.  Interface (the test harness implements it with the oracle):
#   array_device                       where the per-node arrays of the driver live
#   host_buffers(n_rows, m)            -> (row_ptr int64[n_rows + 1] x 2, col int32[m], weights int32[m] = uint32 bit patterns): host
#                                      storage of the quotients (col / weights are overwritten in place, row_ptr alternates)
#   prefetch(row_ptr, col, weights)    hint: these host slices are the arguments of one of the next calls
#   refine_inner(row_ptr, rp_base, col, weights, lo, n_targets, seed, stream_id) -> (colours, is_first, k)   [array_device]
#       rows of the inner nodes [lo, lo + n): row_ptr - rp_base indexes col / weights
#   set_block_map(block_of)            the canonical block map of the whole current graph [array_device]
#   quotient_rows(row_ptr, rp_base, col, weights, lo, is_first, first_block, num_blocks, out_rp, out_col, out_wt, entry_base)
#       -> q_m; writes out_rp[0 .. num_blocks) = entry_base + END offset of every emitted row, out_col / out_wt[0 .. q_m)
#   refine_last_rows(lo, n_targets, seed, stream_id) -> (colours, is_first, k)   [array_device]
#       refine_inner on the rows the last quotient_rows call emitted, while they are still where it made them: they are a batch
#       of the next graph (Q14b), so the next outer iteration needs no upload pass for its local refinement
#   finish()                           everything written into host buffers has landed
# ---------------------------------------------------------------------------------------------------------------------
class CudaBackend:
    """The product path: every step runs in the CUDA kernels behind the C ABI (no CPU fallback).  Uploads run on a copy stream
    one batch ahead of the kernels, quotient rows return on a third stream; host storage is pinned and kept between calls."""

    _host_pool = []  # pinned buffer sets not in use by any backend (pinning costs 0.4 s per GB: kept between calls)

    def __init__(self, device, flags: int = 0, ring_bits: int = 0, host_workspace=None):
        from . import binding
        self.b, self.device, self.flags, self.ring_bits = binding, torch.device(device), flags, ring_bits
        self.array_device = self.device
        self.up = torch.cuda.Stream(self.device)
        self.down = torch.cuda.Stream(self.device)
        self._pre = {}
        self._last_up = None
        self._host_ws = host_workspace
        self._mine = None
        self._pool = None

    def host_buffers(self, n_rows: int, m: int):
        need = (n_rows + 1, n_rows + 1, max(m, 1), max(m, 1))
        if self._host_ws is not None:  # caller-owned pinned bytes: carve the arrays out of it
            ws, off, out = self._host_ws, 0, []
            for cnt, dt, sz in ((need[0], torch.int64, 8), (need[1], torch.int64, 8), (need[2], torch.int32, 4), (need[3], torch.int32, 4)):
                if off + cnt * sz > ws.numel():
                    raise ValueError("host_workspace too small: %d bytes needed" % sharded_host_bytes(n_rows, m))
                out.append(ws[off:off + cnt * sz].view(dt))
                off += (cnt * sz + 255) // 256 * 256
            return tuple(out)
        self.release()
        pool = CudaBackend._host_pool
        fit = [i for i, h in enumerate(pool) if all(t.numel() >= c for t, c in zip(h, need))]
        if fit:
            self._mine = pool.pop(min(fit, key=lambda i: pool[i][2].numel()))
        else:
            if pool:  # too small for this graph: let the largest one go instead of keeping both
                pool.pop(max(range(len(pool)), key=lambda i: pool[i][2].numel()))
            self._mine = (torch.empty(need[0], dtype=torch.int64, pin_memory=True), torch.empty(need[1], dtype=torch.int64, pin_memory=True),
                          torch.empty(need[2], dtype=torch.int32, pin_memory=True), torch.empty(need[3], dtype=torch.int32, pin_memory=True))
        return tuple(h[:c] for h, c in zip(self._mine, need))

    def release(self):
        """hands the pinned quotient storage back to the pool (the driver calls it when a run ends)"""
        if self._pool is not None:
            self._pool.shutdown(wait=True)
            self._pool = None
        if self._mine is not None:
            CudaBackend._host_pool.append(self._mine)
            self._mine = None

    def __del__(self):
        try:
            self.release()
        except Exception:
            pass

    @staticmethod
    def _key(row_ptr, col):
        return (row_ptr.data_ptr(), row_ptr.numel(), col.data_ptr(), col.numel())

    def prefetch(self, row_ptr, col, weights):
        if self._key(row_ptr, col) in self._pre:
            return
        with torch.cuda.stream(self.up):
            d = []
            for t in (row_ptr, col, weights):
                if t is None:
                    d.append(None)
                else:
                    d.append(t.to(self.device, non_blocking=True))
            d = tuple(d)
            ev = torch.cuda.Event()
            ev.record(self.up)
        self._pre[self._key(row_ptr, col)] = (d, ev)
        self._last_up = ev

    def _take(self, row_ptr, col, weights):
        self.prefetch(row_ptr, col, weights)
        d, ev = self._pre.pop(self._key(row_ptr, col))
        cur = torch.cuda.current_stream(self.device)
        cur.wait_event(ev)
        for t in d:
            if t is not None:
                t.record_stream(cur)
        return d

    def refine_inner(self, row_ptr, rp_base, col, weights, lo, n_targets, seed, stream_id):
        drp, dcol, dw = self._take(row_ptr, col, weights)
        if rp_base:
            drp = drp - rp_base
        return self.b.wl_refine_inner(drp, dcol, dw, lo, n_targets, seed, stream_id=stream_id, flags=self.flags,
                                      ring_bits=self.ring_bits)

    def set_block_map(self, block_of: torch.Tensor):
        self.block_of = block_of

    def quotient_rows(self, row_ptr, rp_base, col, weights, lo, is_first, first_block, num_blocks, out_rp, out_col, out_wt,
                      entry_base):
        drp, dcol, dw = self._take(row_ptr, col, weights)
        if rp_base:
            drp = drp - rp_base
        q_rp, q_col, q_wt, qm = self.b.wl_quotient_rows(drp, dcol, dw, lo, self.block_of, is_first, first_block, num_blocks,
                                                        raw=True)
        cur = torch.cuda.current_stream(self.device)
        self.down.wait_stream(cur)
        if self._last_up is not None:  # quotients overwrite their graph in place: what is being uploaded is read first
            self.down.wait_event(self._last_up)
        with torch.cuda.stream(self.down):
            ends = q_rp[1:] + entry_base
            out_rp[:num_blocks].copy_(ends, non_blocking=True)
            out_col[:qm].copy_(q_col[:qm], non_blocking=True)
            out_wt[:qm].copy_(q_wt[:qm], non_blocking=True)
        for t in (q_rp, q_col, q_wt):
            t.record_stream(self.down)
        self._last_rows = (q_rp, q_col[:qm], q_wt[:qm])
        return qm

    def refine_last_rows(self, lo, n_targets, seed, stream_id):
        """Runs on a worker thread and a stream of its own (the C call synchronises its stream once per round; ctypes drops the
        GIL for it), so the quotient rows of the NEXT batch are built meanwhile.  Returns a future of (colours, is_first, k)."""
        q_rp, q_col, q_wt = self._last_rows
        self._last_rows = None
        ev = torch.cuda.Event()
        ev.record(torch.cuda.current_stream(self.device))
        if self._pool is None:
            from concurrent.futures import ThreadPoolExecutor
            self._pool = ThreadPoolExecutor(max_workers=1)
            self.side = torch.cuda.Stream(self.device)

        def work():
            with torch.cuda.device(self.device), torch.cuda.stream(self.side):
                self.side.wait_event(ev)
                for t in (q_rp, q_col, q_wt):
                    t.record_stream(self.side)
                return self.b.wl_refine_inner(q_rp, q_col, q_wt, lo, n_targets, seed, stream_id=stream_id, flags=self.flags,
                                              ring_bits=self.ring_bits)
        return self._pool.submit(work)

    def finish(self):
        self.down.synchronize()


def sharded_host_bytes(n_rows: int, m: int) -> int:
    """bytes of pinned host workspace CudaBackend(host_workspace=...) needs for a rank that owns n_rows nodes and m entries"""
    r = lambda x: (x + 255) // 256 * 256
    return 2 * r(8 * (n_rows + 1)) + r(4 * max(m, 1)) + r(4 * max(m, 1))


# ---------------------------------------------------------------------------------------------------------------------
# the driver
# ---------------------------------------------------------------------------------------------------------------------
class ShardedRefiner:
    """One rank of the sharded Algorithm 2.  `step_*` methods are the phases of an outer iteration; `run` strings them
    together with torch.distributed collectives (or none for a single rank)."""

    def __init__(self, backend, n: int, row_ptr, col, weights, max_batch_edges: int, seed: int = 0, rank: int = 0,
                 world: int = 1, cuts: Optional[List[int]] = None):
        self.backend, self.seed, self.rank, self.world = backend, seed, rank, world
        self.adev = backend.array_device
        self.n0_total = n
        cuts = greedy_cuts(row_ptr, max_batch_edges) if cuts is None else list(cuts)
        self.nb_total = len(cuts) - 1
        self.state = first_iteration_state(n, row_ptr, col, weights, cuts, rank, world)
        self.map0: Optional[torch.Tensor] = None  # original node -> node of the current graph [array device]
        self.outer = 0
        self.boundary_first = 0
        self.host = None  # (row_ptr x 2, col, weights) host storage of the rank's quotients, made when first needed
        self.pre_refined = None

    def _slices(self, node0: int, node1: int):
        """host views of the rows of the nodes [node0, node1) of the own part: (row_ptr slice, its base, col, weights)"""
        s = self.state
        a, b = s.entry(node0), s.entry(node1)
        return (s.row_ptr[node0 - s.n0:node1 - s.n0 + 1], a + s.rp_base, s.col[a:b], None if s.weights is None else s.weights[a:b])

    # -- phase 1: local refinement of the own batches, block ids 0 .. T - 1 in node order ---------------------------------
    def step_local(self):
        s = self.state
        self.outer += 1
        nloc = s.n1 - s.n0
        self.h_local = torch.empty(nloc, dtype=torch.int32, device=self.adev)
        self.first_local = torch.zeros(nloc, dtype=torch.uint8, device=self.adev)
        base, nxt, boundary = 0, s.n0, 0

        def gap(g0, g1):
            nonlocal base, boundary
            if g1 > g0:
                self.h_local[g0 - s.n0:g1 - s.n0] = torch.arange(base, base + g1 - g0, dtype=torch.int32, device=self.adev)
                self.first_local[g0 - s.n0:g1 - s.n0] = 1
                base += g1 - g0
                boundary += g1 - g0

        pre = self.pre_refined  # made by the previous iteration's quotient pass: (colours, is_first, k) per batch
        self.pre_refined = None
        if pre is not None:
            for bt, (c, f, k) in zip(s.batches, pre):
                self.h_local[bt.r0 - s.n0:bt.r1 - s.n0] = c + base
                self.first_local[bt.r0 - s.n0:bt.r1 - s.n0] = f
                base += k
            self.t_local = base
            return base
        work = [bt for bt in s.batches if bt.r1 > bt.r0]
        args = [self._slices(bt.r0, bt.r1) for bt in work]
        if args:
            self.backend.prefetch(args[0][0], args[0][2], args[0][3])
        wi = 0
        for bt in s.batches:
            gap(nxt, bt.r0)
            nxt = max(nxt, bt.r1)
            if bt.r1 == bt.r0:
                continue
            rp, rp_base, col, wt = args[wi]
            if wi + 1 < len(args):  # the next batch travels while this one is refined
                self.backend.prefetch(args[wi + 1][0], args[wi + 1][2], args[wi + 1][3])
            wi += 1
            c, f, k = self.backend.refine_inner(rp, rp_base, col, wt, bt.r0, s.n_total, self.seed, (self.outer << 32) | bt.index)
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
        """block_of: int32 over all nodes of the current graph (the concatenation of every rank's slice), on the array device."""
        self.block_of = block_of
        self.map0 = block_of.clone() if self.map0 is None else block_of[self.map0.long()]
        self.backend.set_block_map(block_of)
        s = self.state
        return self.nb_total == 1 or self.k_total == s.n_total  # Alg. 2 line 15 (L200, Q15)

    # -- phase 3: quotient rows of the own blocks; the next graph stays sharded by node range -----------------------------
    def step_quotient(self):
        s = self.state
        # plan first (every offset is read from the host arrays BEFORE any quotient row is written over them)
        groups, node = [], s.n0
        for j, bt in enumerate(s.batches):
            done = bt.done if j + 1 < len(s.batches) else s.n1
            if done > node:
                groups.append((node, done))
                node = done
        cum_first = torch.cumsum(self.first_local.to(torch.int64), 0)
        if groups:
            idx = torch.tensor([g[1] - s.n0 - 1 for g in groups], dtype=torch.int64, device=self.adev)
            upto = [0] + cum_first[idx].tolist()
        else:
            upto = [0]
        plan = []
        for gi, (g0, g1) in enumerate(groups):
            nblk = upto[gi + 1] - upto[gi]
            if nblk > 0:
                plan.append((g0, g1, nblk, self._slices(g0, g1)))
        del cum_first
        if self.host is None:  # sized by the first graph: a quotient never has more rows or entries than its graph (Def. 4)
            self.host = self.backend.host_buffers(s.n1 - s.n0, s.col.numel())
        rp_out = self.host[self.outer & 1]
        col_out, wt_out = self.host[2], self.host[3]
        rp_out[0] = 0
        batches, refined, block, edges = [], [], self.offset, 0
        if plan:
            self.backend.prefetch(plan[0][3][0], plan[0][3][2], plan[0][3][3])
        for pi, (g0, g1, nblk, (rp, rp_base, col, wt)) in enumerate(plan):
            if pi + 1 < len(plan):
                nx = plan[pi + 1][3]
                self.backend.prefetch(nx[0], nx[2], nx[3])
            b0 = block - self.offset
            qm = self.backend.quotient_rows(rp, rp_base, col, wt, g0, self.first_local[g0 - s.n0:g1 - s.n0], block, nblk,
                                            rp_out[1 + b0:1 + b0 + nblk], col_out[edges:], wt_out[edges:], edges)
            # the rows just emitted are batch len(batches) of the next graph (k_total nodes): refined while still in place
            refined.append(self.backend.refine_last_rows(block, self.k_total, self.seed,
                                                         ((self.outer + 1) << 32) | (self.rank << 24) | len(batches)))
            batches.append(Batch(block, block + nblk, block + nblk, len(batches)))
            edges += qm
            block += nblk
        self.backend.finish()
        self.pre_refined = [r.result() if hasattr(r, "result") else r for r in refined]
        nblocks = block - self.offset
        self.next_rows = (rp_out[:nblocks + 1], col_out[:edges], wt_out[:edges], batches)
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
        """Returns (colours of the original nodes int32[n] (canonical, host), number of colours, outer iterations)."""
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
            return torch.cat([o[:c] for o, c in zip(out, counts)]).to(self.adev)

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
        result = self.map0.cpu()
        if hasattr(self.backend, "release"):
            self.backend.release()
        return result, self.k_total, self.outer


def refine_batched_sharded(n, row_ptr, col, weights=None, *, max_batch_edges: int, seed: int = 0, cuts=None, dist=None,
                           device=None, flags: int = 0, max_outer_iters: int = 1 << 30, host_workspace=None):
    """Algorithm 2 with the batches of every outer iteration spread over the ranks of `dist` (torch.distributed, already
    initialised; None = one process).  Every rank passes the same host CSR (pinned recommended) and gets the same colouring
    back.  host_workspace (optional): pinned uint8 tensor of sharded_host_bytes(rows, entries of the rank's part) bytes for
    the rank's quotients; without it the backend pins its own and keeps it for later calls."""
    rank = dist.get_rank() if dist is not None else 0
    world = dist.get_world_size() if dist is not None else 1
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device())
    backend = CudaBackend(device, flags=flags, host_workspace=host_workspace)
    comm_device = device if (dist is not None and dist.get_backend() == "nccl") else "cpu"
    r = ShardedRefiner(backend, n, row_ptr, col, weights, max_batch_edges, seed, rank, world, cuts)
    return r.run(dist, comm_device, max_outer_iters)
