"""Test-only helpers for paper_2607_02603_b200/sharded.py: a backend made of the CPU oracle (so that the exchange logic can run
on CPU ranks over gloo) and a lock-step runner that plays several virtual ranks in one process."""
import numpy as np
import torch

import oracle


def _u32(weights):
    """host weights as the driver stores them: the caller's integers, or uint32 bit patterns in an int32 tensor"""
    w = weights.numpy()
    return w.view(np.uint32).astype(np.int64) if w.dtype == np.int32 else w.astype(np.int64)


class OracleBackend:
    """The per-batch work of the sharded driver done by the oracle: B3 + B4 as oracle.refine on the explicit local graph (inner
    nodes in one block, every outside target a singleton node, Eq. 3), B6 from Def. 4 with numpy.  Same interface as
    CudaBackend (paper_2607_02603_b200/sharded.py); every array lives on the host."""
    array_device = torch.device("cpu")

    def host_buffers(self, n_rows, m):
        return (torch.empty(n_rows + 1, dtype=torch.int64), torch.empty(n_rows + 1, dtype=torch.int64),
                torch.empty(max(m, 1), dtype=torch.int32), torch.empty(max(m, 1), dtype=torch.int32))

    def prefetch(self, row_ptr, col, weights):
        pass

    def finish(self):
        pass

    def refine_inner(self, row_ptr, rp_base, col, weights, lo, n_targets, seed, stream_id):
        rp, ci = row_ptr.numpy().astype(np.int64) - rp_base, col.numpy().astype(np.int64)
        nr = rp.size - 1
        inside = (ci >= lo) & (ci < lo + nr)
        outs, inv = np.unique(ci[~inside], return_inverse=True)
        loc = np.empty(ci.size, dtype=np.int32)
        loc[inside] = (ci[inside] - lo).astype(np.int32)
        loc[~inside] = (nr + inv).astype(np.int32)
        n_loc = nr + outs.size
        rp_ext = np.concatenate([rp, np.full(outs.size, rp[-1], dtype=np.int64)])
        init = np.concatenate([np.zeros(nr, dtype=np.int32), 1 + np.arange(outs.size, dtype=np.int32)])
        w = None if weights is None else _u32(weights).astype(np.uint32)
        c, _, _ = oracle.refine(n_loc, rp_ext, loc, w, init)
        cin = oracle.canonical(c[:nr])
        first = np.zeros(nr, dtype=np.uint8)
        first[np.unique(cin, return_index=True)[1]] = 1
        return torch.from_numpy(cin), torch.from_numpy(first), int(cin.max()) + 1

    def refine_last_rows(self, lo, n_targets, seed, stream_id):
        rp, col, wt = self._last_rows
        return self.refine_inner(rp, 0, col, wt, lo, n_targets, seed, stream_id)

    def set_block_map(self, block_of):
        self.block_of = block_of.numpy()

    def quotient_rows(self, row_ptr, rp_base, col, weights, lo, is_first, first_block, num_blocks, out_rp, out_col, out_wt,
                      entry_base):
        rp, ci = row_ptr.numpy() - rp_base, col.numpy().copy()  # (the output may overwrite the input: quotients go in place)
        w = np.ones(ci.size, dtype=np.int64) if weights is None else _u32(weights).copy()
        ends, q_col, q_wt = [], [], []
        for i in np.nonzero(is_first.numpy())[0]:
            acc = {}
            for e in range(rp[i], rp[i + 1]):
                b = int(self.block_of[ci[e]])
                acc[b] = acc.get(b, 0) + int(w[e])
            for b in sorted(acc):
                if acc[b]:
                    q_col.append(b)
                    q_wt.append(acc[b])
            ends.append(len(q_col))
        assert len(ends) == num_blocks
        qm = len(q_col)
        self._last_rows = (torch.tensor([0] + ends, dtype=torch.int64), torch.tensor(q_col, dtype=torch.int32),
                           torch.tensor(q_wt, dtype=torch.int64))
        out_rp[:num_blocks] = torch.tensor(ends, dtype=torch.int64) + entry_base
        out_col[:qm] = torch.tensor(q_col, dtype=torch.int32)
        out_wt[:qm] = torch.from_numpy(np.array(q_wt, dtype=np.int64).astype(np.uint32).view(np.int32))
        return qm


def run_lockstep(make_backend, n, row_ptr, col, weights, max_batch_edges, world, seed=0, cuts=None):
    """`world` virtual ranks of the sharded driver in one process, their collectives played by hand."""
    from paper_2607_02603_b200.sharded import ShardedRefiner
    ranks = [ShardedRefiner(make_backend(), n, row_ptr, col, weights, max_batch_edges, seed, r, world, cuts) for r in range(world)]
    while True:
        counts = [r.step_local() for r in ranks]
        slices = [r.step_offsets(counts) for r in ranks]
        block_of = torch.cat(slices)
        stops = [r.step_block_map(block_of) for r in ranks]
        assert len(set(stops)) == 1
        if stops[0]:
            break
        nbat = [r.step_quotient() for r in ranks]
        for r in ranks:
            r.step_advance(nbat)
    for r in ranks[1:]:
        assert torch.equal(r.map0, ranks[0].map0)
    return ranks[0].map0.cpu(), ranks[0].k_total, ranks[0].outer, ranks
