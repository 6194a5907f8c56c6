"""Seeded synthetic graph generators shared by the oracle tests and the CUDA harness.

This module holds NO arithmetic of the refinement method (no weights, no SpMV, no
relabelling).  It only builds inputs: CSR adjacency structures whose rows are the
out-edges of a node ("a_ij = edges from node i to node j", L49 sums over
row i).  Everything is written with device-agnostic torch ops so that the very same code
produces the same graph on the CPU (oracle tests) and on the GPU (bench at full size).

The recipes follow BASELINE.json `configs` / SURVEY.md §8(d); they stand in for the
paper's PyG / WebGraph datasets (Table 1), which are not available here.

Randomness is a counter-based hash (`gmix`), so a draw depends only on (seed, counter):
no generator state, identical on any device and under any chunking.
"""
from __future__ import annotations

from dataclasses import dataclass
from fractions import Fraction
from typing import Optional

import torch

# ---------------------------------------------------------------------------------------
# counter-based hash (generator-only; NOT the method's weight function)
# constants: floor(frac(sqrt(p)) * 2^64) | 1 for p = 5, 7, 11 (checked in tests)
# ---------------------------------------------------------------------------------------
_K1 = 0x3C6EF372FE94F82B
_K2 = 0xA54FF53A5F1D36F1
_K3 = 0x510E527FADE682D1
_MASK64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Two's-complement reinterpretation of a u64 literal as a python int in int64 range."""
    x &= _MASK64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of an int64 tensor holding u64 bit patterns."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def gmix(x: torch.Tensor) -> torch.Tensor:
    """Bijective 64-bit mixer on int64 tensors (wrap-around arithmetic)."""
    x = (x ^ _lsr(x, 33)) * _s64(_K1)
    x = (x ^ _lsr(x, 29)) * _s64(_K2)
    return x ^ _lsr(x, 32)


def gmix_int(x: int) -> int:
    """Pure-python big-int twin of `gmix` (used to pin the tensor version in tests)."""
    x &= _MASK64
    x = ((x ^ (x >> 33)) * _K1) & _MASK64
    x = ((x ^ (x >> 29)) * _K2) & _MASK64
    return x ^ (x >> 32)


def seed_key(seed: int) -> int:
    return gmix_int((seed + _K3) & _MASK64)


def hash_u32(seed: int, counter: torch.Tensor) -> torch.Tensor:
    """Top 32 bits of gmix(counter + key(seed)) as non-negative int64 in [0, 2^32)."""
    return _lsr(gmix(counter + _s64(seed_key(seed))), 32)


def hash_u32_int(seed: int, counter: int) -> int:
    return gmix_int((counter + seed_key(seed)) & _MASK64) >> 32


# ---------------------------------------------------------------------------------------
@dataclass
class Graph:
    """CSR adjacency, rows = sources.  row_ptr int64[n+1], col int32[m], weights uint32-as-int64? no:
    weights is an int64 tensor with values in [1, 2^32) or None (= all ones)."""
    n: int
    row_ptr: torch.Tensor
    col: torch.Tensor
    weights: Optional[torch.Tensor] = None
    name: str = ""

    @property
    def m(self) -> int:
        return int(self.col.numel())

    def to(self, device) -> "Graph":
        return Graph(self.n, self.row_ptr.to(device), self.col.to(device),
                     None if self.weights is None else self.weights.to(device), self.name)

    def numpy(self):
        import numpy as np
        rp = self.row_ptr.cpu().numpy().astype(np.int64)
        ci = self.col.cpu().numpy().astype(np.int32)
        w = None if self.weights is None else self.weights.cpu().numpy().astype(np.uint32)
        return self.n, rp, ci, w


def csr_from_pairs(n: int, src: torch.Tensor, dst: torch.Tensor, *, dedup: bool = True,
                   name: str = "", weights: Optional[torch.Tensor] = None) -> Graph:
    """Sort (src, dst) pairs into CSR.  dedup=True removes duplicate pairs (weights must be None);
    dedup=False keeps multi-edges as repeated entries (a_ij = multiplicity)."""
    src = src.to(torch.int64)
    dst = dst.to(torch.int64)
    key = src * n + dst
    if dedup:
        assert weights is None
        key = torch.unique(key)  # sorted
        w = None
    else:
        key, order = torch.sort(key, stable=True)
        w = None if weights is None else weights[order].to(torch.int64)
    rows = torch.div(key, n, rounding_mode="floor")
    cols = (key - rows * n).to(torch.int32)
    deg = torch.bincount(rows, minlength=n)
    row_ptr = torch.zeros(n + 1, dtype=torch.int64, device=key.device)
    row_ptr[1:] = torch.cumsum(deg, 0)
    return Graph(n, row_ptr, cols, w, name)


def from_edge_list(n: int, edges, weights=None, name: str = "") -> Graph:
    """Small helper for hand-written test graphs: edges = iterable of (i, j), kept as given
    (duplicates are multi-edges)."""
    edges = list(edges)
    if len(edges) == 0:
        return Graph(n, torch.zeros(n + 1, dtype=torch.int64), torch.zeros(0, dtype=torch.int32),
                     None if weights is None else torch.zeros(0, dtype=torch.int64), name)
    e = torch.tensor(edges, dtype=torch.int64)
    w = None if weights is None else torch.tensor(list(weights), dtype=torch.int64)
    return csr_from_pairs(n, e[:, 0], e[:, 1], dedup=False, weights=w, name=name)


# ---------------------------------------------------------------------------------------
# config 1: directed Erdos-Renyi G(n, m) by rejection of repeats
# ---------------------------------------------------------------------------------------
def erdos_renyi(n: int = 10_000, m: int = 50_000, seed: int = 0, device="cpu") -> Graph:
    """Ordered pairs (u, v), u != v, drawn uniformly from the counter hash; the first m distinct
    pairs in draw order are kept (BASELINE.json configs[0]).  u = h(2t) mod n, v = h(2t+1) mod n."""
    assert m <= n * (n - 1)
    draws = int(m * 1.3) + 64
    while True:
        t = torch.arange(draws, dtype=torch.int64, device=device)
        u = hash_u32(seed, 2 * t) % n
        v = hash_u32(seed, 2 * t + 1) % n
        ok = u != v
        key = (u * n + v)[ok]
        # first occurrence in draw order
        uniq, inv = torch.unique(key, return_inverse=True)
        first = torch.full((uniq.numel(),), key.numel(), dtype=torch.int64, device=device)
        first.scatter_reduce_(0, inv, torch.arange(key.numel(), device=device), reduce="amin")
        if uniq.numel() >= m:
            first_sorted, _ = torch.sort(first)
            keep = key[first_sorted[:m]]
            src = torch.div(keep, n, rounding_mode="floor")
            dst = keep - src * n
            return csr_from_pairs(n, src, dst, dedup=True, name=f"er_n{n}_m{m}_s{seed}")
        draws *= 2


# ---------------------------------------------------------------------------------------
# config 2: s x s grid, both directions per link
# ---------------------------------------------------------------------------------------
def grid2d(s: int = 2048, device="cpu") -> Graph:
    """node id = r*s + c; out-edges to the 4-neighbourhood; m = 4 s (s-1)."""
    idx = torch.arange(s * s, dtype=torch.int64, device=device)
    r = torch.div(idx, s, rounding_mode="floor")
    c = idx - r * s
    srcs, dsts = [], []
    for dr, dc in ((-1, 0), (0, -1), (0, 1), (1, 0)):
        ok = (r + dr >= 0) & (r + dr < s) & (c + dc >= 0) & (c + dc < s)
        srcs.append(idx[ok])
        dsts.append(idx[ok] + dr * s + dc)
    return csr_from_pairs(s * s, torch.cat(srcs), torch.cat(dsts), dedup=True, name=f"grid_{s}x{s}")


def grid2d_orbit_colors(s: int) -> torch.Tensor:
    """Closed form for the coarsest stable colouring of the s x s grid from a uniform start: nodes
    fall into the orbits of the dihedral group of the square, i.e. the unordered pair
    {min(r, s-1-r), min(c, s-1-c)}; h(h+1)/2 classes with h = ceil(s/2).
    Returned in canonical first-occurrence numbering."""
    idx = torch.arange(s * s, dtype=torch.int64)
    r = torch.div(idx, s, rounding_mode="floor")
    c = idx - r * s
    a = torch.minimum(r, s - 1 - r)
    b = torch.minimum(c, s - 1 - c)
    lo, hi = torch.minimum(a, b), torch.maximum(a, b)
    return canonical_first_occurrence(lo * s + hi)


def canonical_first_occurrence(labels: torch.Tensor) -> torch.Tensor:
    """Relabel arbitrary integer labels to 0,1,2,... in order of first occurrence (input helper for
    building initial partitions and closed-form expectations; holds no refinement arithmetic)."""
    labels = labels.to(torch.int64)
    uniq, inv = torch.unique(labels, return_inverse=True)
    n = labels.numel()
    first = torch.full((uniq.numel(),), n, dtype=torch.int64, device=labels.device)
    first.scatter_reduce_(0, inv, torch.arange(n, device=labels.device), reduce="amin")
    order = torch.argsort(first)
    rank = torch.empty_like(order)
    rank[order] = torch.arange(order.numel(), device=labels.device)
    return rank[inv].to(torch.int32)


# ---------------------------------------------------------------------------------------
# configs 3-5: R-MAT
# ---------------------------------------------------------------------------------------
def _rmat_thresholds(a, b, c):
    fa, fb, fc = (Fraction(str(x)) for x in (a, b, c))
    two32 = 1 << 32
    return int(fa * two32), int((fa + fb) * two32), int((fa + fb + fc) * two32)


def rmat_draws(scale: int, lo: int, hi: int, seed: int, abc=(0.57, 0.19, 0.19), device="cpu"):
    """(src, dst) of edge draws lo <= e < hi.  Level l of draw e uses hash counter e*64 + l; the
    quadrant (src bit, dst bit) is (0,0) | (0,1) | (1,0) | (1,1) for r below a | a+b | a+b+c | else.
    Bits are filled from the most significant one.  No noise, no vertex permutation."""
    return rmat_draws_at(scale, torch.arange(lo, hi, dtype=torch.int64, device=device), seed, abc)


def rmat_draws_at(scale: int, e: torch.Tensor, seed: int, abc=(0.57, 0.19, 0.19), levels: Optional[int] = None):
    """(src, dst) of the edge draws with indices `e` (int64 tensor); levels < scale: only the top `levels` bits."""
    ta, tab, tabc = _rmat_thresholds(*abc)
    src = torch.zeros_like(e)
    dst = torch.zeros_like(e)
    for l in range(scale if levels is None else levels):
        r = hash_u32(seed, e * 64 + l)
        sbit = (r >= tab).to(torch.int64)
        dbit = (((r >= ta) & (r < tab)) | (r >= tabc)).to(torch.int64)
        src = (src << 1) | sbit
        dst = (dst << 1) | dbit
    return src, dst


def rmat(scale: int, edge_factor: int = 16, seed: int = 1, symmetrize: bool = True,
         abc=(0.57, 0.19, 0.19), device="cpu", chunk: int = 1 << 26, max_bucket_keys: int = 1 << 29) -> Graph:
    """R-MAT graph with 2^scale nodes and edge_factor*2^scale draws; self-loops dropped, duplicates
    removed, reverse edges added when `symmetrize` (BASELINE.json configs[2..4]).  Built in row-range
    buckets so that scale 27 (about 4e9 directed edges) fits one GPU."""
    n = 1 << scale
    draws = edge_factor * n
    srcs, dsts = [], []
    for lo in range(0, draws, chunk):
        s, d = rmat_draws(scale, lo, min(draws, lo + chunk), seed, abc, device)
        keep = s != d
        srcs.append(s[keep].to(torch.int32))
        dsts.append(d[keep].to(torch.int32))
    src = torch.cat(srcs)
    dst = torch.cat(dsts)
    del srcs, dsts
    # row-range buckets from the pre-dedup row histogram
    cnt = torch.bincount(src.to(torch.int64), minlength=n)
    if symmetrize:
        cnt += torch.bincount(dst.to(torch.int64), minlength=n)
    csum = torch.cumsum(cnt, 0)
    total = int(csum[-1])
    bounds = [0]
    while bounds[-1] < n:
        base = int(csum[bounds[-1] - 1]) if bounds[-1] > 0 else 0
        # last row r with csum[r] - base <= max_bucket_keys (at least one row)
        nxt = int(torch.searchsorted(csum, torch.tensor(base + max_bucket_keys, device=csum.device), right=True))
        bounds.append(min(n, max(nxt, bounds[-1] + 1)))
    del cnt, csum
    deg = torch.zeros(n, dtype=torch.int64, device=device)
    cols = []
    for b0, b1 in zip(bounds[:-1], bounds[1:]):
        sel = (src >= b0) & (src < b1)
        key = src[sel].to(torch.int64) * n + dst[sel].to(torch.int64)
        if symmetrize:
            sel = (dst >= b0) & (dst < b1)
            key = torch.cat([key, dst[sel].to(torch.int64) * n + src[sel].to(torch.int64)])
        del sel
        key = torch.unique(key)
        rows = key >> scale
        cols.append((key & (n - 1)).to(torch.int32))
        if rows.numel():
            deg[b0:b1] = torch.bincount(rows - b0, minlength=b1 - b0)
        del key, rows
    row_ptr = torch.zeros(n + 1, dtype=torch.int64, device=device)
    row_ptr[1:] = torch.cumsum(deg, 0)
    col = torch.cat(cols) if cols else torch.zeros(0, dtype=torch.int32, device=device)
    kind = "sym" if symmetrize else "dir"
    _ = total
    return Graph(n, row_ptr, col, None, f"rmat_s{scale}_ef{edge_factor}_{kind}_seed{seed}")


def rmat_directed_to_host(scale: int, edge_factor: int = 16, seed: int = 1, abc=(0.57, 0.19, 0.19), device="cpu",
                          top_bits: int = 7, chunk: int = 1 << 27, pin: bool = False, col_out=None, row_ptr_out=None):
    """The graph rmat(scale, edge_factor, seed, symmetrize=False) built for sizes that exceed one GPU (BASELINE.json
    configs[4]: scale 30, 17e9 edges): draws are grouped by the top `top_bits` bits of their source (which depend on the first
    `top_bits` levels only), every group is completed, deduplicated and sorted on `device`, and its rows are appended to HOST
    arrays.  Returns (n, row_ptr int64[n+1] host, col int32[m] host view).  Same edges, same order as rmat()."""
    n = 1 << scale
    draws = edge_factor * n
    top_bits = min(top_bits, scale)
    nbuck = 1 << top_bits
    bucket = torch.empty(draws, dtype=torch.uint8 if top_bits <= 8 else torch.int16, device=device)
    for lo in range(0, draws, chunk):
        hi = min(draws, lo + chunk)
        s, _ = rmat_draws_at(scale, torch.arange(lo, hi, dtype=torch.int64, device=device), seed, abc, levels=top_bits)
        bucket[lo:hi] = s.to(bucket.dtype)
    col = torch.empty(draws, dtype=torch.int32, pin_memory=pin) if col_out is None else col_out
    deg = torch.zeros(n, dtype=torch.int64, device=device)
    rows_per_bucket = n >> top_bits
    off = 0
    scan_chunk = max(chunk, 1 << 30)
    for b in range(nbuck):
        idx = []
        for lo in range(0, draws, scan_chunk):
            hi = min(draws, lo + scan_chunk)
            e = torch.nonzero(bucket[lo:hi] == b).flatten()
            if e.numel():
                idx.append(e + lo)
        if not idx:
            continue
        e_all = torch.cat(idx)
        del idx
        keys = []
        for lo in range(0, e_all.numel(), chunk):
            s, d = rmat_draws_at(scale, e_all[lo:lo + chunk], seed, abc)
            keep = s != d
            keys.append(s[keep] * n + d[keep])
            del s, d, keep
        del e_all
        key = torch.unique(torch.cat(keys))  # (torch.unique sorts at most 2^31 keys: top_bits must keep a group below that)
        del keys
        b0 = b * rows_per_bucket
        deg[b0:b0 + rows_per_bucket] = torch.bincount((key >> scale) - b0, minlength=rows_per_bucket)
        cnt = key.numel()
        col[off:off + cnt].copy_((key & (n - 1)).to(torch.int32), non_blocking=False)
        off += cnt
        del key
    row_ptr = torch.zeros(n + 1, dtype=torch.int64, pin_memory=pin) if row_ptr_out is None else row_ptr_out
    row_ptr[0] = 0
    row_ptr[1:] = torch.cumsum(deg, 0).cpu()
    return n, row_ptr, col[:off]


# ---------------------------------------------------------------------------------------
# textbook graphs with closed-form stable colourings (test inputs)
# ---------------------------------------------------------------------------------------
def path_graph(n: int) -> Graph:
    e = [(i, i + 1) for i in range(n - 1)] + [(i + 1, i) for i in range(n - 1)]
    return from_edge_list(n, e, name=f"path_{n}")


def directed_path(n: int) -> Graph:
    return from_edge_list(n, [(i, i + 1) for i in range(n - 1)], name=f"dpath_{n}")


def directed_cycle(n: int) -> Graph:
    return from_edge_list(n, [(i, (i + 1) % n) for i in range(n)], name=f"dcycle_{n}")


def star_graph(k: int) -> Graph:
    e = [(0, i) for i in range(1, k + 1)] + [(i, 0) for i in range(1, k + 1)]
    return from_edge_list(k + 1, e, name=f"star_{k}")


def complete_bipartite(a: int, b: int) -> Graph:
    e = [(i, a + j) for i in range(a) for j in range(b)] + [(a + j, i) for i in range(a) for j in range(b)]
    return from_edge_list(a + b, e, name=f"K_{a}_{b}")


def circulant(n: int, offsets) -> Graph:
    """Undirected circulant graph: every node has the same degree (k-regular)."""
    e = set()
    for i in range(n):
        for o in offsets:
            e.add((i, (i + o) % n))
            e.add(((i + o) % n, i))
    e = {(i, j) for (i, j) in e if i != j}
    return from_edge_list(n, sorted(e), name=f"circulant_{n}")


def random_weighted_digraph(n: int, m: int, seed: int, max_w: int = 3, multi: bool = True) -> Graph:
    """Small random weighted directed multigraph (self-loops allowed) for brute-force tests."""
    t = torch.arange(m, dtype=torch.int64)
    u = hash_u32(seed, 3 * t) % n
    v = hash_u32(seed, 3 * t + 1) % n
    w = hash_u32(seed, 3 * t + 2) % max_w + 1
    g = csr_from_pairs(n, u, v, dedup=False, weights=w, name=f"rwd_n{n}_m{m}_s{seed}")
    if not multi:
        raise NotImplementedError
    return g


def random_partition(n: int, k: int, seed: int) -> torch.Tensor:
    """Random initial partition with at most k classes, canonical numbering (int32[n])."""
    t = torch.arange(n, dtype=torch.int64)
    return canonical_first_occurrence(hash_u32(seed ^ 0x5EED, t) % k)


def permute_graph(g: Graph, perm: torch.Tensor) -> Graph:
    """Renumber nodes: new id of old node i is perm[i]."""
    n, m = g.n, g.m
    deg = g.row_ptr[1:] - g.row_ptr[:-1]
    src = torch.repeat_interleave(torch.arange(n, dtype=torch.int64), deg)
    dst = g.col.to(torch.int64)
    return csr_from_pairs(n, perm[src], perm[dst], dedup=False, weights=g.weights, name=g.name + "_perm")


def random_permutation(n: int, seed: int) -> torch.Tensor:
    t = torch.arange(n, dtype=torch.int64)
    return torch.argsort(hash_u32(seed ^ 0xBEEF, t) * n + t)


# ---------------------------------------------------------------------------------------
# edge partitions for the batched algorithm (inputs of Algorithm 2)
# ---------------------------------------------------------------------------------------
def contiguous_row_batches(g: Graph, max_batch_edges: int):
    """Default partition: cut the CSR edge array into consecutive runs of at
    most M_b edges.  Returns int64 tensor `cuts` with cuts[0]=0, cuts[-1]=m; batch k owns edge
    positions [cuts[k], cuts[k+1]).  A cut falls on a row boundary whenever the row that would be
    split fits into one batch by itself."""
    m = g.m
    rp = g.row_ptr
    cuts = [0]
    while cuts[-1] < m:
        start = cuts[-1]
        limit = start + max_batch_edges
        if limit >= m:
            cuts.append(m)
            break
        # largest row boundary <= limit and > start
        r = int(torch.searchsorted(rp, torch.tensor(limit), right=True)) - 1
        b = int(rp[r])
        cuts.append(b if b > start else limit)
    return torch.tensor(cuts, dtype=torch.int64)


def random_edge_batches(g: Graph, num_batches: int, seed: int) -> torch.Tensor:
    """Arbitrary partition (PAPER.md L163 'arbitrary edge partition'): batch id per CSR edge slot."""
    t = torch.arange(g.m, dtype=torch.int64)
    return (hash_u32(seed ^ 0xBA7C4, t) % num_batches).to(torch.int32)


def edge_sources(g: Graph) -> torch.Tensor:
    """Source node of every CSR edge slot (int32[m])."""
    deg = g.row_ptr[1:] - g.row_ptr[:-1]
    return torch.repeat_interleave(torch.arange(g.n, dtype=torch.int32, device=g.row_ptr.device), deg)


def node_hash_edge_batches(g: Graph, num_batches: int, seed: int, flip_percent: int = 0) -> torch.Tensor:
    """An arbitrary partition with few boundary nodes: every edge goes to the batch its SOURCE hashes to (all nodes inner,
    V_k scattered over the id space), then `flip_percent` % of the edges are moved to a hashed batch of their own (their
    sources become boundary nodes, Def. 5)."""
    t = torch.arange(g.m, dtype=torch.int64)
    src = edge_sources(g).to(torch.int64).cpu()
    eb = hash_u32(seed ^ 0x50DE, src) % num_batches
    if flip_percent > 0:
        flip = (hash_u32(seed ^ 0xF11B, t) % 100) < flip_percent
        eb = torch.where(flip, hash_u32(seed ^ 0xBA7C4, t) % num_batches, eb)
    return eb.to(torch.int32)


def coo_batches(g: Graph, edge_batch: torch.Tensor, num_batches: int):
    """The edge partition `edge_batch` (batch id per CSR slot) as COO triples (src, col, weights or None) per batch."""
    src = edge_sources(g).cpu()
    col = g.col.cpu()
    out = []
    for k in range(num_batches):
        sel = torch.nonzero(edge_batch == k).flatten()
        out.append((src[sel].contiguous(), col[sel].contiguous(),
                    None if g.weights is None else g.weights.cpu()[sel].contiguous()))
    return out
