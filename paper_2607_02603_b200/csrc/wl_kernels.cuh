// Kernels of the single-batch path.  sm_100a, integer-only.
#pragma once
#include "wl_device.cuh"

namespace wl {

constexpr int kSpmvThreads = 256;
constexpr int kSpmvIpt = 7;  // odd: 64-bit shared-memory reads at stride IPT are bank-conflict free
constexpr int kSpmvTile = kSpmvThreads * kSpmvIpt;
constexpr u32 kNone = 0xffffffffu;
constexpr int kHubChunk = 4096;  // entries per CTA of spmv_hub_kernel
constexpr int kHubThreads = 256;
constexpr u32 kWinBit = 0x80000000u;


// ---------------------------------------------------------------------------------------------------------------------
// S0: validation of the CSR (WL_EINVAL / WL_ERANGE conditions of include/wl_refine.h)
// ---------------------------------------------------------------------------------------------------------------------
// Offsets may start anywhere (a batch slice indexes the batch's column buffer through a shifted pointer): the caller
// says which first / last offset it expects (0 and m for a whole graph).
__global__ void validate_rows_kernel(int64_t n, const int64_t* __restrict__ row_ptr, const u32* __restrict__ wt,
                                     int64_t expect_first, int64_t expect_last, u32* __restrict__ err) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int64_t a = row_ptr[i], b = row_ptr[i + 1];
  u32 e = 0;
  if (i == 0 && a != expect_first) e |= kErrRowPtr;
  if (i == n - 1 && b != expect_last) e |= kErrRowPtr;
  if (a > b || a < expect_first || b > expect_last) e |= kErrRowPtr;
  if (!e) {
    if (wt) {
      u64 s = 0;
      for (int64_t p = a; p < b; ++p) s += wt[p];
      if (s >= (1ull << 32)) e |= kErrRowSum;  // quotient weights are row-sum bounded and travel as uint32
    } else if ((u64)(b - a) >= (1ull << 32)) {
      e |= kErrRowSum;
    }
  }
  if (e) atomicOr(err, e);
}

// every stored target must be a node id in [0, n_targets); entries [begin, m) of col are checked
__global__ void validate_cols_kernel(int64_t n_targets, int64_t begin, int64_t m, const int* __restrict__ col,
                                     u32* __restrict__ err) {
  const int64_t n = n_targets;
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  bool bad = false;
  for (int64_t p = begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < m; p += stride) {
    int c = col[p];
    bad |= (c < 0) | ((int64_t)c >= n);
  }
  if (bad) atomicOr(err, kErrCol);
}

// ---------------------------------------------------------------------------------------------------------------------
// S0: merge-path tile starts.  The path merges the n row ends (row_ptr[1..n]) with the m entry indices; tile t starts
// at diagonal t*T.  tile_row[t] = number of row ends consumed before that diagonal.
// ---------------------------------------------------------------------------------------------------------------------
__global__ void tile_search_kernel(int64_t n, int64_t m, const int64_t* __restrict__ row_ptr, int64_t ntiles,
                                   int* __restrict__ tile_row) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t > ntiles) return;
  int64_t d = t * (int64_t)kSpmvTile;
  if (d > n + m) d = n + m;
  int64_t lo = d > m ? d - m : 0, hi = d < n ? d : n;
  while (lo < hi) {
    int64_t mid = (lo + hi) >> 1;
    if (row_ptr[mid + 1] <= d - 1 - mid)
      lo = mid + 1;
    else
      hi = mid;
  }
  tile_row[t] = (int)lo;
}

// ---------------------------------------------------------------------------------------------------------------------
// S1+S2, edge-balanced: y_i = sum_j a_ij * w(colour_j)  (Alg. 1 line 5, L120), weights inline from the colour id.
// One CTA owns kSpmvTile consecutive items of the merge path (row ends + entries), so work per CTA is equal whatever
// the degree distribution.  Phase 1 streams the tile's column indices coalesced, gathers the colour of every target and
// leaves a_ij*w in shared memory.  Phase 2 gives every thread IPT consecutive path items: it walks them sequentially and
// flushes each row segment with one no-return 64-bit add at L2.  y must be zero before the launch.
// ---------------------------------------------------------------------------------------------------------------------
template <bool WEIGHTED>
__global__ void __launch_bounds__(kSpmvThreads)
spmv_merge_kernel(int64_t n, int64_t m, const int64_t* __restrict__ row_ptr, const int* __restrict__ col,
                  const u32* __restrict__ wt, const int* __restrict__ colour, u64 key,
                  const int* __restrict__ tile_row, u64* __restrict__ y) {
  __shared__ u64 s_val[kSpmvTile];
  __shared__ int s_rowend[kSpmvTile + 1];
  const int tid = threadIdx.x;
  const int64_t tile = blockIdx.x;
  const int64_t d0 = tile * (int64_t)kSpmvTile;
  const int64_t total = n + m;
  const int64_t d1 = d0 + kSpmvTile < total ? d0 + kSpmvTile : total;
  const int64_t i0 = tile_row[tile], i1 = tile_row[tile + 1];
  const int64_t j0 = d0 - i0, j1 = d1 - i1;
  const int nrows = (int)(i1 - i0);  // row ends inside the tile
  const int nnz = (int)(j1 - j0);    // entries inside the tile

  for (int r = tid; r <= nrows; r += kSpmvThreads) {
    int64_t re = (i0 + r < n) ? row_ptr[i0 + r + 1] - j0 : (int64_t)kSpmvTile + 1;
    s_rowend[r] = re > kSpmvTile + 1 ? kSpmvTile + 1 : (int)re;
  }
  {
    int cidx[kSpmvIpt];
    u32 a[kSpmvIpt];
#pragma unroll
    for (int k = 0; k < kSpmvIpt; ++k) {
      int idx = tid + k * kSpmvThreads;
      cidx[k] = idx < nnz ? ld_stream_i32(col + j0 + idx) : -1;
      if (WEIGHTED) a[k] = idx < nnz ? ld_stream_u32(wt + j0 + idx) : 0u;
    }
    int cc[kSpmvIpt];
#pragma unroll
    for (int k = 0; k < kSpmvIpt; ++k) cc[k] = cidx[k] >= 0 ? __ldg(colour + cidx[k]) : 0;
#pragma unroll
    for (int k = 0; k < kSpmvIpt; ++k) {
      int idx = tid + k * kSpmvThreads;
      if (idx < nnz) {
        u64 w = weight_of(key, (u64)(u32)cc[k]);
        if (WEIGHTED) w *= (u64)a[k];
        s_val[idx] = w;
      }
    }
  }
  __syncthreads();

  const int items = (int)(d1 - d0);
  int d = tid * kSpmvIpt;
  if (d > items) d = items;
  int dend = d + kSpmvIpt;
  if (dend > items) dend = items;
  int lo = d > nnz ? d - nnz : 0, hi = d < nrows ? d : nrows;
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    if (s_rowend[mid] <= d - 1 - mid)
      lo = mid + 1;
    else
      hi = mid;
  }
  int ri = lo, vj = d - lo;
  int rend = s_rowend[ri];
  u64 acc = 0;
  for (int it = d; it < dend; ++it) {
    if (rend <= vj) {  // row i0+ri ends here
      if (acc) red_add_u64(y + i0 + ri, acc);
      acc = 0;
      ++ri;
      rend = s_rowend[ri];
    } else {
      acc += s_val[vj];
      ++vj;
    }
  }
  if (acc) red_add_u64(y + i0 + ri, acc);
}

// Colour id of target node j.  Plain RSC: the dense id colour[j].  Batched local RSC (RANGED): nodes of V_k = [lo, hi)
// carry dense ids (< 2^32) in colour[j - lo]; every other node is an implicit singleton of H_k^0 (Eq. 3) whose id
// is 2^32 + j, a domain disjoint from the dense ids, so all weights stay pairwise distinct.
template <bool RANGED, typename CT>
__device__ __forceinline__ u64 colour_id(const CT* __restrict__ colour, int j, int lo, int hi) {
  if (RANGED) {
    if (j >= lo && j < hi) return (u64)__ldg(colour + (j - lo));
    return (1ull << 32) + (u64)(u32)j;
  }
  return (u64)__ldg(colour + j);
}

// S1+S2, default kernel: one warp owns 32 consecutive rows (or 32 entries of the active row list).
//   * rows with at most kSmallRow entries are summed by their own lane (thread per row, no shuffles, up to kSmallRow
//     independent gathers in flight per lane);
//   * rows of up to kMidRow entries are summed four at a time by groups of eight lanes (up to eight gathers in flight
//     per lane, three-step butterfly per group);
//   * longer rows are processed one after the other by the whole warp (coalesced column loads, four gathers in flight
//     per lane, the last partial step predicated so that its gathers are in flight together, butterfly reduction);
//   * rows longer than hub_threshold are left to spmv_hub_kernel (y = 0 here).
// Everything accumulates in registers: the divergent gathers and shared-memory traffic share the LSU pipe, and staging
// through shared memory (spmv_merge_kernel) more than doubled the time on B200 (profiles/).
// CT = int or unsigned short (narrow colour ids while k <= 65536: the gathered array is half the size and a 32-byte
// sector holds 16 nodes; measured 267 vs 125 G gathers/s on the scale-27 access pattern).
constexpr int kSmallRow = 8;
constexpr int kMidRow = 64;  // rows up to this length are summed by eight lanes

// clamps a column id that is not a node of [0, n_targets) and remembers that it saw one (VALIDATE: S0's range check)
template <bool VALIDATE>
__device__ __forceinline__ int checked_col(int c, int64_t n_targets, bool& bad) {
  if (VALIDATE && (unsigned)c >= (unsigned)n_targets) {
    bad = true;
    return 0;
  }
  return c;
}

// Hot-id table (lever (b) of profiles/r2_gather_microbench.md): a direct-mapped table {tag:16 | colour:16} of kTagSlots entries in
// shared memory, filled with the highest-degree nodes.  tag_mix is a bijection of the id space [0, 2^b), so (slot, tag) =
// (low kTagBits bits, remaining bits) of the mixed id identify the node exactly: a hit costs one LDS instead of an L1-miss sector
// request, a miss falls through to the global gather.
constexpr int kTagBits = 15;
constexpr u32 kTagSlots = 1u << kTagBits;
constexpr u32 kTagEmpty = 0xffffffffu;  // tag 0xffff never occurs: ids have at most 30 bits when the table is used
__host__ __device__ __forceinline__ u32 tag_mix(u32 x, u32 idmask) {
  x ^= x >> 14;
  x = (x * 0x2c1b3c6du) & idmask;
  x ^= x >> 13;
  x = (x * 0x297a2d39u) & idmask;
  x ^= x >> 14;
  return x;
}

template <bool RANGED, bool TAG, typename CT>
__device__ __forceinline__ u64 colour_lookup(const CT* __restrict__ colour, int j, int lo, int hi, const u32* s_tag, u32 idmask) {
  if (TAG) {
    const u32 m = tag_mix((u32)j, idmask);
    const u32 e = s_tag[m & (kTagSlots - 1)];
    if ((e >> 16) == (m >> kTagBits)) return (u64)(e & 0xffffu);
    return (u64)__ldg(colour + j);
  }
  return colour_id<RANGED>(colour, j, lo, hi);
}

// the 32 rows base .. base + 31 of the list (see spmv_rows32_kernel)
// DUAL: rows of at most kMidRow entries are also summed under a second key into y2 (the gathers are shared): the finality test
// of compact_active_kernel wants two independent sums before it lets a block leave for good.
template <bool WEIGHTED, typename CT, bool RANGED, bool VALIDATE, bool TAG, bool DUAL = false>
__device__ __forceinline__ void
rows32_group(const int64_t base, const int lane, int64_t nrows, const int* __restrict__ rows,
             const int64_t* __restrict__ row_ptr, const int* __restrict__ col, const u32* __restrict__ wt,
             const CT* __restrict__ colour, u64 key, u64* __restrict__ y, int64_t hub_threshold, int lo, int hi,
             int64_t n_targets, bool& bad, const u32* s_tag, u32 idmask, u64 key2 = 0, u64* __restrict__ y2 = nullptr,
             bool hub_store = true) {
  const int64_t idx = base + lane;
  const bool valid = idx < nrows;
  int64_t i = 0, a = 0, b = 0;
  if (valid) {
    i = rows ? (int64_t)rows[idx] : idx;
    a = row_ptr[i];
    b = row_ptr[i + 1];
  }
  const int64_t d = b - a;
  const bool small = d <= kSmallRow;
  u64 acc = 0, acc2 = 0;
  {
    const int dd = small ? (int)d : 0;
    int cidx[kSmallRow];
#pragma unroll
    for (int t = 0; t < kSmallRow; ++t) cidx[t] = t < dd ? checked_col<VALIDATE>(__ldg(col + a + t), n_targets, bad) : -1;
#pragma unroll
    for (int t = 0; t < kSmallRow; ++t) {
      if (cidx[t] != -1) {  // -1 = no entry; other negative values are renamed outside targets (RANGED, wl_batched.cu)
        const u64 cid = colour_lookup<RANGED, TAG>(colour, cidx[t], lo, hi, s_tag, idmask);
        u64 v = weight_of(key, cid);
        if (WEIGHTED) v *= (u64)__ldg(wt + a + t);
        acc += v;
        if (DUAL) acc2 += weight_of(key2, cid);
      }
    }
  }
  unsigned big = __ballot_sync(0xffffffffu, valid && !small && d <= hub_threshold);
  {
    // rows of kSmallRow+1 .. kMidRow entries: four at a time, eight lanes each, up to eight gathers in flight per lane
    unsigned med = __ballot_sync(0xffffffffu, valid && !small && d <= kMidRow);
    big &= ~med;
    const int sub = lane & 7, grp = lane >> 3;
    while (med) {
      unsigned mm = med;
      for (int q = 0; q < grp; ++q) mm &= mm - 1;
      const int src = mm ? __ffs(mm) - 1 : -1;
#pragma unroll
      for (int q = 0; q < 4; ++q) med &= med - 1;
      int64_t ra = __shfl_sync(0xffffffffu, a, src < 0 ? 0 : src), rb = __shfl_sync(0xffffffffu, b, src < 0 ? 0 : src);
      if (src < 0) ra = rb = 0;
      int c[kMidRow / 8];
#pragma unroll
      for (int t = 0; t < kMidRow / 8; ++t) {
        const int64_t p = ra + sub + 8 * t;
        c[t] = p < rb ? checked_col<VALIDATE>(ld_stream_i32(col + p), n_targets, bad) : -1;
      }
      u64 s = 0, s2 = 0;
#pragma unroll
      for (int t = 0; t < kMidRow / 8; ++t) {
        if (c[t] != -1) {
          const u64 cid = colour_lookup<RANGED, TAG>(colour, c[t], lo, hi, s_tag, idmask);
          u64 v = weight_of(key, cid);
          if (WEIGHTED) v *= (u64)ld_stream_u32(wt + ra + sub + 8 * t);
          s += v;
          if (DUAL) s2 += weight_of(key2, cid);
        }
      }
      s += __shfl_xor_sync(0xffffffffu, s, 1);
      s += __shfl_xor_sync(0xffffffffu, s, 2);
      s += __shfl_xor_sync(0xffffffffu, s, 4);
      if (DUAL) {
        s2 += __shfl_xor_sync(0xffffffffu, s2, 1);
        s2 += __shfl_xor_sync(0xffffffffu, s2, 2);
        s2 += __shfl_xor_sync(0xffffffffu, s2, 4);
      }
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        const int sg = __shfl_sync(0xffffffffu, src, g * 8);
        const u64 vg = __shfl_sync(0xffffffffu, s, g * 8);
        if (lane == sg) acc = vg;
        if (DUAL) {
          const u64 vg2 = __shfl_sync(0xffffffffu, s2, g * 8);
          if (lane == sg) acc2 = vg2;
        }
      }
    }
  }
  while (big) {
    const int src = __ffs(big) - 1;
    big &= big - 1;
    const int64_t ra = __shfl_sync(0xffffffffu, a, src), rb = __shfl_sync(0xffffffffu, b, src);
    u64 s = 0;
    int64_t p = ra + lane;
    for (; p + 96 < rb; p += 128) {  // four independent gathers in flight per lane
      const int c0 = checked_col<VALIDATE>(ld_stream_i32(col + p), n_targets, bad),
                c1 = checked_col<VALIDATE>(ld_stream_i32(col + p + 32), n_targets, bad),
                c2 = checked_col<VALIDATE>(ld_stream_i32(col + p + 64), n_targets, bad),
                c3 = checked_col<VALIDATE>(ld_stream_i32(col + p + 96), n_targets, bad);
      u64 v0 = weight_of(key, colour_lookup<RANGED, TAG>(colour, c0, lo, hi, s_tag, idmask)),
          v1 = weight_of(key, colour_lookup<RANGED, TAG>(colour, c1, lo, hi, s_tag, idmask)),
          v2 = weight_of(key, colour_lookup<RANGED, TAG>(colour, c2, lo, hi, s_tag, idmask)),
          v3 = weight_of(key, colour_lookup<RANGED, TAG>(colour, c3, lo, hi, s_tag, idmask));
      if (WEIGHTED) {
        v0 *= (u64)ld_stream_u32(wt + p);
        v1 *= (u64)ld_stream_u32(wt + p + 32);
        v2 *= (u64)ld_stream_u32(wt + p + 64);
        v3 *= (u64)ld_stream_u32(wt + p + 96);
      }
      s += (v0 + v1) + (v2 + v3);
    }
    if (p < rb) {  // fewer than 128 entries left: one predicated step, all gathers in flight together
      int c[4];
#pragma unroll
      for (int t = 0; t < 4; ++t)
        c[t] = p + 32 * t < rb ? checked_col<VALIDATE>(ld_stream_i32(col + p + 32 * t), n_targets, bad) : -1;
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        if (c[t] != -1) {
          u64 v = weight_of(key, colour_lookup<RANGED, TAG>(colour, c[t], lo, hi, s_tag, idmask));
          if (WEIGHTED) v *= (u64)ld_stream_u32(wt + p + 32 * t);
          s += v;
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == src) acc = s;
  }
  // (hub_store == false: the hub kernel runs NEXT TO this one on a second stream and adds into y[i], zeroed beforehand)
  if (valid && (hub_store || d <= hub_threshold)) y[i] = acc;
  if (DUAL && valid && d <= kMidRow) y2[i] = acc2;
}

template <bool WEIGHTED, typename CT, bool RANGED, bool VALIDATE, bool DUAL = false>
__global__ void __launch_bounds__(256)
spmv_rows32_kernel(int64_t nrows, const int* __restrict__ rows, const int64_t* __restrict__ row_ptr,
                   const int* __restrict__ col, const u32* __restrict__ wt, const CT* __restrict__ colour, u64 key,
                   u64* __restrict__ y, int64_t hub_threshold, int lo, int hi, int64_t n_targets,
                   u32* __restrict__ err, u64 key2 = 0, u64* __restrict__ y2 = nullptr, int hub_store = 1) {
  const int lane = threadIdx.x & 31;
  const int64_t base = (((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5) << 5;
  if (base >= nrows) return;
  bool bad = false;
  rows32_group<WEIGHTED, CT, RANGED, VALIDATE, false, DUAL>(base, lane, nrows, rows, row_ptr, col, wt, colour, key, y,
                                                            hub_threshold, lo, hi, n_targets, bad, nullptr, 0u, key2, y2,
                                                            hub_store != 0);
  if (VALIDATE && bad) atomicOr(err, kErrCol);
}

// The same rows through the hot-id table: one persistent CTA of 1024 threads per SM holds the table (128 KB of shared memory);
// its warps draw row groups from a ticket counter.
constexpr int kTagThreads = 1024;
constexpr int kTagRun = 1;  // row groups per ticket (measured 1 / 2 / 4 / 16: 19.6 / 20.4 / 22.0 / 26.7 ms on the headline graph)
template <bool WEIGHTED, bool VALIDATE>
__global__ void __launch_bounds__(kTagThreads, 1)
spmv_rows32_tag_kernel(int64_t nrows, const int* __restrict__ rows, const int64_t* __restrict__ row_ptr,
                       const int* __restrict__ col, const u32* __restrict__ wt, const unsigned short* __restrict__ colour,
                       u64 key, u64* __restrict__ y, int64_t hub_threshold, int64_t n_targets, u32* __restrict__ err,
                       const u32* __restrict__ tagtab, u32 idmask, u64* __restrict__ ticket, int run) {
  extern __shared__ u32 s_tag[];
  for (u32 t = threadIdx.x; t < kTagSlots; t += kTagThreads) s_tag[t] = tagtab[t];
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int64_t ngroups = (nrows + 31) >> 5;
  bool bad = false;
  while (true) {
    u64 g0 = 0;
    if (lane == 0) g0 = atomicAdd(ticket, (u64)run);
    g0 = __shfl_sync(0xffffffffu, g0, 0);
    if ((int64_t)g0 >= ngroups) break;
    const int64_t g1 = (int64_t)g0 + run < ngroups ? (int64_t)g0 + run : ngroups;
    for (int64_t g = (int64_t)g0; g < g1; ++g)
      rows32_group<WEIGHTED, unsigned short, false, VALIDATE, true>(g << 5, lane, nrows, rows, row_ptr, col, wt, colour, key, y,
                                                                    hub_threshold, 0, 0, n_targets, bad, s_tag, idmask);
  }
  if (VALIDATE && bad) atomicOr(err, kErrCol);
}

// tag32[s] = {tag | colour} of the node that won slot s (the highest degree among the candidates that map to it)
__global__ void tag_finalize_kernel(const u64* __restrict__ tag64, const unsigned short* __restrict__ colour16, u32 idmask,
                                    u32* __restrict__ tag32) {
  const u32 sl = blockIdx.x * blockDim.x + threadIdx.x;
  if (sl >= kTagSlots) return;
  const u64 e = tag64[sl];
  if (e == 0) {
    tag32[sl] = kTagEmpty;
    return;
  }
  const u32 id = (u32)e;
  tag32[sl] = ((tag_mix(id, idmask) >> kTagBits) << 16) | (u32)colour16[id];
}

// Hub rows (degree > hub_threshold) are cut into chunks of kHubChunk entries, one CTA each; partial sums meet in y
// through one no-return 64-bit add per CTA (exact under any order: sums in Z/2^64).

__global__ void hub_collect_kernel(int64_t n, const int64_t* __restrict__ row_ptr, int64_t hub_threshold,
                                   int2* __restrict__ chunks, u64* __restrict__ counter) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t d = row_ptr[i + 1] - row_ptr[i];
  if (d <= hub_threshold) return;
  const int nc = (int)((d + kHubChunk - 1) / kHubChunk);
  const u64 base = atomicAdd(counter, (u64)nc);
  for (int c = 0; c < nc; ++c) chunks[base + c] = make_int2((int)i, c);
}

// the same for the rows of a list (wl_spmv_rows)
__global__ void hub_collect_rows_kernel(int64_t nrows, const int* __restrict__ rows, const int64_t* __restrict__ row_ptr,
                                        int64_t hub_threshold, int2* __restrict__ chunks, u64* __restrict__ counter) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nrows) return;
  const int i = rows[t];
  const int64_t d = row_ptr[i + 1] - row_ptr[i];
  if (d <= hub_threshold) return;
  const int nc = (int)((d + kHubChunk - 1) / kHubChunk);
  const u64 base = atomicAdd(counter, (u64)nc);
  for (int c = 0; c < nc; ++c) chunks[base + c] = make_int2(i, c);
}

// y of every hub row = 0 (its first chunk does it): the hub kernel may then run next to the row kernel
__global__ void hub_zero_kernel(int64_t nchunks, const int2* __restrict__ chunks, u64* __restrict__ y) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nchunks && chunks[t].y == 0) y[chunks[t].x] = 0;
}

// active == NULL: every hub row; else only rows whose block is still splittable (stamp[colour[row]] == live_stamp)
template <bool WEIGHTED, typename CT, bool RANGED, bool VALIDATE>
__global__ void __launch_bounds__(kHubThreads)
spmv_hub_kernel(const int2* __restrict__ chunks, const int64_t* __restrict__ row_ptr, const int* __restrict__ col,
                const u32* __restrict__ wt, const CT* __restrict__ colour, u64 key, u64* __restrict__ y,
                const int* __restrict__ colour32, const int* __restrict__ stamp, int live_stamp, int lo, int hi,
                int64_t n_targets, u32* __restrict__ err) {
  const int2 ch = chunks[blockIdx.x];
  const int64_t row = ch.x;
  const bool inactive = stamp && stamp[colour32[row]] != live_stamp;
  if (inactive && !VALIDATE) return;
  const int64_t a = row_ptr[row] + (int64_t)ch.y * kHubChunk;
  int64_t b = a + kHubChunk;
  const int64_t rend = row_ptr[row + 1];
  if (b > rend) b = rend;
  u64 acc = 0;
  bool bad = false;
  if (VALIDATE && inactive) {  // a pruned hub row: its columns are only range-checked
    for (int64_t p = a + threadIdx.x; p < b; p += kHubThreads) checked_col<true>(ld_stream_i32(col + p), n_targets, bad);
    if (bad) atomicOr(err, kErrCol);
    return;
  }
#pragma unroll 4
  for (int64_t p = a + threadIdx.x; p < b; p += kHubThreads) {
    u64 v = weight_of(key, colour_id<RANGED>(colour, checked_col<VALIDATE>(ld_stream_i32(col + p), n_targets, bad), lo, hi));
    if (WEIGHTED) v *= (u64)ld_stream_u32(wt + p);
    acc += v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  __shared__ u64 s[kHubThreads / 32];
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    u64 t = 0;
#pragma unroll
    for (int w = 0; w < kHubThreads / 32; ++w) t += s[w];
    if (t) red_add_u64(y + row, t);
  }
}

// ---------------------------------------------------------------------------------------------------------------------
// S1+S2, edge-balanced and register-only: the kernel of the rounds in which (nearly) every row is active.
// The edge array is cut into super-chunks of kEbSuper consecutive entries, one warp each, whatever the degree
// distribution (empty rows cost nothing, a hub row is simply many chunks).  Per sub-chunk of 256 entries lane l owns the
// entries 32 t + l: coalesced streaming column loads, kEbU independent colour gathers in flight per lane (adjacent lanes
// gather for adjacent sorted columns and share sectors), weights inline.  A sub-chunk without a row end just accumulates
// per lane.  Otherwise warp scans give F(q) = sum of the first q products of the sub-chunk and the lanes take one ROW END
// each (row_ptr read coalesced): the row's sum is F(end) - F(previous end), exact in Z/2^64.  A row that lies
// inside the super-chunk is written with a plain store; the (at most two) rows cut by the super-chunk's borders add their
// pieces with no-return 64-bit adds (exact under any order), eb_setup_kernel having zeroed them first.
// VALIDATE folds the column range check of S0 into the first pass that reads the columns (bad ids are clamped).
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kEbU = 8;
constexpr int kEbSub = 32 * kEbU;
constexpr int kEbSubs = 8;
constexpr int kEbSuper = kEbSub * kEbSubs;

// chunk_row[c] = the row that contains entry e_anchor + c * kEbSuper (row 0 for c == 0); a row cut by that border is
// zeroed in y.  e_anchor <= row_ptr[0] is the origin of the chunk grid.
__global__ void eb_setup_kernel(int64_t n, const int64_t* __restrict__ row_ptr, int64_t e_anchor, int64_t nchunks,
                                int* __restrict__ chunk_row, u64* __restrict__ y) {
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= nchunks) return;
  if (c == 0) {
    chunk_row[0] = 0;
    return;
  }
  const int64_t B = e_anchor + c * kEbSuper;  // row_ptr[0] < B < row_ptr[n]
  int64_t lo = 0, hi = n - 1;                 // first row whose end lies beyond B
  while (lo < hi) {
    const int64_t mid = (lo + hi) >> 1;
    if (row_ptr[mid + 1] > B) hi = mid;
    else lo = mid + 1;
  }
  chunk_row[c] = (int)lo;
  if (row_ptr[lo] < B) y[lo] = 0;
}

template <bool WEIGHTED, typename CT, bool RANGED, bool VALIDATE>
__global__ void __launch_bounds__(256)
spmv_eb_kernel(int64_t n, const int64_t* __restrict__ row_ptr, const int* __restrict__ col, const u32* __restrict__ wt,
               const CT* __restrict__ colour, u64 key, u64* __restrict__ y, const int* __restrict__ chunk_row,
               int64_t e_anchor, int64_t e_first, int64_t e_last, int lo, int hi, int64_t n_targets,
               u32* __restrict__ err) {
  constexpr unsigned kFull = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int64_t c = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t E0 = e_anchor + c * kEbSuper;
  if (E0 >= e_last) return;
  const int64_t E1 = E0 + kEbSuper < e_last ? E0 + kEbSuper : e_last;
  int64_t r_open = chunk_row[c];  // the row that is open at the current position
  const int64_t r_first = r_open;
  const bool first_cut = row_ptr[r_open] < E0;  // it started in an earlier super-chunk
  u64 carry = 0;     // products of the open row seen so far in this super-chunk: carry + sum over lanes of lane_acc
  u64 lane_acc = 0;
  bool bad = false;
  for (int64_t Es = E0; Es < E1; Es += kEbSub) {
    const int64_t sub_end = Es + kEbSub < E1 ? Es + kEbSub : E1;
    // entry Es + 32 t + lane: adjacent lanes read adjacent (sorted) columns, so their gathers share sectors
    int ci[kEbU];
    if (Es >= e_first && Es + kEbSub <= sub_end) {
#pragma unroll
      for (int t = 0; t < kEbU; ++t) ci[t] = ld_stream_i32(col + Es + 32 * t + lane);
    } else {
#pragma unroll
      for (int t = 0; t < kEbU; ++t) {
        const int64_t e = Es + 32 * t + lane;
        ci[t] = (e >= e_first && e < sub_end) ? ld_stream_i32(col + e) : -1;
      }
    }
    if (VALIDATE) {
#pragma unroll
      for (int t = 0; t < kEbU; ++t)
        if (ci[t] != -1 && (unsigned)ci[t] >= (unsigned)n_targets) bad = true, ci[t] = 0;
    }
    u64 v[kEbU];
#pragma unroll
    for (int t = 0; t < kEbU; ++t) v[t] = ci[t] != -1 ? colour_id<RANGED>(colour, ci[t], lo, hi) : 0ull;
#pragma unroll
    for (int t = 0; t < kEbU; ++t) {
      v[t] = ci[t] != -1 ? weight_of(key, v[t]) : 0ull;
      if (WEIGHTED) v[t] *= ci[t] != -1 ? (u64)ld_stream_u32(wt + Es + 32 * t + lane) : 0ull;
    }
    // row ends inside the sub-chunk, one per lane (row_ptr is non-decreasing: the lanes that have one form a prefix)
    int64_t r = r_open + lane;
    int64_t endpos = r < n ? row_ptr[r + 1] : (int64_t)0x7fffffffffffffffll;
    unsigned em = __ballot_sync(kFull, endpos <= sub_end);
    if (em == 0) {  // the whole sub-chunk lies inside the open row
#pragma unroll
      for (int t = 0; t < kEbU; ++t) lane_acc += v[t];
      continue;
    }
    // S[t] of lane l = sum of the products at positions 0 .. 32 t + l of the sub-chunk
    u64 T = 0;
#pragma unroll
    for (int t = 0; t < kEbU; ++t) {
      u64 inc = v[t];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const u64 x = __shfl_up_sync(kFull, inc, o);
        if (lane >= o) inc += x;
      }
      v[t] = T + inc;
      T += __shfl_sync(kFull, inc, 31);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lane_acc += __shfl_xor_sync(kFull, lane_acc, o);
    carry += lane_acc;
    lane_acc = 0;
    u64 Fprev = 0;
    bool first_trip = true;
    while (true) {  // 32 row ends per trip
      const bool is_end = endpos <= sub_end;
      const int cnt = __popc(em);
      const int qm = is_end ? (int)(endpos - Es) - 1 : -1;  // F(q) = S at position q - 1; F(0) = 0
      const int src = qm & 31, tt = qm >> 5;
      u64 Fq = 0;
#pragma unroll
      for (int t = 0; t < kEbU; ++t) {
        const u64 g = __shfl_sync(kFull, v[t], src);
        if (tt == t) Fq = g;
      }
      u64 Fp = __shfl_up_sync(kFull, Fq, 1);
      if (lane == 0) Fp = Fprev;
      u64 sum = Fq - Fp;
      if (lane == 0 && first_trip) sum += carry;
      if (is_end) {
        if (first_cut && r == r_first) {
          if (sum) red_add_u64(y + r, sum);
        } else {
          y[r] = sum;
        }
      }
      Fprev = __shfl_sync(kFull, Fq, cnt - 1);
      first_trip = false;
      r_open += cnt;
      if (cnt < 32) break;
      r = r_open + lane;
      endpos = r < n ? row_ptr[r + 1] : (int64_t)0x7fffffffffffffffll;
      em = __ballot_sync(kFull, endpos <= sub_end);
      if (em == 0) break;
    }
    carry = T - Fprev;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) lane_acc += __shfl_xor_sync(kFull, lane_acc, o);
  carry += lane_acc;
  if (lane == 0 && carry != 0 && r_open < n) red_add_u64(y + r_open, carry);  // continues in the next super-chunk
  if (VALIDATE && bad) atomicOr(err, kErrCol);
}

// narrow copy of caller-supplied colour ids (wl_spmv_round with WL_FLAG_NARROW_COLORS; wl_refine keeps its own mirror)
__global__ void narrow_kernel(int64_t n, const int* __restrict__ colour, unsigned short* __restrict__ colour16) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) colour16[i] = (unsigned short)colour[i];
}

// Active-set pruning (SURVEY.md §8(d) option 6): a node whose block is a singleton can never split again and keeps its
// id, so its row needs neither y nor a relabel.  next = nodes of `nodes` (NULL: all) whose block still has >= 2 members
// after round `round`; counters[0] += |next|, counters[1] += sum of their out-degrees.  Rows without out-edges are
// dropped as soon as their block's representative has none either (their y is 0 in every round).
// final_col != NULL: blocks whose neighbourhood is final are dropped as well (see below; k_prev = colour count before the
// round that just ended).
// check_col != NULL (the column range check of S0 is still pending): the rows dropped here are never read
// by a row kernel, so their columns are range-checked now, one warp per row (hub rows are left to spmv_hub_kernel).
constexpr int kFinalRow = 32;  // rows up to this length are tested for finality
__global__ void __launch_bounds__(256)
compact_active_kernel(int64_t count, const int* __restrict__ nodes, const int* __restrict__ colour,
                      const int* __restrict__ stamp, const int* __restrict__ rep, int round,
                      const int64_t* __restrict__ row_ptr, int64_t hub_threshold, int* __restrict__ next,
                      u64* __restrict__ counters, u64* __restrict__ hub_counter, const int* __restrict__ check_col,
                      int64_t n_targets, u32* __restrict__ err, const int* __restrict__ final_col, int k_prev,
                      const u64* __restrict__ y2) {
  int64_t t = (int64_t)blockIdx.x * 256 + threadIdx.x;
  bool keep = false;
  int i = 0;
  u64 deg = 0;
  if (check_col) {
    int64_t a = 0, b = 0;
    bool dropped = false;
    if (t < count) {
      const int node = nodes ? nodes[t] : (int)t;
      a = row_ptr[node];
      b = row_ptr[node + 1];
      dropped = stamp[colour[node]] != round && b > a && b - a <= hub_threshold;
    }
    unsigned todo = __ballot_sync(0xffffffffu, dropped);
    bool bad = false;
    while (todo) {
      const int src = __ffs(todo) - 1;
      todo &= todo - 1;
      const int64_t ra = __shfl_sync(0xffffffffu, a, src), rb = __shfl_sync(0xffffffffu, b, src);
      for (int64_t p = ra + (threadIdx.x & 31); p < rb; p += 32) checked_col<true>(ld_stream_i32(check_col + p), n_targets, bad);
    }
    if (bad) atomicOr(err, kErrCol);
  }
  if (t < count) {
    i = nodes ? nodes[t] : (int)t;
    const int c = colour[i];
    keep = stamp[c] == round;
    if (keep) {
      deg = (u64)(row_ptr[i + 1] - row_ptr[i]);
      if ((int64_t)deg > hub_threshold) atomicAdd(hub_counter, 1ull);  // rare: hubs still in a splittable block
      if (deg == 0) {
        // y_i = 0 in every round.  If the block's representative has no out-edge either, every member with an
        // out-edge is compared against y[rep] = 0 and leaves on its own; the edgeless members never need another look.
        const int r = rep[c];
        keep = row_ptr[r + 1] != row_ptr[r];
      } else if (final_col && deg <= kFinalRow) {
        // Final block (R5): every out-neighbour's colour existed before this round (id < k_prev) and its block was
        // already out of the loop then (singleton or dropped: not seen with two members in the previous round).  This
        // round's y was computed from exactly those colours, so the nodes that share this block have the same
        // neighbour colours, all of which never change again: the block can never split.  "Share this block" is decided
        // by TWO independent sums: the round's y (the relabel key) and y2, the same sum under a second key (DUAL rows of
        // the row kernel); a node whose y2 differs from its representative's stays active, so a wrong merge can only
        // become permanent if the same pair collides under both keys.
        const int64_t a = row_ptr[i];
        bool all_final = true;
        for (int64_t p = a; p < a + (int64_t)deg; ++p) {
          const int cj = colour[final_col[p]];
          if (cj >= k_prev || stamp[cj] >= round - 1) {
            all_final = false;
            break;
          }
        }
        keep = !all_final || y2[i] != y2[rep[c]];
      }
    }
  }
  int total;
  const int rank = block_rank<256>(keep, &total);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) deg += __shfl_xor_sync(0xffffffffu, deg, o);
  __shared__ u64 s_deg[8];
  __shared__ u64 s_base;
  if ((threadIdx.x & 31) == 0) s_deg[threadIdx.x >> 5] = deg;
  __syncthreads();
  if (threadIdx.x == 0 && total > 0) {
    u64 d = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) d += s_deg[w];
    s_base = atomicAdd(counters, (u64)total);
    atomicAdd(counters + 1, d);
  }
  __syncthreads();
  if (keep) next[s_base + rank] = i;
}

// ---------------------------------------------------------------------------------------------------------------------
// S3+S4: relabel (colour_i, y_i) -> dense id (Alg. 1 line 6, L122; Q6: exact 96-bit pairs, never a hash of them).
// A block keeps its id for the sub-block that agrees with its representative rep[c]; every other distinct pair
// (c, y) claims a slot of an exact-key hash table with one 128-bit CAS and gets a fresh id k, k+1, ...  (block-
// aggregated counter, S4).  One kernel per round:
//   phase 1  every thread compares with its representative and, if different, finds or claims the slot of its key
//            (no thread waits on another one here); a claimed slot carries the id kPending;
//   phase 2  the winners of the CTA take consecutive ids, publish them in the slot, become the representative of the
//            new colour and record the slot in slot_of[id] (relabel_finish_kernel re-empties exactly those slots);
//   phase 3  a node that found its key claimed by somebody else reads the id from the slot; if it is still pending it
//            polls.  The winner publishes without waiting on anything but its own CTA's phase 1, so the poll ends.
// stamp[c] == round  <=>  block c has at least two nodes after this round (no atomics: plain idempotent stores).
// colour16 (optional) mirrors the ids as 16 bits while k <= 65536 (narrow gathers in the SpMV).  nodes == NULL: all nodes.
// changed (optional): list of the nodes whose id changed.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kRelabelThreads = 256;
constexpr u32 kPending = 0xffffffffu;

__device__ __forceinline__ u32 ld_slot_id(const Slot* p) {
  u32 v;
  asm volatile("ld.global.relaxed.gpu.u32 %0, [%1];" : "=r"(v) : "l"(reinterpret_cast<const u32*>(p) + 3) : "memory");
  return v;
}
__device__ __forceinline__ void st_slot_id(Slot* p, u32 id) {
  asm volatile("st.global.relaxed.gpu.u32 [%0], %1;" ::"l"(reinterpret_cast<u32*>(p) + 3), "r"(id) : "memory");
}

__global__ void __launch_bounds__(kRelabelThreads)
relabel_kernel(int64_t count, const int* __restrict__ nodes, int* __restrict__ colour,
               unsigned short* __restrict__ colour16, const u64* __restrict__ y, int* __restrict__ rep,
               int* __restrict__ stamp, int round, Slot* __restrict__ table, u32 table_mask,
               u32* __restrict__ slot_of, const u64* __restrict__ k_ptr, u64* __restrict__ new_counter,
               int* __restrict__ changed, u64* __restrict__ n_changed, u64 ymask) {
  const int k_old = (int)*k_ptr;  // device-resident colour count: rounds can be queued without a host round trip
  int64_t t = (int64_t)blockIdx.x * kRelabelThreads + threadIdx.x;
  bool win = false, lose = false;
  u32 slot = 0, id = kPending;
  int i = -1;
  if (t < count) {
    i = nodes ? nodes[t] : (int)t;
    const int c = colour[i];
    const int r = rep[c];
    const u64 yi = y[i] & ymask;  // ymask = the ring mask (all ones in the product; all ones for the densify step)
    const u64 yr = y[r] & ymask;
    if (yi == yr) {
      if (i != r && stamp[c] != round) stamp[c] = round;
    } else {
      const Slot mine = {yi, (u64)(u32)c | ((u64)kPending << 32)};
      const Slot empty = {kEmpty, kEmpty};
      slot = (u32)slot_hash((u32)c, yi) & table_mask;
      while (true) {
        Slot v = load_slot(table + slot);
        if (v.y == kEmpty || v.cx == kEmpty) {  // empty, or a torn view of a slot being claimed: decide with the CAS
          v = cas128(table + slot, empty, mine);
          if (v.y == kEmpty && v.cx == kEmpty) {
            win = true;
            break;
          }
        }
        if (v.y == yi && (u32)v.cx == (u32)c) {
          lose = true;
          id = (u32)(v.cx >> 32);
          break;
        }
        slot = (slot + 1) & table_mask;
      }
    }
  }
  int total;
  const int rank = block_rank<kRelabelThreads>(win, &total);
  __shared__ u64 s_base;
  if (threadIdx.x == 0 && total > 0) s_base = atomicAdd(new_counter, (u64)total);
  __syncthreads();
  if (win) {
    id = (u32)(k_old + (int)s_base + rank);
    st_slot_id(table + slot, id);
    rep[id] = i;
    slot_of[id] = slot;
  } else if (lose) {
    while (id == kPending) id = ld_slot_id(table + slot);
    if (stamp[id] != round) stamp[id] = round;  // (a blind store measured no faster: 4.03 against 3.99 ms on the headline round)
  }
  if (win || lose) {
    colour[i] = (int)id;
    if (colour16) colour16[i] = (unsigned short)id;
  }
  if (changed) {  // the nodes that got a new id, for the worklist regime (wl_deep.cuh); one atomic per warp
    const bool ch = win || lose;
    const unsigned bal = __ballot_sync(0xffffffffu, ch);
    if (bal) {
      const int lane = threadIdx.x & 31, leader = __ffs(bal) - 1;
      u64 base = 0;
      if (lane == leader) base = atomicAdd(n_changed, (u64)__popc(bal));
      base = __shfl_sync(0xffffffffu, base, leader);
      if (ch) changed[base + __popc(bal & ((1u << lane) - 1))] = i;
    }
  }
}

// S0 + round 1 in one pass for a uniform start with unit weights (R2): z_i = outdeg(i) * w(0), so the round only reads
// row_ptr.  Per node: offsets validated (as validate_rows_kernel), hub rows cut into chunks (as hub_collect_kernel), the
// key (0, z_i) relabelled exactly as relabel_kernel does (node 0 represents colour 0), and the node appended to the active
// list unless it has no out-edge (the class of edgeless nodes is represented by an edgeless node: it never needs another
// look, see compact_active_kernel).  z is not stored: round 2 recomputes it for every listed row before reading it.
// The list is a superset of what compact_active_kernel would keep (it keeps the few nodes whose degree is unique);
// counters[0] = listed rows, counters[1] = their out-degree sum (= m), *hub_rows = listed rows longer than hub_threshold.
// Degree classes repeat: 63 M listed rows of the headline graph share 3 855 keys, so every CTA keeps the ids it has already
// seen in shared memory (s_id[d] = id of the class of out-degree d, bit 30 = "stamp[id] is known to be set"); only the first
// sight of a degree in a CTA goes to the global table.  One CTA per super-tile of kR1Sub * 256 nodes (the loop is grid-stride, but
// a grid of all super-tiles keeps the active list closest to node order, which the row kernel of round 2 likes best).
constexpr int kR1Cache = 4096;       // out-degrees below this are cached per CTA (16 KB)
constexpr int kR1Sub = 8;            // sub-tiles of kRelabelThreads nodes per list reservation
constexpr int kR1Stamped = 1 << 30;  // round-1 ids stay far below 2^30 (at most sqrt(2m) + 1 distinct degrees)
__global__ void __launch_bounds__(kRelabelThreads)
round1_uniform_kernel(int64_t n, const int64_t* __restrict__ row_ptr, int64_t expect_first, int64_t expect_last, u64 w0,
                      int* __restrict__ colour, unsigned short* __restrict__ colour16, int* __restrict__ rep,
                      int* __restrict__ stamp, Slot* __restrict__ table, u32 table_mask, u32* __restrict__ slot_of,
                      u64* __restrict__ new_counter, int64_t hub_threshold, int2* __restrict__ chunks, int64_t hub_cap,
                      u64* __restrict__ hub_counter, int* __restrict__ active, u64* __restrict__ counters,
                      u64* __restrict__ hub_rows, u32* __restrict__ err, u64 ymask, u64* __restrict__ tag64,
                      int64_t tag_threshold, u32 idmask) {
  constexpr int round = 1, k_old = 1;
  constexpr int kWarps = kRelabelThreads / 32;
  __shared__ int s_id[kR1Cache];
  __shared__ u64 s_base, s_list;
  __shared__ int s_stamp0;
  __shared__ int s_cnt[kR1Sub * kWarps];
  for (int j = threadIdx.x; j < kR1Cache; j += kRelabelThreads) s_id[j] = -1;
  if (threadIdx.x == 0) s_stamp0 = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // the representative of colour 0 is node 0
  int64_t d0 = row_ptr[1] - row_ptr[0];
  if (d0 < 0 || (u64)d0 >= (1ull << 32)) d0 = 0;
  const u64 y0 = ((u64)d0 * w0) & ymask;
  constexpr int64_t kSuper = (int64_t)kR1Sub * kRelabelThreads;
  const int64_t supers = (n + kSuper - 1) / kSuper;
  for (int64_t sup = blockIdx.x; sup < supers; sup += gridDim.x) {
    unsigned kb[kR1Sub];  // per sub-tile: which lanes of this warp list their node
#pragma unroll
    for (int q = 0; q < kR1Sub; ++q) {
      const int64_t t = sup * kSuper + (int64_t)q * kRelabelThreads + threadIdx.x;
      const bool valid = t < n;
      const int i = (int)t;
      int64_t d = 0;
      if (valid) {
        const int64_t a = row_ptr[t], b = row_ptr[t + 1];
        u32 e = 0;
        if (t == 0 && a != expect_first) e |= kErrRowPtr;
        if (t == n - 1 && b != expect_last) e |= kErrRowPtr;
        if (a > b || a < expect_first || b > expect_last) e |= kErrRowPtr;
        d = e ? 0 : b - a;
        if ((u64)d >= (1ull << 32)) e |= kErrRowSum, d = 0;
        if (d > hub_threshold) {
          const int nc = (int)((d + kHubChunk - 1) / kHubChunk);
          const u64 base = atomicAdd(hub_counter, (u64)nc);
          if ((int64_t)(base + nc) <= hub_cap) {
            for (int c = 0; c < nc; ++c) chunks[base + c] = make_int2(i, c);
          } else {
            e |= kErrRowPtr;  // only overlapping (malformed) rows can exceed the capacity derived from m
          }
          atomicAdd(hub_rows, 1ull);
        }
        if (e) atomicOr(err, e);
        // hot-id table of the coming rounds: the highest-degree node wins its slot (out-degree stands in for the number of
        // gathers a node receives; any choice is correct, a miss falls through to the global gather)
        if (tag64 && d >= tag_threshold) atomicMax(tag64 + (tag_mix((u32)i, idmask) & (kTagSlots - 1)), ((u64)d << 32) | (u64)(u32)i);
      }
      bool win = false, lose = false;
      u32 slot = 0, id = 0;
      if (valid) {
        const u64 yi = ((u64)d * w0) & ymask;
        if (yi == y0) {
          if (i != 0 && !s_stamp0) {
            if (stamp[0] != round) stamp[0] = round;
            s_stamp0 = 1;
          }
        } else {
          const int e = d < kR1Cache ? s_id[d] : -1;
          if (e >= 0) {  // this CTA has met the class before: same out-degree, same key, same id
            id = (u32)(e & (kR1Stamped - 1));
            if (!(e & kR1Stamped)) {
              if (stamp[id] != round) stamp[id] = round;
              s_id[d] = e | kR1Stamped;
            }
          } else {
            id = kPending;
            const Slot mine = {yi, (u64)kPending << 32};
            const Slot empty = {kEmpty, kEmpty};
            slot = (u32)slot_hash(0u, yi) & table_mask;
            while (true) {
              Slot v = load_slot(table + slot);
              if (v.y == kEmpty || v.cx == kEmpty) {
                v = cas128(table + slot, empty, mine);
                if (v.y == kEmpty && v.cx == kEmpty) {
                  win = true;
                  break;
                }
              }
              if (v.y == yi && (u32)v.cx == 0u) {
                lose = true;
                id = (u32)(v.cx >> 32);
                break;
              }
              slot = (slot + 1) & table_mask;
            }
          }
        }
      }
      if (__syncthreads_or(win)) {  // rare after the first tiles of a CTA: some thread claimed a new class
        int total;
        const int rank = block_rank<kRelabelThreads>(win, &total);
        if (threadIdx.x == 0) s_base = atomicAdd(new_counter, (u64)total);
        __syncthreads();
        if (win) {
          id = (u32)(k_old + (int)s_base + rank);
          st_slot_id(table + slot, id);
          rep[id] = i;
          slot_of[id] = slot;
          if (d < kR1Cache && id < (u32)kR1Stamped) s_id[d] = (int)id;
        }
      }
      if (lose) {
        while (id == kPending) id = ld_slot_id(table + slot);
        if (stamp[id] != round) stamp[id] = round;
        if (d < kR1Cache && id < (u32)kR1Stamped) s_id[d] = (int)id | kR1Stamped;
      }
      if (valid) {
        colour[i] = (int)id;
        colour16[i] = (unsigned short)id;
      }
      // active list: every node with an out-edge
      kb[q] = __ballot_sync(0xffffffffu, valid && d > 0);
      if (lane == 0) s_cnt[q * kWarps + wid] = __popc(kb[q]);
    }
    // one list reservation per super-tile (the same-address atomic is what bounds a tile-per-atomic version); node order kept
    __syncthreads();
    if (wid == 0) {
      static_assert(kR1Sub * kWarps == 64, "one warp scans two counts per lane");
      const int c0 = s_cnt[2 * lane], c1 = s_cnt[2 * lane + 1];
      int x = c0 + c1;
      const int mine = x;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int u = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += u;
      }
      s_cnt[2 * lane] = x - mine;
      s_cnt[2 * lane + 1] = x - mine + c0;
      if (lane == 31 && x > 0) s_list = atomicAdd(counters, (u64)x);
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kR1Sub; ++q)
      if ((kb[q] >> lane) & 1u)
        active[s_list + s_cnt[q * kWarps + wid] + __popc(kb[q] & ((1u << lane) - 1))] =
            (int)(sup * kSuper + (int64_t)q * kRelabelThreads + threadIdx.x);
    __syncthreads();  // s_cnt / s_list are rewritten by the next super-tile
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) counters[1] = (u64)(expect_last - expect_first);
}

// End of a round (S4): if `clean`, the slots claimed by this round's new ids are emptied again (the table is empty
// between rounds; with clean == 0 the host does it once it knows how many ids there were: relabel_clean_kernel or a
// memset), then the last CTA to finish does k += new ids, logs k for the host and re-arms the counter.
// scal layout: see wl_device.cuh.
__global__ void __launch_bounds__(256)
relabel_finish_kernel(Slot* __restrict__ table, const u32* __restrict__ slot_of, u64* __restrict__ scal,
                      u64* __restrict__ log, int log_slot, int clean) {
  const u64 k_old = scal[kScalK], n_new = scal[kScalNew];
  if (clean) {
    const u64 stride = (u64)gridDim.x * blockDim.x;
    for (u64 j = (u64)blockIdx.x * blockDim.x + threadIdx.x; j < n_new; j += stride)
      store_slot(table + slot_of[k_old + j], kEmpty, kEmpty);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    const u64 ticket = atomicAdd(scal + kScalTicket, 1ull);
    if (ticket == (u64)gridDim.x - 1) {  // every other CTA has read k_old / n_new before taking its ticket
      scal[kScalK] = k_old + n_new;
      scal[kScalNew] = 0;
      scal[kScalTicket] = 0;
      if (log) log[log_slot] = k_old + n_new;
    }
  }
}

// empties the slots of the ids [first_id, first_id + count)
__global__ void relabel_clean_kernel(Slot* __restrict__ table, const u32* __restrict__ slot_of, int64_t first_id,
                                     int64_t count) {
  int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j < count) store_slot(table + slot_of[first_id + j], kEmpty, kEmpty);
}

// rep[c] = some node of colour c (any one: benign race)
__global__ void set_rep_kernel(int64_t n, const int* __restrict__ colour, int* __restrict__ rep) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) rep[colour[i]] = (int)i;
}

// densify helper: y_i = init label (must be non-negative), colour_i = 0
__global__ void init_labels_kernel(int64_t n, const int* __restrict__ init, int* __restrict__ colour,
                                   unsigned short* __restrict__ colour16, u64* __restrict__ y,
                                   u32* __restrict__ err) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int v = init ? init[i] : 0;
  if (v < 0) atomicOr(err, kErrInit);
  colour[i] = 0;
  colour16[i] = 0;
  y[i] = (u64)(u32)v;
}

// ---------------------------------------------------------------------------------------------------------------------
// S6: canonical first-occurrence ids.  first[c] = min node of colour c; blocks are ranked by their first node.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanChunk = kScanThreads * kScanItems;

__global__ void fill_i32_kernel(int64_t n, int* __restrict__ a, int v) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) a[i] = v;
}

// four nodes per thread (strided by the CTA width): the colour loads, then the four dependent first[] loads, are in flight together
constexpr int kFirstItems = 4;
__global__ void __launch_bounds__(256)
first_node_kernel(int64_t n, const int* __restrict__ colour, int* __restrict__ first) {
  const int64_t base = (int64_t)blockIdx.x * (256 * kFirstItems) + threadIdx.x;
  int c[kFirstItems], f[kFirstItems];
#pragma unroll
  for (int k = 0; k < kFirstItems; ++k) c[k] = base + k * 256 < n ? colour[base + k * 256] : -1;
#pragma unroll
  for (int k = 0; k < kFirstItems; ++k) f[k] = c[k] >= 0 ? first[c[k]] : 0;
#pragma unroll
  for (int k = 0; k < kFirstItems; ++k)
    if (c[k] >= 0 && f[k] > (int)(base + k * 256)) atomicMin(first + c[k], (int)(base + k * 256));
}

// flags: one bit per node, "node i is the first node of its block", kCanonWords words per chunk of kScanChunk nodes (word
// 8 k + w of a chunk = nodes 32 (8 k + w) .. + 31 of it).  Written once here; the rank and apply passes read the bits
// instead of gathering first[colour[i]] again.
constexpr int kCanonWords = kScanChunk / 32;
__global__ void __launch_bounds__(kScanThreads)
canon_count_kernel(int64_t n, const int* __restrict__ colour, const int* __restrict__ first, int* __restrict__ bsum,
                   u32* __restrict__ flags) {
  const int64_t base = (int64_t)blockIdx.x * kScanChunk;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int cnt = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    int64_t i = base + threadIdx.x + k * kScanThreads;
    const bool f = i < n && first[colour[i]] == (int)i;
    const unsigned b = __ballot_sync(0xffffffffu, f);
    if (lane == 0) flags[(int64_t)blockIdx.x * kCanonWords + k * (kScanThreads / 32) + wid] = b;
    cnt += f;
  }
  __shared__ int s[kScanThreads / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  if (lane == 0) s[wid] = cnt;
  __syncthreads();
  if (threadIdx.x == 0) {
    int t = 0;
    for (int w = 0; w < kScanThreads / 32; ++w) t += s[w];
    bsum[blockIdx.x] = t;
  }
}

// exclusive scan of nb block sums by one CTA; total -> out_total
__global__ void __launch_bounds__(1024) scan_bsum_kernel(int64_t nb, int* __restrict__ bsum, u64* __restrict__ out_total) {
  __shared__ int s_w[32];
  __shared__ int s_carry;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int64_t base = 0; base < nb; base += 1024) {
    int64_t i = base + threadIdx.x;
    int v = i < nb ? bsum[i] : 0;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += t;
    }
    if (lane == 31) s_w[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int t = s_w[lane];
      int xs = t;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int u = __shfl_up_sync(0xffffffffu, xs, o);
        if (lane >= o) xs += u;
      }
      s_w[lane] = xs - t;  // exclusive warp offsets
    }
    __syncthreads();
    const int carry = s_carry;
    if (i < nb) bsum[i] = carry + s_w[wid] + x - v;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = carry + s_w[wid] + x;
    __syncthreads();
  }
  if (threadIdx.x == 0) *out_total = (u64)s_carry;
}

// the flag words of this CTA's chunk and their exclusive prefix counts (both in shared memory)
__device__ __forceinline__ void canon_chunk_prefix(const u32* __restrict__ flags, u32* s_word, int* s_pref) {
  static_assert(kCanonWords == 64, "two warps scan the flag words of a chunk");
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __shared__ int s_half;
  if (wid < 2) {
    const u32 w = flags[(int64_t)blockIdx.x * kCanonWords + threadIdx.x];
    const int c = __popc(w);
    int x = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += t;
    }
    s_word[threadIdx.x] = w;
    s_pref[threadIdx.x] = x - c;
    if (threadIdx.x == 31) s_half = x;
  }
  __syncthreads();
  if (wid == 1) s_pref[threadIdx.x] += s_half;
  __syncthreads();
}

// cid[c] = rank of block c among the blocks ordered by their first node (the flagged nodes, in node order)
__global__ void __launch_bounds__(kScanThreads)
canon_rank_kernel(int64_t n, const int* __restrict__ colour, const u32* __restrict__ flags,
                  const int* __restrict__ bsum, int* __restrict__ cid) {
  __shared__ u32 s_word[kCanonWords];
  __shared__ int s_pref[kCanonWords];
  canon_chunk_prefix(flags, s_word, s_pref);
  const int64_t base = (int64_t)blockIdx.x * kScanChunk;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int r0 = bsum[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const int wi = k * (kScanThreads / 32) + wid;
    const u32 w = s_word[wi];
    if ((w >> lane) & 1u) {
      const int64_t i = base + threadIdx.x + k * kScanThreads;
      cid[colour[i]] = r0 + s_pref[wi] + __popc(w & ((1u << lane) - 1));
    }
  }
}

// out[i] = canonical id of node i's block: its own rank for a first node (from the flag bits), cid[colour[i]] otherwise
__global__ void __launch_bounds__(kScanThreads)
canon_apply_kernel(int64_t n, const int* __restrict__ colour, const int* __restrict__ cid, const u32* __restrict__ flags,
                   const int* __restrict__ bsum, int* __restrict__ out) {
  __shared__ u32 s_word[kCanonWords];
  __shared__ int s_pref[kCanonWords];
  canon_chunk_prefix(flags, s_word, s_pref);
  const int64_t base = (int64_t)blockIdx.x * kScanChunk;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int r0 = bsum[blockIdx.x];
  int c[kScanItems], v[kScanItems];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {  // colours of the nodes that are not the first of their block (the others need none)
    const int64_t i = base + threadIdx.x + k * kScanThreads;
    const u32 w = s_word[k * (kScanThreads / 32) + wid];
    c[k] = (i < n && !((w >> lane) & 1u)) ? colour[i] : -1;
  }
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) v[k] = c[k] >= 0 ? cid[c[k]] : 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) {
    const int64_t i = base + threadIdx.x + k * kScanThreads;
    if (i >= n) continue;
    const int wi = k * (kScanThreads / 32) + wid;
    const u32 w = s_word[wi];
    out[i] = ((w >> lane) & 1u) ? r0 + s_pref[wi] + __popc(w & ((1u << lane) - 1)) : v[k];
  }
}

}  // namespace wl
