// Batched path: Algorithm 2 (RBSC) over host-resident edge batches, and its step-level pieces.
//
// SURVEY.md §8(a) rows and where they are:
//   B1 stream      upload_batch(): pinned/pageable host -> two device buffers on a copy stream, the next batch is
//                  uploaded while the current one is refined (event-ordered double buffering)
//   B2 inner mask  row-aligned batches (the library's own partition, Q13): V_k is a contiguous node range computed on the
//                  host from the cuts (inner_range()); arbitrary partitions: inner_labels_kernel (wl_inner_labels)
//   B3 local init  implicit: targets outside V_k get the id 2^32 + j inside the SpMV kernels (colour_id<RANGED>)
//   B4 local RSC   refine_core(ranged = true) on the rows of V_k only
//   B5 merge       merge_kernel: global id = running offset + local id; boundary nodes get fresh ids (Eq. 4)
//   B6 quotient    quot_insert_kernel / quot_emit_kernel: representative rows mapped through the block map and merged in
//                  an exact-key hash table (key = (block, target block), value = summed weight), Def. 4 / Eq. 1
//   B7 outer loop  wl_refine_batched(): re-batch the quotient, stop at N_b = 1 or |V| unchanged (L200), compose block maps
//   B8 verify      lives in the test harness (oracle_is_stable on the original graph)
// COO-form (arbitrary) first partitions are not accepted by wl_refine_batched yet (WL_EINVAL); wl_inner_labels covers
// their Def. 5 mask.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <condition_variable>
#include <functional>
#include <map>
#include <mutex>
#include <thread>
#include <vector>

#include "wl_host.h"

namespace wl {

// ---------------------------------------------------------------------------------------------------------------------
// kernels
// ---------------------------------------------------------------------------------------------------------------------

// Def. 5 (L139-L145) by the method of L463: a node is inner to batch k iff all its out-edges carry label k.
__global__ void inner_labels_kernel(int64_t n, const int64_t* __restrict__ row_ptr, const int* __restrict__ edge_batch,
                                    const int* __restrict__ sink_batch, int* __restrict__ label) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t a = row_ptr[i], b = row_ptr[i + 1];
  if (a == b) {
    label[i] = sink_batch[i];
    return;
  }
  const int k = edge_batch[a];
  bool inner = true;
  for (int64_t p = a + 1; p < b; ++p) inner &= (edge_batch[p] == k);
  label[i] = inner ? k : -1;
}

// Eq. 4: blocks of H_k inside V_k enter the global partition with ids base + local id
__global__ void merge_kernel(int64_t n_local, const int* __restrict__ local_colour, int base, int* __restrict__ H) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_local) H[i] = base + local_colour[i];
}

// One helper thread per wl_refine_batched call (WL_FLAG_INHERIT_BATCHES): the local refinement of the rows the quotient pass has
// just emitted synchronises its stream once per round, and while the calling thread sat in it the next emission could not be
// queued.  The helper runs those refinements one after the other (their block ids build on each other); the caller submits a
// piece and waits for it only when the piece's buffers are needed again.
class PieceWorker {
 public:
  explicit PieceWorker(int device) : device_(device) {}
  ~PieceWorker() {
    if (!th_.joinable()) return;
    {
      std::lock_guard<std::mutex> g(mu_);
      stop_ = true;
    }
    cv_.notify_all();
    const auto t0 = std::chrono::steady_clock::now();
    th_.join();
    if (debug_enabled())
      std::fprintf(stderr, "[wl_refine_batched] helper thread joined in %9.3f ms\n",
                   std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count());
  }
  void submit(std::function<int()> f) {  // at most one task is outstanding: wait() first
    if (!th_.joinable()) th_ = std::thread([this] { loop(); });
    {
      std::lock_guard<std::mutex> g(mu_);
      task_ = std::move(f);
      busy_ = true;
    }
    cv_.notify_all();
  }
  int wait() {  // result of the last task (WL_OK when none was submitted)
    std::unique_lock<std::mutex> g(mu_);
    cv_.wait(g, [this] { return !busy_; });
    const int r = result_;
    result_ = WL_OK;
    return r;
  }

 private:
  void loop() {
    cudaSetDevice(device_);
    std::unique_lock<std::mutex> g(mu_);
    while (true) {
      cv_.wait(g, [this] { return stop_ || (busy_ && task_); });
      if (stop_) return;
      std::function<int()> f = std::move(task_);
      task_ = nullptr;
      g.unlock();
      const int r = f();
      g.lock();
      result_ = r;
      busy_ = false;
      cv_.notify_all();
    }
  }
  int device_;
  std::thread th_;
  std::mutex mu_;
  std::condition_variable cv_;
  std::function<int()> task_;
  bool busy_ = false, stop_ = false;
  int result_ = WL_OK;
};

// every stored target of an uploaded slice must be a node id in [0, n)
__global__ void slice_cols_check_kernel(int64_t n, int64_t count, const int* __restrict__ col, u32* __restrict__ err) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  bool bad = false;
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < count; p += stride)
    bad |= (unsigned)col[p] >= (unsigned)n;
  if (bad) atomicOr(err, kErrCol);
}

__global__ void fill_kernel(int64_t n, int* __restrict__ a, int v) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) a[i] = v;
}

__global__ void iota_kernel(int64_t n, int* __restrict__ a) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) a[i] = (int)i;
}

// Eq. 4 for one batch whose local colours have just been made canonical inside the batch (first-occurrence ids): the global
// id is base + local canonical id.  Batches and the boundary nodes between them are taken in node order, so the global ids are
// canonical as well and no pass over all n nodes is needed.  isrep[i] = 1 for the first node of every block (Q17).
__global__ void merge_canon_kernel(int64_t nr, const int* __restrict__ local_colour, const int* __restrict__ first, int base,
                                   int* __restrict__ Hc, unsigned char* __restrict__ isrep) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nr) return;
  Hc[i] += base;
  isrep[i] = first[local_colour[i]] == (int)i;
}

// Alg. 2 lines 11-12: the boundary nodes g0 .. g0 + count - 1 become singleton blocks base, base + 1, ...
__global__ void gap_singletons_kernel(int64_t g0, int64_t count, int base, int* __restrict__ Hc,
                                      unsigned char* __restrict__ isrep) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  Hc[g0 + t] = base + (int)t;
  isrep[g0 + t] = 1;
}

// one block made of the nodes [0, count): id `id`, representative = the first one (a piece of edgeless nodes)
__global__ void one_block_kernel(int64_t count, int id, int* __restrict__ Hc, unsigned char* __restrict__ isrep) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  Hc[t] = id;
  isrep[t] = t == 0;
}

// counts[q] = number of representatives i with queries[q - 1] <= i < queries[q] (queries increasing, queries[-1] = 0): the host
// prefix-sums them into "blocks whose first node lies before queries[q]"
__global__ void count_reps_kernel(int64_t n, const unsigned char* __restrict__ isrep, const int64_t* __restrict__ queries, int nq,
                                  u64* __restrict__ counts) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int q = -1;
  if (i < n && isrep[i]) {
    int lo = 0, hi = nq;  // first q with queries[q] > i (nq: beyond the last query)
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (queries[mid] > i) hi = mid;
      else lo = mid + 1;
    }
    q = lo;
  }
  const unsigned peers = __match_any_sync(0xffffffffu, q);
  if (q >= 0 && (int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(counts + q, (u64)__popc(peers));
}

// *out = max(*out, max of a[0 .. n)) (the longest row of the quotient being emitted: its row lengths are the block counters)
__global__ void max_i32_kernel(int64_t n, const int* __restrict__ a, int* __restrict__ out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int v = i < n ? a[i] : 0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0 && v > 0) atomicMax(out, v);
}

// res[1] = the largest row offset <= limit (rp increasing, rp[0] <= limit): the greedy cut (Q13); res[0] = the first index that has it
__global__ void cut_search_kernel(const int64_t* __restrict__ rp, int64_t n, int64_t limit, int64_t* __restrict__ res) {
  if (blockIdx.x || threadIdx.x) return;
  int64_t lo = 0, hi = n;  // invariant: rp[lo] <= limit
  while (lo < hi) {
    const int64_t mid = (lo + hi + 1) >> 1;
    if (rp[mid] <= limit) lo = mid;
    else hi = mid - 1;
  }
  // rows without entries that sit exactly on the cut belong to the NEXT batch (inner_range: its first node is the first one
  // whose row starts at or after the cut): back to the first index with this offset
  const int64_t edge = rp[lo];
  int64_t a = 0, b = lo;  // first index in [0, lo] with rp[index] >= edge
  while (a < b) {
    const int64_t mid = (a + b) >> 1;
    if (rp[mid] >= edge) b = mid;
    else a = mid + 1;
  }
  res[0] = a;
  res[1] = edge;
}

// the window of per-block counters moves on by `len` blocks: the counter of the block whose row is still open (index len)
// becomes index 0, everything else is zero again
__global__ void window_carry_kernel(int* __restrict__ cnt, int64_t len, int* __restrict__ carry, int phase) {
  if (blockIdx.x || threadIdx.x) return;
  if (phase == 0) *carry = cnt[len];
  else cnt[0] = *carry;
}

// initial classes (wl_options.batched_init_colors, reading Q18): the class of a block is the class of its nodes (every local
// colouring refines its start, so all writers of one entry store the same value)
__global__ void class_of_blocks_kernel(int64_t n, const int* __restrict__ block_of, const int* __restrict__ cls, int* __restrict__ cls_next) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) cls_next[block_of[i]] = cls[i];
}
// classes of the gathered rows of a COO batch: local node t is node order[t]
__global__ void gather_class_kernel(int64_t nl, const int* __restrict__ order, const int* __restrict__ cls, int* __restrict__ out) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < nl) out[t] = cls[order[t]];
}

__global__ void compose_kernel(int64_t n0, int* __restrict__ map0, const int* __restrict__ Hc) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n0) map0[i] = Hc[map0[i]];
}

// rep_of_block[b] = first node of canonical block b (colours canonical => ids ordered by first node)
__global__ void block_rep_kernel(int64_t n, const int* __restrict__ canon, int* __restrict__ rep_of_block) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int b = canon[i];
  if (rep_of_block[b] > (int)i) atomicMin(rep_of_block + b, (int)i);
}

// lower_bound of each query in the increasing array rep_of_block[0..k): number of blocks whose first node is < x
__global__ void rep_lower_bound_kernel(const int* __restrict__ rep_of_block, int64_t k, const int64_t* __restrict__ queries,
                                       int nq, int64_t* __restrict__ out) {
  int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= nq) return;
  const int64_t x = queries[q];
  int64_t lo = 0, hi = k;
  while (lo < hi) {
    int64_t mid = (lo + hi) >> 1;
    if ((int64_t)rep_of_block[mid] < x) lo = mid + 1;
    else hi = mid;
  }
  out[q] = lo;
}

// Quotient, step 1: every entry (i_B, j) of a representative row becomes key (B, H(j)); equal keys meet in one slot whose
// value accumulates the weights (a'_{B,B'} = sum_{l in B'} a_{i_B,l}, Eq. 1).  Slot = {key + 1 : 64 | weight sum : 64},
// empty = {0, 0}.  A new key claims its slot together with its first weight by one 128-bit CAS; only a repeated key
// needs a second atomic (the add).  Returns true when the entry claimed a slot (= one more distinct target for block B).
__device__ __forceinline__ bool quot_insert_one(Slot* __restrict__ table, u64 mask, int b, int target, u64 weight) {
  const u64 key1 = (((u64)(u32)b << 32) | (u64)(u32)target) + 1;
  u64 slot = slot_hash((u32)b, key1) & mask;
  while (true) {
    Slot v = load_slot(table + slot);
    if (v.y == 0) {
      const Slot empty = {0ull, 0ull}, mine = {key1, weight};
      v = cas128(table + slot, empty, mine);
      if (v.y == 0) return true;
    }
    if (v.y == key1) {
      atomicAdd(&table[slot].cx, weight);
      return false;
    }
    slot = (slot + 1) & mask;
  }
}

// The same insertion, but the probe sequence of an entry of row [A, A + len) of the edge array STARTS inside the row's own region
// of the table, slots [2 A, 2 (A + len)) mod the table size (equal keys can only meet inside one row, so nothing is lost; keys
// still carry the block, so regions that wrap or overlap - a row longer than the table, a cut row next to later batches - are
// merely less local, never wrong).  The slots of a short row then share a few 128-byte lines instead of one random sector per
// entry, and the emission, which sweeps the table in slot order, finds the entries of a block next to each other: its output
// positions are consecutive and its writes coalesce.
__device__ __forceinline__ bool quot_insert_at(Slot* __restrict__ table, u64 mask, u64 region_base, u64 region_size, int b,
                                               int target, u64 weight) {
  const u64 key1 = (((u64)(u32)b << 32) | (u64)(u32)target) + 1;
  u64 slot = (region_base + __umul64hi(slot_hash((u32)target, key1), region_size)) & mask;
  while (true) {
    Slot v = load_slot(table + slot);
    if (v.y == 0) {
      const Slot empty = {0ull, 0ull}, mine = {key1, weight};
      v = cas128(table + slot, empty, mine);
      if (v.y == 0) return true;
    }
    if (v.y == key1) {
      atomicAdd(&table[slot].cx, weight);
      return false;
    }
    slot = (slot + 1) & mask;
  }
}
// region of the row whose entries are the positions [A, E) of the edge array (unclipped)
__device__ __forceinline__ void quot_region(int64_t A, int64_t E, u64 mask, u64* base, u64* size) {
  const u64 len = (u64)(E - A);
  *base = 2ull * (u64)A;
  *size = len == 0 ? 1 : (2 * len > mask + 1 ? mask + 1 : 2 * len);
}

constexpr int kQuotLongRow = 4096;  // longer pieces are left to quot_insert_long_kernel (whole grid per row)

// Eight lanes per row of [row_base, row_base + n_rows) (a warp owns four consecutive rows); only the representative row of a block
// contributes (Def. 4, Q17).  The piece of the row inside the uploaded edge range [clip_lo, clip_hi) is inserted: pieces of up to
// kQuotGroupRow entries by the row's eight lanes, longer ones by the whole warp in turn, pieces longer than kQuotLongRow are queued
// in long_rows (a single warp would walk a hub row of 10^5-10^6 entries alone).  (One warp per row left 27 of 32 lanes idle in
// the batches of the low-degree node ranges, 5 entries per row on average: 1.45 ms per 33 M entries at 25 % issue activity and 35
// warps stalled on memory per issue, ncu.)
constexpr int kQuotGroupRow = 64;
// kQuotGroup lanes per row in batches of short rows (4: no different, measured); batches whose rows average more than
// kQuotGroupAvg entries keep one warp per row: there the rows are few (a hub-heavy batch of 33 M entries has 10 000 of them) and
// four rows per warp left three quarters of the warp slots empty (12-38 % warps active, 0.95-2.2 ms per batch, ncu)
constexpr int kQuotGroupShort = 8;
constexpr int kQuotGroupAvg = 24;
template <int kQuotGroup>
__global__ void __launch_bounds__(256)
quot_insert_kernel(int64_t row_base, int64_t n_rows, const int64_t* __restrict__ row_ptr, int64_t clip_lo, int64_t clip_hi,
                   const int* __restrict__ col, const u32* __restrict__ wt, const int* __restrict__ Hc,
                   const int* __restrict__ rep_of_block, const unsigned char* __restrict__ isrep, Slot* __restrict__ table,
                   u64 table_mask, int* __restrict__ cnt, int* __restrict__ long_rows, u32* __restrict__ long_count) {
  constexpr int kQuotRowsPerWarp = 32 / kQuotGroup;
  const int lane = threadIdx.x & 31, sub = lane / kQuotGroup, sl = lane % kQuotGroup;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t w = warp * kQuotRowsPerWarp + sub;
  if (warp * kQuotRowsPerWarp >= n_rows) return;  // (whole warps only)
  int b = 0;
  int64_t a = 0, e = 0;
  u64 rbase = 0, rsize = 1;
  bool live = false;
  if (w < n_rows) {
    const int64_t i = row_base + w;
    b = Hc[i];
    live = isrep ? isrep[i] != 0 : rep_of_block[b] == (int)i;  // representative = first node of its block (Q17)
    if (live) {
      a = row_ptr[w];
      e = row_ptr[w + 1];
      quot_region(a, e, table_mask, &rbase, &rsize);
      if (a < clip_lo) a = clip_lo;
      if (e > clip_hi) e = clip_hi;
      if (e - a > kQuotLongRow) {
        if (sl == 0) long_rows[atomicAdd(long_count, 1u)] = (int)w;
        live = false;
      }
    }
  }
  const bool big = kQuotGroup < 32 && live && e - a > kQuotGroupRow;
  int fresh = 0;
  if (live && !big)
    for (int64_t p = a + sl; p < e; p += kQuotGroup)
      fresh += quot_insert_at(table, table_mask, rbase, rsize, b, Hc[col[p]], wt ? (u64)wt[p] : 1ull) ? 1 : 0;
#pragma unroll
  for (int o = kQuotGroup / 2; o > 0; o >>= 1) fresh += __shfl_xor_sync(0xffffffffu, fresh, o);
  if (sl == 0 && fresh) atomicAdd(cnt + b, fresh);
#pragma unroll 1
  for (int g = 0; g < (kQuotGroup < 32 ? kQuotRowsPerWarp : 0); ++g) {  // the longer pieces of the warp's rows, one after the other, by all 32 lanes
    const int src = g * kQuotGroup;
    if (!__shfl_sync(0xffffffffu, big ? 1 : 0, src)) continue;
    const int64_t ga = __shfl_sync(0xffffffffu, a, src), ge = __shfl_sync(0xffffffffu, e, src);
    const u64 gbase = __shfl_sync(0xffffffffu, rbase, src), gsize = __shfl_sync(0xffffffffu, rsize, src);
    const int gb = __shfl_sync(0xffffffffu, b, src);
    int f = 0;
    for (int64_t p = ga + lane; p < ge; p += 32)
      f += quot_insert_at(table, table_mask, gbase, gsize, gb, Hc[col[p]], wt ? (u64)wt[p] : 1ull) ? 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) f += __shfl_xor_sync(0xffffffffu, f, o);
    if (lane == 0 && f) atomicAdd(cnt + gb, f);
  }
}

// the queued long pieces, cut into chunks of kQuotChunk entries that the CTAs take in turn (chunk g of the whole list goes to CTA
// g mod gridDim: every CTA walks the short list of pieces and keeps the running chunk count, so no prefix array is needed).  The
// work is spread by entries, whatever the mix of 5 k-entry rows and 10^6-entry hub rows (one CTA per piece left most SMs idle:
// 1.19 ms per 33 M-entry batch for the 10-20 % of the entries that sit in such rows).
constexpr int64_t kQuotChunk = 2048;
__global__ void __launch_bounds__(256)
quot_insert_long_kernel(int64_t row_base, const int64_t* __restrict__ row_ptr, int64_t clip_lo, int64_t clip_hi,
                        const int* __restrict__ col, const u32* __restrict__ wt, const int* __restrict__ Hc,
                        Slot* __restrict__ table, u64 table_mask, int* __restrict__ cnt,
                        const int* __restrict__ long_rows, const u32* __restrict__ long_count) {
  const u32 n_long = *long_count;
  u32 chunk0 = 0;  // chunks of the pieces before piece j, mod gridDim (32-bit arithmetic: every thread walks the whole list, and
                   // two 64-bit remainders per piece made this walk most of the kernel: 64 % issue activity for 0.2 GB of DRAM, ncu)
  for (u32 j = 0; j < n_long; ++j) {
    const int64_t w = long_rows[j];
    int64_t a = row_ptr[w], e = row_ptr[w + 1];
    const int64_t a_row = a, e_row = e;
    if (a < clip_lo) a = clip_lo;
    if (e > clip_hi) e = clip_hi;
    const int64_t nch = (e - a + kQuotChunk - 1) / kQuotChunk;  // (kQuotChunk is a power of two)
    // first chunk of this piece that is mine: the smallest q >= 0 with (chunk0 + q) mod gridDim == blockIdx
    u32 q32 = blockIdx.x + gridDim.x - chunk0;
    if (q32 >= gridDim.x) q32 -= gridDim.x;
    chunk0 = (chunk0 + (u32)nch) % gridDim.x;  // (a row has fewer than 2^32 entries: nch < 2^21)
    int64_t q = q32;
    if (q >= nch) continue;
    u64 rbase, rsize;
    quot_region(a_row, e_row, table_mask, &rbase, &rsize);
    const int b = Hc[row_base + w];
    int fresh = 0;
    for (; q < nch; q += gridDim.x) {
      const int64_t ca = a + q * kQuotChunk, ce = ca + kQuotChunk < e ? ca + kQuotChunk : e;
      for (int64_t p = ca + threadIdx.x; p < ce; p += blockDim.x)
        fresh += quot_insert_at(table, table_mask, rbase, rsize, b, Hc[col[p]], wt ? (u64)wt[p] : 1ull) ? 1 : 0;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) fresh += __shfl_xor_sync(0xffffffffu, fresh, o);
    if ((threadIdx.x & 31) == 0 && fresh) atomicAdd(cnt + b, fresh);
  }
}

// Quotient, step 2: every occupied slot is one entry of A'; rows fill from q_row_ptr with an atomic cursor (order inside a
// row is unspecified); the slot is emptied for the next batch.
// Only blocks b_lo <= B < b_hi are emitted (a representative row that continues in the next batch stays in the table).
__global__ void quot_emit_kernel(u64* __restrict__ table, u64 table_slots, const int64_t* __restrict__ q_row_ptr,
                                 int64_t out_base, int* __restrict__ cursor, int* __restrict__ q_col,
                                 u32* __restrict__ q_wt, int b_lo, int b_hi) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  u64 key1 = 0;
  if (s < (int64_t)table_slots) key1 = table[2 * s];
  const u64 key = key1 - 1;
  const int b = (int)(key >> 32), t = (int)(key & 0xffffffffu);
  const bool live = key1 != 0 && b >= b_lo && b < b_hi;
  // neighbouring slots mostly hold entries of one block (quot_insert_at): the lanes of a block reserve their positions together
  const unsigned peers = __match_any_sync(0xffffffffu, live ? b : -1 - lane);
  const int leader = __ffs(peers) - 1;
  int base = 0;
  if (live && lane == leader) base = atomicAdd(cursor + b, __popc(peers));
  base = __shfl_sync(0xffffffffu, base, leader);
  if (!live) return;
  const u64 sum = table[2 * s + 1];
  const int64_t pos = q_row_ptr[b] - out_base + base + __popc(peers & ((1u << lane) - 1));
  q_col[pos] = t;
  q_wt[pos] = (u32)sum;
  table[2 * s] = 0;
  table[2 * s + 1] = 0;
}


// ---------------------------------------------------------------------------------------------------------------------
// COO-form (arbitrary) edge partitions: the first outer iteration of Algorithm 2 for batches given as (src, col, weight)
// triples (Thm 2: "an arbitrary edge partition of E").  Later iterations run on the library's own host CSR quotients.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kLabelNone = -2, kLabelBoundary = -1;

// B2 (Def. 5, by the method of L463): every edge tags its source with its batch; a source seen with two different
// batches is a boundary node.  Also: range check of both endpoints (S0), out-degree and weighted row sum per node.
__global__ void coo_mask_kernel(int64_t ne, const int* __restrict__ src, const int* __restrict__ col,
                                const u32* __restrict__ wt, int k, int64_t n, int* __restrict__ label, int* __restrict__ deg,
                                u64* __restrict__ rowsum, u32* __restrict__ err) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  bool bad = false;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < ne; e += stride) {
    const int s = src[e], c = col[e];
    if ((unsigned)s >= (unsigned)n || (unsigned)c >= (unsigned)n) {
      bad = true;
      continue;
    }
    int old = label[s];
    if (old == kLabelNone) old = atomicCAS(label + s, kLabelNone, k);
    if (old != kLabelNone && old != k && old != kLabelBoundary) label[s] = kLabelBoundary;  // idempotent plain store
    atomicAdd(deg + s, 1);
    if (rowsum) atomicAdd(rowsum + s, (u64)wt[e]);
  }
  if (bad) atomicOr(err, kErrCol);
}

// nodes without out-edges are inner to batch 0 (Q9); per label (index label + 1; 0 = boundary): node and edge counts;
// row sums >= 2^32 (Theorem 1's precondition, L129) and rows of 2^31 entries or more are reported
__global__ void coo_census_kernel(int64_t n, int* __restrict__ label, const int* __restrict__ deg,
                                  const u64* __restrict__ rowsum, u64* __restrict__ nodes_of, u64* __restrict__ edges_of,
                                  u32* __restrict__ err) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = i < n;
  int lab = -3;
  int d = 0;
  if (valid) {
    lab = label[i];
    d = deg[i];
    if (lab == kLabelNone) label[i] = lab = 0;
    if (d < 0 || (rowsum && rowsum[i] >= (1ull << 32))) atomicOr(err, kErrRowSum);
  }
  const unsigned peers = __match_any_sync(0xffffffffu, lab);
  u64 dsum = 0;  // out-degree sum over the lanes that share my label
  for (unsigned mpeers = peers; mpeers; mpeers &= mpeers - 1) dsum += (u64)(u32)__shfl_sync(peers, d, __ffs(mpeers) - 1);
  if (valid && (int)(threadIdx.x & 31) == __ffs(peers) - 1) {
    atomicAdd(nodes_of + (lab + 1), (u64)__popc(peers));
    atomicAdd(edges_of + (lab + 1), dsum);
  }
}

// V_k as a node list: order[off[k] + l] = the l-th inner node of batch k (any order), lid[node] = l
__global__ void coo_order_kernel(int64_t n, const int* __restrict__ label, const int64_t* __restrict__ off,
                                 u32* __restrict__ cursor, int* __restrict__ order, int* __restrict__ lid) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int lab = label[i];
  if (lab < 0) return;
  const u32 l = atomicAdd(cursor + lab, 1u);
  order[off[lab] + l] = (int)i;
  lid[i] = (int)l;
}

// rows of A|E_k restricted to V_k (Alg. 2 line 9 needs only them: a singleton can never split): lengths ...
__global__ void coo_rowlen_kernel(int64_t ne, const int* __restrict__ src, int k, const int* __restrict__ label,
                                  const int* __restrict__ lid, int* __restrict__ rowlen) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < ne; e += stride) {
    const int s = src[e];
    if (label[s] == k) atomicAdd(rowlen + lid[s], 1);
  }
}
// ... and entries.  A target inside V_k is renamed to its local index; any other target j becomes -2 - j (negative, never the
// kernels' "no entry" mark -1), which the RANGED SpMV kernels turn into the implicit singleton id 2^32 + (u32)(-2 - j) of
// H_k^0 (Eq. 3): distinct per node and disjoint from the dense ids.  Entry order inside a row is arbitrary (sums in
// Z/2^64 commute).
__global__ void coo_fill_kernel(int64_t ne, const int* __restrict__ src, const int* __restrict__ col,
                                const u32* __restrict__ wt, int k, const int* __restrict__ label, const int* __restrict__ lid,
                                const int64_t* __restrict__ lrp, int* __restrict__ cursor, int* __restrict__ lcol,
                                u32* __restrict__ lwt) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < ne; e += stride) {
    const int s = src[e];
    if (label[s] != k) continue;
    const int l = lid[s], c = col[e];
    const int64_t p = lrp[l] + atomicAdd(cursor + l, 1);
    lcol[p] = label[c] == k ? lid[c] : -2 - c;
    if (lwt) lwt[p] = wt[e];
  }
}

// Eq. 4 for a node list: H[order[l]] = base + local colour of l
__global__ void coo_merge_kernel(int64_t n_local, const int* __restrict__ order, const int* __restrict__ local_colour, int base,
                                 int* __restrict__ H) {
  const int64_t l = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (l < n_local) H[order[l]] = base + local_colour[l];
}

// Alg. 2 lines 11-12: every boundary node becomes a singleton block with a fresh id (any distinct ids: canonicalised later)
__global__ void coo_boundary_ids_kernel(int64_t n, const int* __restrict__ label, int base, u32* __restrict__ counter,
                                        int* __restrict__ H) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool b = i < n && label[i] == kLabelBoundary;
  const unsigned bal = __ballot_sync(0xffffffffu, b);
  if (!bal) return;
  const int lane = threadIdx.x & 31, leader = __ffs(bal) - 1;
  u32 first = 0;
  if (lane == leader) first = atomicAdd(counter, (u32)__popc(bal));
  first = __shfl_sync(0xffffffffu, first, leader);
  if (b) H[i] = base + (int)(first + __popc(bal & ((1u << lane) - 1)));
}

// the given ids (a host list uploaded in one copy) become singleton blocks base, base + 1, ...
__global__ void singleton_ids_kernel(int64_t count, const int* __restrict__ nodes, int base, int* __restrict__ H) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < count) H[nodes[t]] = base + (int)t;
}

__global__ void max_i32_kernel(int64_t n, const int* __restrict__ a, unsigned long long* __restrict__ out) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  int m = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) m = max(m, a[i]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, (unsigned long long)m);
}

__global__ void rep_degree_kernel(int64_t K, const int* __restrict__ rep_of_block, const int* __restrict__ deg,
                                  int* __restrict__ out) {
  const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b < K) out[b] = deg[rep_of_block[b]];
}

// largest b in (b0, K] with prefix[b] - prefix[b0] <= budget (b0 + 1 if even one row exceeds it)
__global__ void prefix_upper_bound_kernel(const int64_t* __restrict__ prefix, int64_t K, int64_t b0, int64_t budget,
                                          int64_t* __restrict__ out) {
  if (blockIdx.x || threadIdx.x) return;
  const int64_t base = prefix[b0];
  int64_t lo = b0 + 1, hi = K;  // answer in [lo, hi]
  while (lo < hi) {
    const int64_t mid = (lo + hi + 1) >> 1;
    if (prefix[mid] - base <= budget) lo = mid;
    else hi = mid - 1;
  }
  out[0] = lo;
  out[1] = prefix[lo] - base;
}

// which batches hold entries of the representative rows of blocks [b_lo, b_hi): the batch a representative is inner to, or
// every batch for a boundary representative (need[nb] = 1)
__global__ void coo_need_kernel(int64_t b_lo, int64_t b_hi, const int* __restrict__ rep_of_block, const int* __restrict__ label,
                                const int* __restrict__ deg, int nb, int* __restrict__ need) {
  const int64_t b = b_lo + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= b_hi) return;
  const int r = rep_of_block[b];
  if (deg[r] == 0) return;
  const int lab = label[r];
  const int slot = lab < 0 ? nb : lab;
  if (need[slot] == 0) need[slot] = 1;
}

// quotient, COO form: thread per edge; only entries of representative rows of blocks [b_lo, b_hi) are inserted (Def. 4, Q17)
__global__ void quot_insert_coo_kernel(int64_t ne, const int* __restrict__ src, const int* __restrict__ col,
                                       const u32* __restrict__ wt, const int* __restrict__ Hc,
                                       const int* __restrict__ rep_of_block, int b_lo, int b_hi, Slot* __restrict__ table,
                                       u64 table_mask, int* __restrict__ cnt) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < ne; e += stride) {
    const int s = src[e];
    const int b = Hc[s];
    if (b < b_lo || b >= b_hi || rep_of_block[b] != s) continue;
    if (quot_insert_one(table, table_mask, b, Hc[col[e]], wt ? (u64)wt[e] : 1ull)) atomicAdd(cnt + b, 1);
  }
}


// ---------------------------------------------------------------------------------------------------------------------
// Compressed quotient weights.  A quotient entry of an UNWEIGHTED input is a multiplicity whose row sums to the out-degree of the
// block's representative (L447), so almost every weight is tiny: on the host (and on the link, which bounds the batched path) a
// weight travels as ONE byte, 255 meaning "look it up in the overflow list of this emission" ({position inside the emission,
// weight} pairs; a row of out-degree d has at most d / 255 of them).  The kernels themselves keep working on uint32 weights.
// ---------------------------------------------------------------------------------------------------------------------
__global__ void wt_pack_kernel(int64_t tot, const u32* __restrict__ w32, unsigned char* __restrict__ w8, u64* __restrict__ ovf,
                               u32* __restrict__ ovf_count, u32 ovf_cap) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= tot) return;
  const u32 w = w32[i];
  w8[i] = (unsigned char)(w < 255u ? w : 255u);
  if (w >= 255u) {
    const u32 idx = atomicAdd(ovf_count, 1u);
    if (idx < ovf_cap) ovf[idx] = (u64)(u32)i | ((u64)w << 32);
  }
}
__global__ void wt_expand_kernel(int64_t cnt, const unsigned char* __restrict__ w8, u32* __restrict__ w32) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < cnt) w32[i] = (u32)w8[i];
}
// overflow entries of one emission that starts `base_rel` entries after the first entry of the uploaded slice
__global__ void wt_patch_kernel(u32 count, const u64* __restrict__ ovf, int64_t base_rel, int64_t cnt, u32* __restrict__ w32) {
  const u32 t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  const u64 e = ovf[t];
  const int64_t pos = (int64_t)(u32)e + base_rel;
  if (pos >= 0 && pos < cnt) w32[pos] = (u32)(e >> 32);
}

// exclusive scan int32 counts -> int64 offsets (3 kernels)
constexpr int kScanT = 256, kScanI = 8, kScanC = kScanT * kScanI;
static_assert(kScanC == kScan32Chunk, "wl_refine.cu sizes the scan scratch with kScan32Chunk");

__global__ void __launch_bounds__(kScanT)
scan32_sum_kernel(const int* __restrict__ in, int64_t n, u64* __restrict__ bsum) {
  const int64_t base = (int64_t)blockIdx.x * kScanC;
  u64 s = 0;
#pragma unroll
  for (int k = 0; k < kScanI; ++k) {
    int64_t i = base + threadIdx.x + k * kScanT;
    if (i < n) s += (u64)(u32)in[i];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  __shared__ u64 sh[kScanT / 32];
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    u64 t = 0;
    for (int w = 0; w < kScanT / 32; ++w) t += sh[w];
    bsum[blockIdx.x] = t;
  }
}

// exclusive scan of the nb block sums by one CTA (nb = n / 2048: at most 2^20 sums for 2^31 nodes); total -> *total
__global__ void __launch_bounds__(1024) scan64_bsum_kernel(u64* __restrict__ bsum, int64_t nb, u64* __restrict__ total) {
  __shared__ u64 s_w[32];
  __shared__ u64 s_carry;
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int64_t base = 0; base < nb; base += 1024) {
    const int64_t i = base + threadIdx.x;
    const u64 v = i < nb ? bsum[i] : 0;
    u64 x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const u64 t = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += t;
    }
    if (lane == 31) s_w[wid] = x;
    __syncthreads();
    if (wid == 0) {
      const u64 t = s_w[lane];
      u64 xs = t;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const u64 u = __shfl_up_sync(0xffffffffu, xs, o);
        if (lane >= o) xs += u;
      }
      s_w[lane] = xs - t;  // exclusive warp offsets
    }
    __syncthreads();
    const u64 carry = s_carry;
    if (i < nb) bsum[i] = carry + s_w[wid] + x - v;
    __syncthreads();
    if (threadIdx.x == 1023) s_carry = carry + s_w[wid] + x;
    __syncthreads();
  }
  if (threadIdx.x == 0) *total = s_carry;
}

__global__ void __launch_bounds__(kScanT)
scan32_apply_kernel(const int* __restrict__ in, int64_t n, const u64* __restrict__ bsum, int64_t base_off,
                    int64_t* __restrict__ out) {
  const int64_t base = (int64_t)blockIdx.x * kScanC + (int64_t)threadIdx.x * kScanI;
  u32 v[kScanI];
  u64 s = 0;
#pragma unroll
  for (int k = 0; k < kScanI; ++k) {
    v[k] = base + k < n ? (u32)in[base + k] : 0u;
    s += v[k];
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  u64 x = s;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    u64 t = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += t;
  }
  __shared__ u64 sw[kScanT / 32];
  if (lane == 31) sw[wid] = x;
  __syncthreads();
  u64 woff = 0;
  for (int w = 0; w < wid; ++w) woff += sw[w];
  u64 r = (u64)base_off + bsum[blockIdx.x] + woff + x - s;
#pragma unroll
  for (int k = 0; k < kScanI; ++k) {
    if (base + k < n) out[base + k] = (int64_t)r;
    r += v[k];
    if (base + k == n - 1) out[n] = (int64_t)r;
  }
}

// ---------------------------------------------------------------------------------------------------------------------
// host helpers
// ---------------------------------------------------------------------------------------------------------------------
// wl_options.device_workspace for wl_refine_batched: the buffers of an outer iteration are sized by that iteration and given back
// at its end, and cudaFree / cudaMalloc of the same gigabytes once per iteration cost 18 ms each time and now and then 0.4 s
// (measured at scale 26: the whole spread between two runs of the same call; a cudaMemPool of the call's own only moves the cost
// to its destruction).  With a caller-owned arena the call makes no allocation at all: blocks are cut from it first-fit at
// 256-byte granularity and merged with their free neighbours when they come back.  Without one: cudaMalloc / cudaFree.
struct DevPool {
  char* base = nullptr;
  size_t size = 0;
  std::map<size_t, size_t> free_blocks;  // offset -> bytes, disjoint, never adjacent
  std::mutex mu;
  void init(void* arena, size_t bytes) {
    const size_t mis = (size_t)((uintptr_t)arena & 255u);
    const size_t skip = mis ? 256 - mis : 0;
    if (!arena || bytes < skip + 256) return;
    base = (char*)arena + skip;
    size = (bytes - skip) / 256 * 256;
    free_blocks[0] = size;
  }
  void* take(size_t bytes) {
    if (!base) return nullptr;
    const size_t need = (bytes + 255) / 256 * 256;
    std::lock_guard<std::mutex> lock(mu);
    for (auto it = free_blocks.begin(); it != free_blocks.end(); ++it) {
      if (it->second < need) continue;
      const size_t off = it->first, rest = it->second - need;
      free_blocks.erase(it);
      if (rest) free_blocks[off + need] = rest;
      return base + off;
    }
    return nullptr;
  }
  void give(void* p, size_t bytes) {
    size_t off = (size_t)((char*)p - base), len = (bytes + 255) / 256 * 256;
    std::lock_guard<std::mutex> lock(mu);
    auto next = free_blocks.lower_bound(off);
    if (next != free_blocks.end() && next->first == off + len) {
      len += next->second;
      next = free_blocks.erase(next);
    }
    if (next != free_blocks.begin()) {
      auto prev = std::prev(next);
      if (prev->first + prev->second == off) {
        prev->second += len;
        return;
      }
    }
    free_blocks[off] = len;
  }
};
static thread_local DevPool* g_dev_pool = nullptr;  // the arena of the call running on this thread, if any

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  DevPool* from = nullptr;  // where p came from (NULL: cudaMalloc)
  ~DevBuf() { free_now(); }
  void free_now() {
    if (!p) return;
    if (from) {
      cudaDeviceSynchronize();  // what cudaFree implies: nothing on any stream still uses the block when it is handed out again
      from->give(p, bytes);
    } else {
      cudaFree(p);
    }
    p = nullptr;
    from = nullptr;
  }
  int alloc(size_t b, size_t* used, size_t cap) {
    bytes = b ? b : 256;
    if (cap && *used + bytes > cap) return WL_ENOMEM;
    if (g_dev_pool && (p = g_dev_pool->take(bytes))) from = g_dev_pool;
    // (no arena, or no free block of that size left in it although the bytes fit the cap)
    if (!p && cudaMalloc(&p, bytes) != cudaSuccess) {
      cudaGetLastError();
      p = nullptr;
      return WL_ENOMEM;
    }
    *used += bytes;
    return WL_OK;
  }
  void release(size_t* used) {  // give the memory back before the end of the scope
    if (!p) return;
    free_now();
    if (*used >= bytes) *used -= bytes;
    bytes = 0;
  }
  void take(DevBuf& o) {  // becomes the owner of o's block (its own, if any, is freed)
    free_now();
    p = o.p;
    bytes = o.bytes;
    from = o.from;
    o.p = nullptr;
    o.from = nullptr;
  }
  template <typename T>
  T* as() const { return (T*)p; }
};

// Pinned host storage of the quotient graphs (Alg. 2 line 13): two offset arrays (the graph being read and the quotient
// being written) and ONE array pair for the weighted entries.  The first quotient is written while the caller's graph is
// streamed; every later quotient overwrites its predecessor in place: its rows come out in the order of its graph's
// rows and never hold more entries (Def. 4), so the write position never passes the position the streaming pass has
// already uploaded.
struct HostQuot {
  char* base = nullptr;
  bool owned = false;
  int64_t* rp[2] = {nullptr, nullptr};
  int* col = nullptr;
  u32* wt = nullptr;
  int64_t cap_nodes = 0, cap_edges = 0;
  // consume_col / consume_wt: the quotients are written over the caller's own column (and weight) array, so the scratch holds
  // the offset arrays only (plus a weight array when the input has none): WL_FLAG_CONSUME_INPUT
  // wt8 != NULL: weights stored as one byte each + per-emission overflow lists (see wt_pack_kernel); the overflow lists of the
  // two quotient generations alive at a time live in library-owned pinned memory (a few bytes per 255 entries)
  unsigned char* wt8 = nullptr;
  struct Emission {
    int64_t q_begin, q_end;  // entries of the quotient this emission wrote
    size_t ovf_off;          // its overflow list inside Generation::ovf
    u32 count;
  };
  struct Generation {
    std::vector<Emission> em;
    u64* ovf = nullptr;  // {position inside the emission : 32 | weight : 32}
    size_t cap = 0, used = 0;
    bool owned = false;  // pinned by the library (else: inside the caller's workspace)
  } gen[2];
  char* spare = nullptr;  // what the caller's workspace holds beyond the arrays above: room for the overflow lists
  size_t spare_bytes = 0;
  // bytes of overflow lists a workspace should hold on top of bytes_for (two generations)
  static size_t overflow_bytes_for(int64_t m) { return 2 * align_up(sizeof(u64) * (size_t)(m / 255 + 8192)); }
  static size_t bytes_for(int64_t n, int64_t m, bool consume_col = false, bool consume_wt = false, bool compressed = false) {
    return 2 * align_up(sizeof(int64_t) * (size_t)(n + 1)) + (consume_col ? 0 : align_up(sizeof(int) * (size_t)m)) +
           (consume_wt ? 0 : align_up((compressed ? 1 : sizeof(int)) * (size_t)m));
  }
  // start generation g with room for `entries` overflow entries (the weights of a quotient of an unweighted graph sum to at
  // most its edge count, so at most m / 255 of them reach 255)
  int reserve_generation(int g, size_t entries) {
    Generation& G = gen[g];
    G.em.clear();
    G.used = 0;
    const size_t half = spare_bytes / 2 / 256 * 256;
    if (half >= sizeof(u64) * std::max<size_t>(1, entries)) {  // inside the caller's workspace: no cudaHostAlloc / cudaFreeHost
      if (G.ovf && G.owned) cudaFreeHost(G.ovf);               // (they cost up to hundreds of milliseconds now and then)
      G.ovf = (u64*)(spare + (size_t)g * half);
      G.cap = half / sizeof(u64);
      G.owned = false;
      return WL_OK;
    }
    if (G.ovf && (G.cap < entries || !G.owned)) {
      if (G.owned) cudaFreeHost(G.ovf);
      G.ovf = nullptr;
    }
    if (!G.ovf) {
      if (cudaHostAlloc((void**)&G.ovf, sizeof(u64) * std::max<size_t>(1, entries), cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError();
        G.ovf = nullptr;
        return WL_ENOMEM;
      }
      G.cap = entries;
      G.owned = true;
    }
    return WL_OK;
  }
  int init(int64_t n, int64_t m, void* ws, size_t ws_bytes, int* consume_col = nullptr, u32* consume_wt = nullptr,
           bool compressed = false) {
    if (base) return WL_OK;
    const size_t need = bytes_for(n, m, consume_col != nullptr, consume_wt != nullptr, compressed);
    if (ws && ws_bytes >= need) {
      base = (char*)ws;
    } else {
      if (cudaHostAlloc((void**)&base, need, cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError();
        base = nullptr;
        return WL_ENOMEM;
      }
      owned = true;
    }
    size_t off = 0;
    rp[0] = (int64_t*)(base + off);
    off += align_up(sizeof(int64_t) * (size_t)(n + 1));
    rp[1] = (int64_t*)(base + off);
    off += align_up(sizeof(int64_t) * (size_t)(n + 1));
    if (consume_col) {
      col = consume_col;
    } else {
      col = (int*)(base + off);
      off += align_up(sizeof(int) * (size_t)m);
    }
    wt = consume_wt ? consume_wt : (u32*)(base + off);
    if (!consume_wt) off += align_up((compressed ? 1 : sizeof(int)) * (size_t)m);
    if (compressed) {
      wt8 = (unsigned char*)wt;
      wt = nullptr;
    }
    if (!owned && ws_bytes > off) {  // what lies behind the arrays laid out above
      spare = base + off;
      spare_bytes = ws_bytes - off;
    }
    cap_nodes = n;
    cap_edges = m;
    return WL_OK;
  }
  ~HostQuot() {
    if (owned && base) cudaFreeHost(base);
    for (Generation& G : gen)
      if (G.ovf && G.owned) cudaFreeHost(G.ovf);
  }
};

// exclusive scan of cnt[0..n) into out[0..n] starting at base_off (device arrays); bsum: ceil(n / kScanC) + 1 u64
void launch_scan32(const int* cnt, int64_t n, int64_t base_off, int64_t* out, u64* bsum, u64* total, cudaStream_t st) {
  if (n == 0) return;
  const int64_t nb = (n + kScanC - 1) / kScanC;
  ++g_launches; scan32_sum_kernel<<<(unsigned)nb, kScanT, 0, st>>>(cnt, n, bsum);
  ++g_launches; scan64_bsum_kernel<<<1, 1024, 0, st>>>(bsum, nb, total);
  ++g_launches; scan32_apply_kernel<<<(unsigned)nb, kScanT, 0, st>>>(cnt, n, bsum, base_off, out);
}

// step 1 of the quotient for the rows [row_base, row_base + n_rows) whose offsets are row_ptr[0..n_rows]; long_rows needs
// (clip_hi - clip_lo) / kQuotLongRow + 2 ints, *long_count is zeroed here
static void launch_quot_insert(int64_t row_base, int64_t n_rows, const int64_t* row_ptr, int64_t clip_lo, int64_t clip_hi,
                               const int* col, const u32* wt, const int* Hc, const int* rep_of_block,
                               const unsigned char* isrep, u64* table, u64 table_mask, int* cnt, int* long_rows,
                               u32* long_count, cudaStream_t st, int64_t entries_hint) {  // entries_hint: entries of these rows, roughly
  if (n_rows <= 0) return;
  cudaMemsetAsync(long_count, 0, sizeof(u32), st);
  if (entries_hint > kQuotGroupAvg * n_rows) {
    ++g_launches; quot_insert_kernel<32><<<blocks_for(n_rows * 32, 256), 256, 0, st>>>(row_base, n_rows, row_ptr, clip_lo, clip_hi, col, wt, Hc, rep_of_block, isrep, (Slot*)table, table_mask, cnt, long_rows, long_count);
  } else {
    constexpr int rpw = 32 / kQuotGroupShort;
    ++g_launches; quot_insert_kernel<kQuotGroupShort><<<blocks_for((n_rows + rpw - 1) / rpw * 32, 256), 256, 0, st>>>(row_base, n_rows, row_ptr, clip_lo, clip_hi, col, wt, Hc, rep_of_block, isrep, (Slot*)table, table_mask, cnt, long_rows, long_count);
  }
  ++g_launches; quot_insert_long_kernel<<<148 * 8, 256, 0, st>>>(row_base, row_ptr, clip_lo, clip_hi, col, wt, Hc, (Slot*)table, table_mask, cnt, long_rows, long_count);
}

static u64 quot_table_slots(int64_t entries) {
  u64 s = 1024;
  while (s < 2ull * (u64)entries) s <<= 1;
  return s;
}

// Greedy cuts of the CSR edge array (Q13): consecutive runs of at most cap entries, cut on the largest row boundary that
// fits, inside the row only when the row alone exceeds the cap.
static void greedy_cuts(int64_t n, const int64_t* rp, int64_t cap, std::vector<int64_t>& cuts) {
  const int64_t m = rp[n];
  cuts.assign(1, 0);
  while (cuts.back() < m) {
    const int64_t start = cuts.back(), limit = start + cap;
    if (limit >= m) {
      cuts.push_back(m);
      break;
    }
    // largest r with rp[r] <= limit
    const int64_t r = (std::upper_bound(rp, rp + n + 1, limit) - rp) - 1;
    const int64_t b = rp[r];
    cuts.push_back(b > start ? b : limit);
  }
  if (cuts.size() == 1) cuts.push_back(m);  // m == 0: one empty batch
}

// V_k for the batch owning edge positions [c0, c1) (Q9, Q13): nodes whose row position lies in [c0, c1), minus the last
// one if its row crosses c1; the last batch also owns the trailing edgeless nodes.
static void inner_range(int64_t n, const int64_t* rp, int64_t c0, int64_t c1, bool last, int64_t* r0, int64_t* r1) {
  int64_t a = std::lower_bound(rp, rp + n, c0) - rp;  // first node with rp[i] >= c0 (among 0..n-1)
  int64_t b = last ? n : (std::lower_bound(rp, rp + n, c1) - rp);
  if (b > a && rp[b] > c1) --b;  // rows are [rp[i], rp[i+1]): node b-1 crosses the cut
  if (b < a) b = a;
  *r0 = a;
  *r1 = b;
}

}  // namespace wl

using namespace wl;

extern "C" {

int wl_inner_labels(int64_t n, const int64_t* row_ptr, const int32_t* edge_batch, const int32_t* sink_batch,
                    int32_t* label, void* cuda_stream) {
  if (n < 0) return WL_EINVAL;
  if (n == 0) return WL_OK;
  if (!row_ptr || !sink_batch || !label) return WL_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  ++g_launches; inner_labels_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, row_ptr, edge_batch, sink_batch, label);
  int rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  return check_cuda(cudaGetLastError());
}

size_t wl_refine_batched_host_bytes(int64_t n, int64_t m) {
  if (n < 0 || m < 0 || n > kMaxNodes) return 0;
  return HostQuot::bytes_for(n, m);
}

size_t wl_refine_batched_host_bytes_consume(int64_t n, int64_t m, int weighted) {
  if (n < 0 || m < 0 || n > kMaxNodes) return 0;
  return HostQuot::bytes_for(n, m, true, weighted != 0, /*compressed=*/weighted == 0);
}

size_t wl_refine_batched_host_overflow_bytes(int64_t m) { return m < 0 ? 0 : HostQuot::overflow_bytes_for(m); }

size_t wl_quotient_workspace_bytes(int64_t n, int64_t m) {
  if (n < 0 || m < 0 || n > kMaxNodes) return 0;
  size_t off = 0;
  off += align_up(sizeof(u64) * 2 * quot_table_slots(m));
  off += align_up(sizeof(int) * (size_t)n) * 3;  // rep_of_block, cnt, cursor (k <= n)
  off += align_up(sizeof(u64) * (size_t)((n + kScanC - 1) / kScanC + 2));
  off += 256;
  off += align_up(sizeof(int) * (size_t)(m / kQuotLongRow + 2));  // queue of long rows
  return off;
}

int wl_quotient(const wl_csr* g, const int32_t* colors, int64_t k, int64_t* q_row_ptr, int32_t* q_col, uint32_t* q_weights,
                int64_t q_cap, int64_t* q_m, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  int rc = basic_csr_check(g);
  if (rc) return rc;
  const int64_t n = g->n, m = g->m;
  if (k < 0 || k > n || !q_m) return WL_EINVAL;
  *q_m = 0;
  if (n == 0) return WL_OK;
  if (!colors || !q_row_ptr || !workspace || (q_cap > 0 && (!q_col || !q_weights))) return WL_EINVAL;
  if (workspace_bytes < wl_quotient_workspace_bytes(n, m)) return WL_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  size_t off = 0;
  const u64 slots = quot_table_slots(m);
  u64* table = (u64*)(ws + off);
  off += align_up(sizeof(u64) * 2 * slots);
  int* rep_of_block = (int*)(ws + off);
  off += align_up(sizeof(int) * (size_t)n);
  int* cnt = (int*)(ws + off);
  off += align_up(sizeof(int) * (size_t)n);
  int* cursor = (int*)(ws + off);
  off += align_up(sizeof(int) * (size_t)n);
  u64* bsum = (u64*)(ws + off);
  off += align_up(sizeof(u64) * (size_t)((n + kScanC - 1) / kScanC + 2));
  u64* total = (u64*)(ws + off);
  off += 256;
  int* long_rows = (int*)(ws + off);
  cudaMemsetAsync(table, 0, sizeof(u64) * 2 * slots, st);
  if (k > 0) { ++g_launches; fill_kernel<<<blocks_for(k, 256), 256, 0, st>>>(k, rep_of_block, kNoNode); }
  cudaMemsetAsync(cnt, 0, sizeof(int) * (size_t)k, st);
  cudaMemsetAsync(cursor, 0, sizeof(int) * (size_t)k, st);
  ++g_launches; block_rep_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, colors, rep_of_block);
  launch_quot_insert(0, n, g->row_ptr, 0, m, g->col_idx, g->weights, colors, rep_of_block, nullptr, table, slots - 1, cnt, long_rows,
                     (u32*)(total + 1), st, m);
  launch_scan32(cnt, k, 0, q_row_ptr, bsum, total, st);
  u64 h_total = 0;
  cudaMemcpyAsync(&h_total, total, sizeof(u64), cudaMemcpyDeviceToHost, st);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  if (k == 0) h_total = 0;
  *q_m = (int64_t)h_total;
  if ((int64_t)h_total > q_cap) return WL_ENOMEM;
  ++g_launches; quot_emit_kernel<<<blocks_for((int64_t)slots, 256), 256, 0, st>>>(table, slots, q_row_ptr, 0, cursor, q_col, q_weights, 0, (int)k);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  return check_cuda(cudaGetLastError());
}

// ---------------------------------------------------------------------------------------------------------------------
// Algorithm 2
// ---------------------------------------------------------------------------------------------------------------------
}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// Step-level pieces of one outer iteration on DEVICE buffers: what one GPU does for one batch when the batches of Algorithm 2
// are spread over several GPUs (L213, L239; paper_2607_02603_b200/sharded.py drives them and exchanges the block maps).
// ---------------------------------------------------------------------------------------------------------------------
extern "C" {

size_t wl_refine_inner_workspace_bytes(int64_t n_rows, int64_t m) {
  if (n_rows < 0 || m < 0 || n_rows > kMaxNodes) return 0;
  return make_layout(n_rows, m).bytes;
}

int wl_refine_inner(const wl_csr* rows, int64_t lo, int64_t n_targets, uint64_t seed, int32_t* local_colors,
                    uint8_t* is_first, int64_t* num_colors, const wl_options* opt, void* workspace, size_t workspace_bytes,
                    void* cuda_stream) {
  if (!rows || rows->n < 0 || rows->m < 0 || lo < 0 || n_targets < lo + rows->n || n_targets > kMaxNodes) return WL_EINVAL;
  if (num_colors) *num_colors = 0;
  const int64_t nr = rows->n;
  if (nr == 0) return WL_OK;
  if (!rows->row_ptr || (rows->m > 0 && !rows->col_idx) || !local_colors || !is_first || !workspace) return WL_EINVAL;
  const Layout L = make_layout(nr, rows->m);
  if (workspace_bytes < L.bytes) return WL_ENOMEM;
  if ((uintptr_t)workspace % 256) return WL_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  wl_options lo_opt{};
  if (opt) lo_opt = *opt;
  lo_opt.flags &= (WL_FLAG_NO_VALIDATE | WL_FLAG_NO_PRUNE | WL_FLAG_EDGE_BALANCED);
  lo_opt.round_colors = nullptr;
  CoreResult cr{};
  int rc = refine_core(rows, nullptr, seed, &lo_opt, /*ranged=*/true, (int)lo, (int)(lo + nr), n_targets, /*edge_first=*/0,
                       workspace, workspace_bytes, L, st, &cr);
  if (rc) return rc;
  char* wsb = (char*)workspace;
  int* first_l = (int*)(wsb + L.o_tmp);
  launch_canonical(L, nr, cr.colour, local_colors, first_l, (int*)(wsb + L.o_rep), (int*)(wsb + L.o_bsum),
                   (u64*)(wsb + L.o_scal) + kScalCanon, st, cr.k);
  ++g_launches; merge_canon_kernel<<<blocks_for(nr, 256), 256, 0, st>>>(nr, cr.colour, first_l, 0, local_colors, is_first);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  if (num_colors) *num_colors = cr.k;
  return check_cuda(cudaGetLastError());
}

size_t wl_quotient_rows_workspace_bytes(int64_t n_rows, int64_t m, int64_t num_blocks) {
  if (n_rows < 0 || m < 0 || num_blocks < 0) return 0;
  size_t off = 0;
  off += align_up(sizeof(u64) * 2 * quot_table_slots(m));
  off += align_up(sizeof(int) * (size_t)(num_blocks + 1)) * 2;  // cnt, cursor
  off += align_up(sizeof(u64) * (size_t)((num_blocks + kScanC - 1) / kScanC + 2));
  off += 256;
  off += align_up(sizeof(int) * (size_t)(m / kQuotLongRow + 2));
  return off;
}

int wl_quotient_rows(const wl_csr* rows, int64_t lo, const int32_t* block_of, const uint8_t* is_first, int64_t first_block,
                     int64_t num_blocks, int64_t* q_row_ptr, int32_t* q_col, uint32_t* q_weights, int64_t q_cap, int64_t* q_m,
                     void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!rows || rows->n < 0 || rows->m < 0 || lo < 0 || first_block < 0 || num_blocks < 0 || !q_m) return WL_EINVAL;
  *q_m = 0;
  const int64_t nr = rows->n, m = rows->m;
  if (nr == 0 || num_blocks == 0) return WL_OK;
  if (!rows->row_ptr || (m > 0 && !rows->col_idx) || !block_of || !is_first || !q_row_ptr || !workspace) return WL_EINVAL;
  if (q_cap > 0 && (!q_col || !q_weights)) return WL_EINVAL;
  if (workspace_bytes < wl_quotient_rows_workspace_bytes(nr, m, num_blocks)) return WL_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  size_t off = 0;
  const u64 slots = quot_table_slots(m);
  u64* table = (u64*)(ws + off);
  off += align_up(sizeof(u64) * 2 * slots);
  int* cnt = (int*)(ws + off);
  off += align_up(sizeof(int) * (size_t)(num_blocks + 1));
  int* cursor = (int*)(ws + off);
  off += align_up(sizeof(int) * (size_t)(num_blocks + 1));
  u64* bsum = (u64*)(ws + off);
  off += align_up(sizeof(u64) * (size_t)((num_blocks + kScanC - 1) / kScanC + 2));
  u64* total = (u64*)(ws + off);
  off += 256;
  int* long_rows = (int*)(ws + off);
  cudaMemsetAsync(table, 0, sizeof(u64) * 2 * slots, st);
  cudaMemsetAsync(cnt, 0, sizeof(int) * (size_t)(num_blocks + 1), st);
  cudaMemsetAsync(cursor, 0, sizeof(int) * (size_t)(num_blocks + 1), st);
  // the kernels index the block map by global node id and the counters by global block id
  launch_quot_insert(lo, nr, rows->row_ptr, /*clip_lo=*/INT64_MIN / 2, /*clip_hi=*/INT64_MAX / 2, rows->col_idx, rows->weights,
                     block_of, nullptr, is_first - lo, table, slots - 1, cnt - first_block, long_rows, (u32*)(total + 1), st, rows->m);
  launch_scan32(cnt, num_blocks, 0, q_row_ptr, bsum, total, st);
  u64 h_total = 0;
  cudaMemcpyAsync(&h_total, total, sizeof(u64), cudaMemcpyDeviceToHost, st);
  int rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  *q_m = (int64_t)h_total;
  if ((int64_t)h_total > q_cap) return WL_ENOMEM;
  ++g_launches; quot_emit_kernel<<<blocks_for((int64_t)slots, 256), 256, 0, st>>>(table, slots, q_row_ptr - first_block, 0, cursor - first_block, q_col, q_weights, (int)first_block, (int)(first_block + num_blocks));
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  return check_cuda(cudaGetLastError());
}

}  // extern "C"


// ---------------------------------------------------------------------------------------------------------------------
// First outer iteration of Algorithm 2 for COO-form batches (arbitrary edge partition, Thm 2).  Three streaming passes
// over the host-resident batches (double-buffered on copy_st):
//   1. mask    B2: inner labels of Def. 5 by the method of L463 (coo_mask_kernel), out-degrees, validation;
//   2. local   B3-B5: per batch, the rows of V_k are gathered into a local CSR with targets renamed (coo_fill_kernel), refined
//              by refine_core(ranged) and merged (Eq. 4); boundary nodes become singletons;
//   3. quotient B6: block-range major.  The representative rows of an arbitrary partition are scattered over the batches, so
//              the blocks are cut into ranges whose representative rows fit the device table (by out-degree), and for each
//              range the batches that hold entries of those rows are streamed again; rows leave in block order, so the host
//              quotient is the same CSR the CSR-slice path writes.
// On return *K = number of blocks, d_map0 = canonical block map of the original nodes; unless *stopped (N_b = 1 or K = n:
// Alg. 2 line 15), the quotient is in hq.rp[1] / hq.col / hq.wt with *q_m entries.
// ---------------------------------------------------------------------------------------------------------------------
struct CooStats {
  int64_t K = 0, q_m = 0, boundary = 0, bytes_h2d = 0, bytes_d2h = 0, edges_streamed = 0, spmv_alg_bytes = 0;
  double ms_spmv = 0, ms_relabel = 0, ms_spmv_kernel = 0;
  int32_t spmv_launches = 0;
  bool stopped = false;
};

static int coo_first_iteration(int64_t n, int nb, const wl_edge_batch* batches, int64_t m_total, uint64_t seed, uint32_t flags,
                               const wl_options* opt, size_t cap, size_t* used_persistent, DevBuf& d_map0, HostQuot& hq,
                               bool build_quotient, cudaStream_t st, cudaStream_t copy_st, cudaStream_t down_st, CooStats* out,
                               const int* d_cls = nullptr) {  // d_cls: DEVICE int32[n] initial classes or NULL
  bool weighted = false;
  for (int k = 0; k < nb; ++k) weighted |= batches[k].num_edges > 0 && batches[k].weights != nullptr;
  int64_t max_e = 1;
  for (int k = 0; k < nb; ++k) {
    const wl_edge_batch& b = batches[k];
    if (b.num_edges < 0) return WL_EINVAL;
    if (b.num_edges > 0 && (!b.src || !b.col_idx || (b.weights != nullptr) != weighted)) return WL_EINVAL;
    max_e = std::max(max_e, b.num_edges);
  }
  u64* hs = host_scal();
  if (!hs) return WL_ECUDA;
  int rc = WL_OK;
  size_t used = *used_persistent;
  cudaEvent_t ev_up[2], ev_done[2], ev_emit[2], ev_down[2], ev_fence;
  for (int b = 0; b < 2; ++b) {
    cudaEventCreateWithFlags(&ev_up[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_done[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_emit[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_down[b], cudaEventDisableTiming);
  }
  cudaEventCreateWithFlags(&ev_fence, cudaEventDisableTiming);
  struct EvGuard {
    cudaEvent_t* e[9];
    cudaStream_t s[3];
    ~EvGuard() {
      for (cudaStream_t q : s) cudaStreamSynchronize(q);
      for (cudaEvent_t* p : e) cudaEventDestroy(*p);
    }
  } guard{{&ev_up[0], &ev_up[1], &ev_done[0], &ev_done[1], &ev_emit[0], &ev_emit[1], &ev_down[0], &ev_down[1], &ev_fence},
          {st, copy_st, down_st}};

  DevBuf d_label, d_deg, d_rowsum, d_order, d_lid, d_src[2], d_col[2], d_wt[2], d_misc, d_cnts, d_off, d_lcur;
#define COO_ALLOC(buf, bytes) \
  if (!rc) rc = buf.alloc((bytes), &used, cap);
  COO_ALLOC(d_label, sizeof(int) * (size_t)n);
  COO_ALLOC(d_deg, sizeof(int) * (size_t)n);
  if (weighted) COO_ALLOC(d_rowsum, sizeof(u64) * (size_t)n);
  COO_ALLOC(d_order, sizeof(int) * (size_t)n);
  COO_ALLOC(d_lid, sizeof(int) * (size_t)n);
  for (int b = 0; b < 2; ++b) {
    COO_ALLOC(d_src[b], sizeof(int) * (size_t)max_e);
    COO_ALLOC(d_col[b], sizeof(int) * (size_t)max_e);
    if (weighted) COO_ALLOC(d_wt[b], sizeof(u32) * (size_t)max_e);
  }
  COO_ALLOC(d_misc, 4096);
  COO_ALLOC(d_cnts, sizeof(u64) * 2 * (size_t)(nb + 1));
  COO_ALLOC(d_off, sizeof(int64_t) * (size_t)(nb + 1));
  COO_ALLOC(d_lcur, sizeof(u32) * (size_t)(nb + 1));
  if (rc) return rc;
  u32* d_err = (u32*)d_misc.p;                 // validation bits
  u32* d_bcount = (u32*)d_misc.p + 2;          // boundary-id counter
  u64* d_total = (u64*)d_misc.p + 8;           // scan totals
  int64_t* d_ub = (int64_t*)d_misc.p + 16;     // prefix_upper_bound_kernel's two results
  u64* d_nodes_of = d_cnts.as<u64>();
  u64* d_edges_of = d_nodes_of + (nb + 1);

  // one batch into buffer `buf` on the copy stream
  auto upload = [&](int k, int buf, bool with_col_wt) {
    const wl_edge_batch& b = batches[k];
    if (b.num_edges > 0) {
      cudaMemcpyAsync(d_src[buf].p, b.src, sizeof(int) * (size_t)b.num_edges, cudaMemcpyHostToDevice, copy_st);
      out->bytes_h2d += sizeof(int) * b.num_edges;
      if (with_col_wt) {
        cudaMemcpyAsync(d_col[buf].p, b.col_idx, sizeof(int) * (size_t)b.num_edges, cudaMemcpyHostToDevice, copy_st);
        out->bytes_h2d += sizeof(int) * b.num_edges;
        if (weighted) {
          cudaMemcpyAsync(d_wt[buf].p, b.weights, sizeof(u32) * (size_t)b.num_edges, cudaMemcpyHostToDevice, copy_st);
          out->bytes_h2d += sizeof(u32) * b.num_edges;
        }
      }
    }
    cudaEventRecord(ev_up[buf], copy_st);
  };
  // stream the batches `ks` through the two buffers; body(k, buf) queues the work of batch k on `st`.  sync_each: the body
  // leaves `st` idle (it synchronises), so no event is needed before a buffer is overwritten.
  auto stream_batches = [&](const std::vector<int>& ks, auto&& body) -> int {
    if (ks.empty()) return WL_OK;
    cudaEventRecord(ev_fence, st);  // everything queued so far may still read the buffers
    cudaStreamWaitEvent(copy_st, ev_fence, 0);
    upload(ks[0], 0, true);
    for (size_t t = 0; t < ks.size(); ++t) {
      const int buf = (int)(t & 1);
      if (t + 1 < ks.size()) {
        if (t >= 1) cudaStreamWaitEvent(copy_st, ev_done[buf ^ 1], 0);
        upload(ks[t + 1], buf ^ 1, true);
      }
      cudaStreamWaitEvent(st, ev_up[buf], 0);
      const int brc = body(ks[t], buf);
      cudaEventRecord(ev_done[buf], st);
      if (brc) return brc;
    }
    return WL_OK;
  };
  std::vector<int> all(nb);
  for (int k = 0; k < nb; ++k) all[k] = k;

  // ---- pass 1: B2 -------------------------------------------------------------------------------------------------------
  ++g_launches; fill_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, d_label.as<int>(), kLabelNone);
  cudaMemsetAsync(d_deg.p, 0, sizeof(int) * (size_t)n, st);
  if (weighted) cudaMemsetAsync(d_rowsum.p, 0, sizeof(u64) * (size_t)n, st);
  cudaMemsetAsync(d_misc.p, 0, 4096, st);
  cudaMemsetAsync(d_cnts.p, 0, sizeof(u64) * 2 * (size_t)(nb + 1), st);
  rc = stream_batches(all, [&](int k, int buf) -> int {
    const int64_t ne = batches[k].num_edges;
    if (ne > 0) {
      ++g_launches; coo_mask_kernel<<<(unsigned)std::min<int64_t>(blocks_for(ne, 256), 148 * 16), 256, 0, st>>>(ne, d_src[buf].as<int>(), d_col[buf].as<int>(), weighted ? d_wt[buf].as<u32>() : nullptr, k, n, d_label.as<int>(), d_deg.as<int>(), weighted ? d_rowsum.as<u64>() : nullptr, d_err);
    }
    return WL_OK;
  });
  if (rc) return rc;
  ++g_launches; coo_census_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, d_label.as<int>(), d_deg.as<int>(), weighted ? d_rowsum.as<u64>() : nullptr, d_nodes_of, d_edges_of, d_err);
  std::vector<u64> h_cnts(2 * (size_t)(nb + 1));
  cudaMemcpyAsync(h_cnts.data(), d_cnts.p, sizeof(u64) * h_cnts.size(), cudaMemcpyDeviceToHost, st);
  cudaMemcpyAsync(hs, d_misc.p, sizeof(u64), cudaMemcpyDeviceToHost, st);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  {
    const u32 e = (u32)hs[0];
    if (e & kErrCol) return WL_EINVAL;
    if (e & kErrRowSum) return WL_ERANGE;
  }
  const u64* h_nodes_of = h_cnts.data();
  const u64* h_edges_of = h_cnts.data() + (nb + 1);
  out->boundary = (int64_t)h_nodes_of[0];
  std::vector<int64_t> off(nb + 1, 0);
  int64_t max_nl = 1, max_el = 1;
  for (int k = 0; k < nb; ++k) {
    off[k + 1] = off[k] + (int64_t)h_nodes_of[k + 1];
    max_nl = std::max<int64_t>(max_nl, (int64_t)h_nodes_of[k + 1]);
    max_el = std::max<int64_t>(max_el, (int64_t)h_edges_of[k + 1]);
  }
  cudaMemcpyAsync(d_off.p, off.data(), sizeof(int64_t) * (size_t)(nb + 1), cudaMemcpyHostToDevice, st);
  cudaMemsetAsync(d_lcur.p, 0, sizeof(u32) * (size_t)(nb + 1), st);
  ++g_launches; coo_order_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, d_label.as<int>(), d_off.as<int64_t>(), d_lcur.as<u32>(), d_order.as<int>(), d_lid.as<int>());

  // ---- pass 2: B3-B5 ----------------------------------------------------------------------------------------------------
  const int64_t nscan = (n + kCanonChunk - 1) / kCanonChunk;
  DevBuf d_H, d_Hc, d_first, d_cof, d_bsum, d_ws, d_rowlen, d_lrp, d_lcol, d_lwt, d_sbsum;
  size_t ws_bytes = 0;
  for (int k = 0; k < nb; ++k)
    ws_bytes = std::max(ws_bytes, make_layout((int64_t)h_nodes_of[k + 1], (int64_t)h_edges_of[k + 1]).bytes);
  COO_ALLOC(d_H, sizeof(int) * (size_t)n);
  COO_ALLOC(d_Hc, sizeof(int) * (size_t)n);
  COO_ALLOC(d_first, sizeof(int) * (size_t)n);
  COO_ALLOC(d_cof, sizeof(int) * (size_t)n);
  COO_ALLOC(d_bsum, sizeof(int) * canon_scratch_ints(n));
  COO_ALLOC(d_ws, ws_bytes);
  COO_ALLOC(d_rowlen, sizeof(int) * (size_t)max_nl);
  COO_ALLOC(d_lrp, sizeof(int64_t) * (size_t)(max_nl + 1));
  COO_ALLOC(d_lcol, sizeof(int) * (size_t)max_el);
  if (weighted) COO_ALLOC(d_lwt, sizeof(u32) * (size_t)max_el);
  COO_ALLOC(d_sbsum, sizeof(u64) * (size_t)(max_nl / kScanC + 3));
  DevBuf d_lcls;
  if (d_cls) COO_ALLOC(d_lcls, sizeof(int) * (size_t)max_nl);
  if (rc) return rc;
  int64_t base_id = 0;
  rc = stream_batches(all, [&](int k, int buf) -> int {
    const int64_t ne = batches[k].num_edges, nl = (int64_t)h_nodes_of[k + 1], el = (int64_t)h_edges_of[k + 1];
    if (nl == 0) return WL_OK;
    const unsigned egrid = (unsigned)std::max<int64_t>(1, std::min<int64_t>(blocks_for(ne, 256), 148 * 16));
    cudaMemsetAsync(d_rowlen.p, 0, sizeof(int) * (size_t)nl, st);
    if (ne > 0) { ++g_launches; coo_rowlen_kernel<<<egrid, 256, 0, st>>>(ne, d_src[buf].as<int>(), k, d_label.as<int>(), d_lid.as<int>(), d_rowlen.as<int>()); }
    launch_scan32(d_rowlen.as<int>(), nl, 0, d_lrp.as<int64_t>(), d_sbsum.as<u64>(), d_total, st);
    cudaMemsetAsync(d_rowlen.p, 0, sizeof(int) * (size_t)nl, st);  // now the fill cursor
    if (ne > 0) { ++g_launches; coo_fill_kernel<<<egrid, 256, 0, st>>>(ne, d_src[buf].as<int>(), d_col[buf].as<int>(), weighted ? d_wt[buf].as<u32>() : nullptr, k, d_label.as<int>(), d_lid.as<int>(), d_lrp.as<int64_t>(), d_rowlen.as<int>(), d_lcol.as<int>(), weighted ? d_lwt.as<u32>() : nullptr); }
    wl_csr lg;
    lg.n = nl;
    lg.m = el;
    lg.row_ptr = d_lrp.as<int64_t>();
    lg.col_idx = d_lcol.as<int>();
    lg.weights = weighted ? d_lwt.as<u32>() : nullptr;
    wl_options lo{};
    lo.flags = (flags & (WL_FLAG_NO_PRUNE | WL_FLAG_EDGE_BALANCED)) | WL_FLAG_NO_VALIDATE;  // validated in pass 1
    lo.max_rounds = opt ? opt->max_rounds : 0;
    lo.ring_bits = opt ? opt->ring_bits : 0;
    lo.stream_id = (1ull << 32) | (u64)(u32)k;
    const Layout L = make_layout(nl, el);
    CoreResult cr{};
    if (d_cls) { ++g_launches; gather_class_kernel<<<blocks_for(nl, 256), 256, 0, st>>>(nl, d_order.as<int>() + off[k], d_cls, d_lcls.as<int>()); }
    const int prc = refine_core(&lg, d_cls ? d_lcls.as<int>() : nullptr, seed, &lo, /*ranged=*/true, 0, (int)nl, n, 0, d_ws.p, L.bytes, L, st, &cr);
    if (prc) return prc;
    ++g_launches; coo_merge_kernel<<<blocks_for(nl, 256), 256, 0, st>>>(nl, d_order.as<int>() + off[k], cr.colour, (int)base_id, d_H.as<int>());
    base_id += cr.k;
    out->edges_streamed += cr.edges_streamed;
    out->ms_spmv += cr.ms_spmv;
    out->ms_relabel += cr.ms_relabel;
    out->ms_spmv_kernel += cr.ms_spmv_kernel;
    out->spmv_alg_bytes += cr.spmv_alg_bytes;
    out->spmv_launches += cr.spmv_launches;
    return check_cuda(cudaStreamSynchronize(st));  // the workspace and the local CSR are reused by the next batch
  });
  if (rc) return rc;
  if (out->boundary > 0) {
    ++g_launches; coo_boundary_ids_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, d_label.as<int>(), (int)base_id, d_bcount, d_H.as<int>());
    base_id += out->boundary;
  }
  Layout Lc{};
  Lc.nscan = nscan;
  launch_canonical(Lc, n, d_H.as<int>(), d_Hc.as<int>(), d_first.as<int>(), d_cof.as<int>(), d_bsum.as<int>(), d_total, st);
  cudaMemcpyAsync(hs, d_total, sizeof(u64), cudaMemcpyDeviceToHost, st);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  const int64_t K = (int64_t)hs[0];
  out->K = K;
  if ((rc = d_map0.alloc(sizeof(int) * (size_t)n, used_persistent, cap))) return rc;
  used += d_map0.bytes;
  cudaMemcpyAsync(d_map0.p, d_Hc.p, sizeof(int) * (size_t)n, cudaMemcpyDeviceToDevice, st);
  out->stopped = (nb == 1) || (K == n) || !build_quotient;
  if (out->stopped) return check_cuda(cudaStreamSynchronize(st));

  // ---- pass 3: B6, block-range major --------------------------------------------------------------------------------------
  cudaStreamSynchronize(st);
  d_H.release(&used);
  d_first.release(&used);
  d_cof.release(&used);
  d_ws.release(&used);
  d_rowlen.release(&used);
  d_lrp.release(&used);
  d_lcol.release(&used);
  d_lwt.release(&used);
  d_order.release(&used);
  d_lid.release(&used);
  if ((rc = hq.init(n, m_total, opt ? opt->host_workspace : nullptr, opt ? opt->host_workspace_bytes : 0))) return rc;
  int64_t* nrp = hq.rp[1];
  DevBuf d_rep, d_cnt, d_cursor, d_qrp, d_prefix, d_qtab, d_qcol[2], d_qwt[2], d_sb2, d_need;
  COO_ALLOC(d_rep, sizeof(int) * (size_t)K);
  COO_ALLOC(d_cnt, sizeof(int) * (size_t)K);
  COO_ALLOC(d_cursor, sizeof(int) * (size_t)K);
  COO_ALLOC(d_qrp, sizeof(int64_t) * (size_t)(K + 1));
  COO_ALLOC(d_prefix, sizeof(int64_t) * (size_t)(K + 1));
  COO_ALLOC(d_sb2, sizeof(u64) * (size_t)((K + kScanC - 1) / kScanC + 2));
  COO_ALLOC(d_need, sizeof(int) * (size_t)(nb + 1));
  if (rc) return rc;
  ++g_launches; fill_kernel<<<blocks_for(K, 256), 256, 0, st>>>(K, d_rep.as<int>(), kNoNode);
  ++g_launches; block_rep_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, d_Hc.as<int>(), d_rep.as<int>());
  ++g_launches; rep_degree_kernel<<<blocks_for(K, 256), 256, 0, st>>>(K, d_rep.as<int>(), d_deg.as<int>(), d_cnt.as<int>());
  launch_scan32(d_cnt.as<int>(), K, 0, d_prefix.as<int64_t>(), d_sb2.as<u64>(), d_total, st);
  cudaMemsetAsync(d_cnt.p, 0, sizeof(int) * (size_t)K, st);
  cudaMemsetAsync(d_cursor.p, 0, sizeof(int) * (size_t)K, st);
  int64_t max_deg = 0;
  // out_cap: entries one range may hold = max(largest batch, longest row): a range always holds at least one whole row
  {
    int64_t* d_max = d_ub + 4;
    cudaMemsetAsync(d_max, 0, sizeof(int64_t), st);
    ++g_launches; max_i32_kernel<<<(unsigned)std::max<int64_t>(1, std::min<int64_t>(blocks_for(n, 256), 148 * 8)), 256, 0, st>>>(n, d_deg.as<int>(), (unsigned long long*)d_max);
    cudaMemcpyAsync(hs, d_max, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    max_deg = (int64_t)hs[0];
  }
  const int64_t out_cap = std::max<int64_t>(max_e, max_deg);
  const u64 qslots = quot_table_slots(out_cap);
  COO_ALLOC(d_qtab, sizeof(u64) * 2 * qslots);
  for (int b = 0; b < 2; ++b) {
    COO_ALLOC(d_qcol[b], sizeof(int) * (size_t)out_cap);
    COO_ALLOC(d_qwt[b], sizeof(u32) * (size_t)out_cap);
  }
  if (rc) return rc;
  cudaMemsetAsync(d_qtab.p, 0, sizeof(u64) * 2 * qslots, st);
  int64_t q_off = 0, b0 = 0;
  int n_emit = 0;
  std::vector<int> h_need(nb + 1);
  while (b0 < K) {
    ++g_launches; prefix_upper_bound_kernel<<<1, 1, 0, st>>>(d_prefix.as<int64_t>(), K, b0, out_cap, d_ub);
    cudaMemcpyAsync(hs, d_ub, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    const int64_t b1 = (int64_t)hs[0];
    cudaMemsetAsync(d_need.p, 0, sizeof(int) * (size_t)(nb + 1), st);
    ++g_launches; coo_need_kernel<<<blocks_for(b1 - b0, 256), 256, 0, st>>>(b0, b1, d_rep.as<int>(), d_label.as<int>(), d_deg.as<int>(), nb, d_need.as<int>());
    cudaMemcpyAsync(h_need.data(), d_need.p, sizeof(int) * (size_t)(nb + 1), cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    std::vector<int> ks;
    for (int k = 0; k < nb; ++k)
      if ((h_need[k] || h_need[nb]) && batches[k].num_edges > 0) ks.push_back(k);
    rc = stream_batches(ks, [&](int k, int buf) -> int {
      const int64_t ne = batches[k].num_edges;
      ++g_launches; quot_insert_coo_kernel<<<(unsigned)std::min<int64_t>(blocks_for(ne, 256), 148 * 16), 256, 0, st>>>(ne, d_src[buf].as<int>(), d_col[buf].as<int>(), weighted ? d_wt[buf].as<u32>() : nullptr, d_Hc.as<int>(), d_rep.as<int>(), (int)b0, (int)b1, (Slot*)d_qtab.p, qslots - 1, d_cnt.as<int>());
      return WL_OK;
    });
    if (rc) return rc;
    launch_scan32(d_cnt.as<int>() + b0, b1 - b0, q_off, d_qrp.as<int64_t>() + b0, d_sb2.as<u64>(), d_total, st);
    cudaMemcpyAsync(hs, d_total, sizeof(u64), cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    const int64_t tot = (int64_t)hs[0];
    if (tot > out_cap || q_off + tot > hq.cap_edges || b1 > hq.cap_nodes) return WL_ECUDA;  // unreachable (Def. 4)
    const int ob = n_emit & 1;
    if (n_emit >= 2) cudaStreamWaitEvent(st, ev_down[ob], 0);
    ++n_emit;
    ++g_launches; quot_emit_kernel<<<blocks_for((int64_t)qslots, 256), 256, 0, st>>>(d_qtab.as<u64>(), qslots, d_qrp.as<int64_t>(), q_off, d_cursor.as<int>(), d_qcol[ob].as<int>(), d_qwt[ob].as<u32>(), (int)b0, (int)b1);
    cudaEventRecord(ev_emit[ob], st);
    cudaStreamWaitEvent(down_st, ev_emit[ob], 0);
    if (tot) {
      cudaMemcpyAsync(hq.col + q_off, d_qcol[ob].p, sizeof(int) * (size_t)tot, cudaMemcpyDeviceToHost, down_st);
      cudaMemcpyAsync(hq.wt + q_off, d_qwt[ob].p, sizeof(u32) * (size_t)tot, cudaMemcpyDeviceToHost, down_st);
      out->bytes_d2h += (sizeof(int) + sizeof(u32)) * tot;
    }
    cudaMemcpyAsync(nrp + b0, d_qrp.as<int64_t>() + b0, sizeof(int64_t) * (size_t)(b1 - b0 + 1), cudaMemcpyDeviceToHost, down_st);
    out->bytes_d2h += sizeof(int64_t) * (b1 - b0 + 1);
    cudaEventRecord(ev_down[ob], down_st);
    q_off += tot;
    b0 = b1;
  }
  rc = check_cuda(cudaStreamSynchronize(down_st));
  if (!rc) rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  nrp[(size_t)K] = q_off;
  out->q_m = q_off;
  return WL_OK;
#undef COO_ALLOC
}

// Algorithm 2 for a given M_b (the exported entry point below picks M_b from the device cap when the caller gives none)
constexpr int kCompressOverflow = -100;  // internal: an emission held more heavy weights than the device list takes
static thread_local bool g_input_consumed = false;  // WL_FLAG_CONSUME_INPUT: the caller's arrays have been written to (no retry)

static int batched_run(int64_t n, int32_t num_batches, const wl_edge_batch* batches, const wl_csr* whole, uint64_t seed,
                       size_t device_cap_bytes, int64_t max_batch_edges, int32_t* out_colors, wl_stats* stats,
                       const wl_options* opt, void* cuda_stream, bool allow_compress = true) {
  const auto t_entry = std::chrono::steady_clock::now();
  if (stats) std::memset(stats, 0, sizeof(*stats));
  if (n < 0 || num_batches < 0 || max_batch_edges <= 0) return WL_EINVAL;
  if (n > kMaxNodes) return WL_ERANGE;
  if (n == 0) return WL_OK;
  if (!out_colors) return WL_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const uint32_t flags = opt ? opt->flags : 0u;
  const int max_outer = (opt && opt->max_outer_iters > 0) ? opt->max_outer_iters : (1 << 30);

  // ---- the host-resident graph of the current outer iteration ------------------------------------------------------
  const int64_t* rp = nullptr;
  const int* col = nullptr;
  const u32* wt = nullptr;
  std::vector<int64_t> cuts;
  // COO form = arbitrary edge partition (Thm 2): some batch names its sources and none gives CSR offsets (an empty batch
  // may leave all its pointers NULL)
  bool coo = false;
  for (int k = 0; k < num_batches && batches; ++k) coo |= batches[k].src != nullptr;
  if (!coo && num_batches > 0 && batches) {
    bool all_empty = true;
    for (int k = 0; k < num_batches; ++k) all_empty &= batches[k].num_edges == 0 && !batches[k].row_ptr;
    coo = all_empty;  // no edges at all and no offsets: every node is a sink
  }
  int64_t coo_edges = 0;
  if (coo) {
    if (flags & WL_FLAG_INHERIT_BATCHES) return WL_EINVAL;  // Q14b is defined for row-contiguous partitions only
    for (int k = 0; k < num_batches; ++k) {
      if (batches[k].num_edges < 0 || (batches[k].num_edges > 0 && !batches[k].src)) return WL_EINVAL;  // the forms do not mix
      coo_edges += batches[k].num_edges;
    }
  } else if (num_batches > 0) {
    if (!batches) return WL_EINVAL;
    // CSR-slice form: all batches share one row_ptr and tile the edge array consecutively
    rp = batches[0].row_ptr;
    if (!rp) return WL_EINVAL;
    int64_t pos = 0;
    cuts.push_back(0);
    for (int k = 0; k < num_batches; ++k) {
      const wl_edge_batch& b = batches[k];
      if (b.src) return WL_EINVAL;  // the two forms do not mix
      if (b.row_ptr != rp || b.edge_begin != pos || b.num_edges < 0) return WL_EINVAL;
      if (b.num_edges > 0 && !b.col_idx) return WL_EINVAL;
      pos += b.num_edges;
      cuts.push_back(pos);
    }
    if (pos != rp[n]) return WL_EINVAL;
  } else {
    int rc = basic_csr_check(whole);
    if (rc) return rc;
    if (whole->n != n) return WL_EINVAL;
    rp = whole->row_ptr;
    col = whole->col_idx;
    wt = whole->weights;
    if (rp[0] != 0 || rp[n] != whole->m) return WL_EINVAL;
    greedy_cuts(n, rp, max_batch_edges, cuts);
  }
  // per-batch host pointers of iteration 1 (slices may live in separate allocations)
  auto batch_col = [&](int k) -> const int* { return num_batches > 0 ? batches[k].col_idx : col + cuts[k]; };
  auto batch_wt = [&](int k) -> const u32* {
    return num_batches > 0 ? batches[k].weights : (wt ? wt + cuts[k] : nullptr);
  };
  bool weighted = num_batches > 0 ? (batches[0].weights != nullptr) : (wt != nullptr);
  // WL_FLAG_CONSUME_INPUT: the quotient of iteration 1 is written over the rows it was made from (its rows come out in row order
  // and never hold more entries, Def. 4), exactly as every later quotient overwrites its predecessor
  const bool consume = (flags & WL_FLAG_CONSUME_INPUT) != 0;
  if (consume && num_batches != 0) return WL_EINVAL;  // only the whole-CSR form owns one contiguous column array
  // quotient weights of an unweighted input travel as one byte + overflow lists (wt_pack_kernel)
  const bool compress = allow_compress && !coo && !weighted;
  // S0 on the host side of the CSR forms: the offsets steer the cuts, the inner ranges and every upload size
  int64_t max_row_cur = INT64_MAX;  // longest row of the current graph, when known (it bounds the rows of its quotient, Def. 4)
  if (!coo && !(flags & WL_FLAG_NO_VALIDATE)) {
    if (rp[0] != 0) return WL_EINVAL;
    // (one pass over 8 (n + 1) bytes of host memory: 72 ms on one core at n = 2^26, so it is spread over a few threads)
    const int nth = n < (1 << 20) ? 1 : (int)std::min<unsigned>(8, std::max(1u, std::thread::hardware_concurrency()));
    std::vector<int64_t> longest_of(nth, 0);
    std::vector<int> bad_of(nth, 0);
    auto scan = [&](int t) {
      const int64_t i0 = n * t / nth, i1 = n * (t + 1) / nth;
      int64_t longest = 0;
      int bad = 0;
      for (int64_t i = i0; i < i1; ++i) {
        const int64_t d = rp[i + 1] - rp[i];
        if (d < 0) bad |= 1;
        else if ((u64)d >= (1ull << 32)) bad |= 2;
        longest = std::max(longest, d);
      }
      longest_of[t] = longest;
      bad_of[t] = bad;
    };
    {
      std::vector<std::thread> pool;
      for (int t = 1; t < nth; ++t) pool.emplace_back(scan, t);
      scan(0);
      for (std::thread& th : pool) th.join();
    }
    int64_t longest = 0;
    int bad = 0;
    for (int t = 0; t < nth; ++t) {
      longest = std::max(longest, longest_of[t]);
      bad |= bad_of[t];
    }
    if (bad & 1) return WL_EINVAL;
    if (bad & 2) return WL_ERANGE;
    max_row_cur = longest;
  }

  // initial classes (reading Q18): the class of every node of the CURRENT graph stays on the device (d_cls, below)
  const int32_t* init_host = opt ? opt->batched_init_colors : nullptr;
  if (init_host && !(flags & WL_FLAG_NO_VALIDATE))
    for (int64_t i = 0; i < n; ++i)
      if (init_host[i] < 0) return WL_EINVAL;

  u64* hs = host_scal();
  if (!hs) return WL_ECUDA;
  int dev_id = 0;
  cudaGetDevice(&dev_id);
  // the caller's device arena, if any (declared before every DevBuf and before the helper thread: it goes last)
  struct PoolScope {
    DevPool pool;
    DevPool* before;
    PoolScope(void* arena, size_t bytes) : before(g_dev_pool) {
      pool.init(arena, bytes);
      g_dev_pool = pool.base ? &pool : nullptr;
    }
    ~PoolScope() { g_dev_pool = before; }
  } pool_scope(opt ? opt->device_workspace : nullptr, opt ? opt->device_workspace_bytes : 0);
  PieceWorker piece_worker(dev_id);  // (declared before everything its tasks touch: it is joined last)
  cudaStream_t copy_st, down_st, side_st;  // uploads; return of quotient rows; refinement of emitted pieces (inherit)
  if (cudaStreamCreateWithFlags(&copy_st, cudaStreamNonBlocking) != cudaSuccess) return check_cuda(cudaGetLastError());
  if (cudaStreamCreateWithFlags(&down_st, cudaStreamNonBlocking) != cudaSuccess) {
    cudaStreamDestroy(copy_st);
    return check_cuda(cudaGetLastError());
  }
  if (cudaStreamCreateWithFlags(&side_st, cudaStreamNonBlocking) != cudaSuccess) {
    cudaStreamDestroy(copy_st);
    cudaStreamDestroy(down_st);
    return check_cuda(cudaGetLastError());
  }
  cudaEvent_t ev_begin, ev_end, ev_up[2], ev_ins[2], ev_emit[2], ev_down[2], ev_piece[2], ev_stage[2], ev_staged[2];
  cudaEventCreate(&ev_begin);
  cudaEventCreate(&ev_end);
  for (int b = 0; b < 2; ++b) {
    cudaEventCreateWithFlags(&ev_up[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_ins[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_emit[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_down[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_piece[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_stage[b], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&ev_staged[b], cudaEventDisableTiming);
  }
  cudaEventRecord(ev_begin, st);
  auto cleanup = [&]() {
    cudaStreamSynchronize(copy_st);
    cudaStreamSynchronize(down_st);
    cudaStreamSynchronize(side_st);
    cudaEventDestroy(ev_begin);
    cudaEventDestroy(ev_end);
    for (int b = 0; b < 2; ++b) {
      cudaEventDestroy(ev_up[b]);
      cudaEventDestroy(ev_ins[b]);
      cudaEventDestroy(ev_emit[b]);
      cudaEventDestroy(ev_down[b]);
      cudaEventDestroy(ev_piece[b]);
      cudaEventDestroy(ev_stage[b]);
      cudaEventDestroy(ev_staged[b]);
    }
    cudaStreamDestroy(copy_st);
    cudaStreamDestroy(down_st);
    cudaStreamDestroy(side_st);
  };

  const int64_t n0 = n;
  size_t used = 0;
  DevBuf d_map0;  // original node -> node of the current graph (identity in iteration 1: left unallocated until needed)
  bool map0_identity = true;
  // under a tight device cap the composed map stays on the host (see the compose step)
  const bool map0_on_host = !coo && device_cap_bytes > 0 && (size_t)n0 * sizeof(int) * 8 > device_cap_bytes;
  HostQuot hq;  // quotient graphs of later iterations (pinned host memory)
  const int64_t rp0_edges = coo ? coo_edges : rp[n];
  DevBuf d_cls, d_cls_next;  // initial classes of the nodes of the current graph / of its quotient (persistent: counted in `used`)
  if (init_host) {
    const int arc = d_cls.alloc(sizeof(int) * (size_t)n0, &used, device_cap_bytes);
    if (arc) {
      cleanup();
      return arc;
    }
    cudaMemcpyAsync(d_cls.p, init_host, sizeof(int) * (size_t)n0, cudaMemcpyHostToDevice, st);
  }

  int64_t n_t = n;
  int outer = 0;
  int64_t nb_last = 0, boundary_first = 0, edges_streamed = 0, bytes_h2d = 0, bytes_d2h = 0, K_final = 0;
  double ms_spmv = 0, ms_relabel = 0, ms_spmv_kernel = 0;
  int64_t spmv_alg_bytes = 0;
  int32_t spmv_launches = 0;
  const int64_t launches_at_entry = g_launches;
  int rc = WL_OK;
  bool hit_limit = false;
  if (init_host) bytes_h2d += sizeof(int) * n0;

  // WL_FLAG_INHERIT_BATCHES (reading Q14b): the local refinement of the NEXT outer iteration runs on the quotient rows while
  // they are still on the device, batch = the rows emitted together; the next iteration then starts at the merge.
  const bool inherit = (flags & WL_FLAG_INHERIT_BATCHES) != 0;
  bool have_next = false;          // the coming iteration's local refinement is done already
  DevBuf d_Hnext_keep, d_isrep_keep;  // ... its canonical block map and representative flags
  std::vector<int64_t> node_cuts;  // ... and the node ranges of its batches
  int64_t next_base_id = 0;
  const bool debug = debug_enabled();
  auto wall = [] { return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count(); };
  double t_mark = wall();
  if (debug)
    std::fprintf(stderr, "[wl_refine_batched] host pass over the offsets (S0), streams, events %9.3f ms\n",
                 std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_entry).count());
  auto phase = [&](const char* what) {  // WL_DEBUG: host wall-clock per phase (each phase ends on a synchronised stream)
    if (!debug) return;
    cudaStreamSynchronize(st);
    const double t = wall();
    std::fprintf(stderr, "[wl_refine_batched] outer %d %-22s %9.3f ms\n", outer, what, 1e3 * (t - t_mark));
    t_mark = t;
  };
  // COO-form batches: the first outer iteration has its own three-pass driver; its quotient is an ordinary host CSR, so
  // the loop below takes over from iteration 2
  bool loop_done = false;
  if (coo) {
    outer = 1;
    CooStats cs;
    rc = coo_first_iteration(n, num_batches, batches, coo_edges, seed, flags, opt, device_cap_bytes, &used, d_map0, hq,
                             /*build_quotient=*/max_outer > 1, st, copy_st, down_st, &cs, init_host ? d_cls.as<int>() : nullptr);
    edges_streamed += cs.edges_streamed;
    bytes_h2d += cs.bytes_h2d;
    bytes_d2h += cs.bytes_d2h;
    ms_spmv += cs.ms_spmv;
    ms_relabel += cs.ms_relabel;
    ms_spmv_kernel += cs.ms_spmv_kernel;
    spmv_alg_bytes += cs.spmv_alg_bytes;
    spmv_launches += cs.spmv_launches;
    if (rc) {
      loop_done = true;
    } else {
      map0_identity = false;
      nb_last = num_batches;
      K_final = cs.K;
      boundary_first = cs.boundary;
      if (cs.stopped) {
        loop_done = true;
        hit_limit = !(num_batches == 1 || cs.K == n);  // stopped by max_outer_iters only
      } else {
        if (init_host) {  // classes of the blocks, through the composed map of iteration 1
          rc = d_cls_next.alloc(sizeof(int) * (size_t)cs.K, &used, device_cap_bytes);
          if (!rc) {
            ++g_launches; class_of_blocks_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, d_map0.as<int>(), d_cls.as<int>(), d_cls_next.as<int>());
            rc = check_cuda(cudaStreamSynchronize(st));
          }
          d_cls.release(&used);
          d_cls.take(d_cls_next);
          if (rc) loop_done = true;
        }
        rp = hq.rp[1];
        n_t = cs.K;
        weighted = true;
        std::vector<int64_t> next_cuts;
        greedy_cuts(n_t, rp, max_batch_edges, next_cuts);
        if ((flags & WL_FLAG_AGGRESSIVE_STOP) && (int64_t)next_cuts.size() - 1 >= num_batches) loop_done = true;  // L328
        else cuts.swap(next_cuts);
      }
    }
    phase("COO first iteration");
  }
  while (!loop_done) {
    ++outer;
    const int nb = (int)cuts.size() - 1;
    // inner ranges and sizes
    std::vector<int64_t> r0(nb), r1(nb);
    int64_t max_rows = 1, max_edges = 1;
    for (int k = 0; k < nb; ++k) {
      if (have_next) {  // inherited batches hold whole rows of a known node range
        r0[k] = node_cuts[k];
        r1[k] = node_cuts[k + 1];
      } else {
        inner_range(n_t, rp, cuts[k], cuts[k + 1], k == nb - 1, &r0[k], &r1[k]);
      }
      max_rows = std::max(max_rows, r1[k] - r0[k]);
      max_edges = std::max(max_edges, cuts[k + 1] - cuts[k]);
    }
    size_t ws_bytes = 0;
    for (int k = 0; k < nb && !have_next; ++k)
      ws_bytes = std::max(ws_bytes, make_layout(r1[k] - r0[k], rp[r1[k]] - rp[r0[k]]).bytes);

    // ---- device memory of this outer iteration ---------------------------------------------------------------------
    // Per node of the current graph the device holds the canonical block map (4 B) and a representative flag (1 B), plus the
    // composed map of the original nodes (4 B per original node); everything else is sized by a batch (O(n / N_b)): the
    // batches and the boundary nodes between them are merged in node order with locally canonical ids, so the global ids
    // are canonical without a pass over all nodes, and the per-block counters of the quotient pass live in a window.
    size_t used_iter = used;
    DevBuf d_Hc, d_isrep, d_ws, d_col[2], d_wt[2], d_rp[2], d_cnt, d_cursor, d_qrp[2], d_qtab, d_qcol[2], d_qwt[2], d_sbsum,
        d_misc, d_query, d_long, d_Hnext, d_isrep_next, d_ws2, d_wt8[2], d_ovf_up[2], d_qwt8[2], d_qovf[2], d_stg_rp[2],
        d_stg_col[2], d_stg_wt[2];
    // the graph of this iteration has compressed weights (it is a quotient this call wrote)
    const bool read_compressed = compress && outer > 1;
    HostQuot::Generation& Gr = hq.gen[(outer & 1) ^ 1];  // overflow lists of the graph being read
    size_t max_up_ovf = 1;
    if (read_compressed) {
      for (int k = 0; k < nb; ++k) {  // overflow entries a batch may need: those of the emissions it overlaps
        size_t need = 0;
        for (const HostQuot::Emission& e : Gr.em)
          if (e.q_begin < cuts[k + 1] && e.q_end > cuts[k]) need += e.count;
        max_up_ovf = std::max(max_up_ovf, need);
      }
    }
    // every allocation of the iteration goes through here: the first failure (device cap or cudaMalloc) sticks
#define WL_ALLOC(buf, bytes) \
  if (!rc) rc = buf.alloc((bytes), &used_iter, device_cap_bytes);
    if (have_next) {  // made by the previous iteration's quotient pass
      d_Hc.take(d_Hnext_keep);
      d_isrep.take(d_isrep_keep);
      used_iter += d_Hc.bytes + d_isrep.bytes;
      if (device_cap_bytes && used_iter > device_cap_bytes) rc = WL_ENOMEM;
    } else {
      WL_ALLOC(d_Hc, sizeof(int) * (size_t)n_t);
      WL_ALLOC(d_isrep, (size_t)n_t);
    }
    WL_ALLOC(d_ws, ws_bytes);
    for (int b = 0; b < 2; ++b) {
      WL_ALLOC(d_col[b], sizeof(int) * (size_t)max_edges);
      if (weighted) WL_ALLOC(d_wt[b], sizeof(u32) * (size_t)max_edges);
      if (read_compressed) {
        WL_ALLOC(d_wt8[b], (size_t)max_edges);
        WL_ALLOC(d_ovf_up[b], sizeof(u64) * max_up_ovf);
      }
      WL_ALLOC(d_rp[b], sizeof(int64_t) * (size_t)(max_rows + 4));  // the quotient pass adds the rows cut at either end
    }
    WL_ALLOC(d_misc, 4096);
    if (rc) break;
    cudaMemsetAsync(d_misc.p, 0, 4096, st);
    // weights of the edge positions [c0, c1) of the current graph into d_wt[buf], on the copy stream
    auto upload_weights = [&](int k, int buf, int64_t c0, int64_t c1) {
      if (!weighted || c1 <= c0) return;
      const int64_t cnt = c1 - c0;
      if (!read_compressed) {
        const u32* hw = (outer == 1) ? batch_wt(k) : hq.wt + c0;
        cudaMemcpyAsync(d_wt[buf].p, hw, sizeof(u32) * (size_t)cnt, cudaMemcpyHostToDevice, copy_st);
        bytes_h2d += sizeof(u32) * cnt;
        return;
      }
      cudaMemcpyAsync(d_wt8[buf].p, hq.wt8 + c0, (size_t)cnt, cudaMemcpyHostToDevice, copy_st);
      bytes_h2d += cnt;
      ++g_launches; wt_expand_kernel<<<blocks_for(cnt, 256), 256, 0, copy_st>>>(cnt, d_wt8[buf].as<unsigned char>(), d_wt[buf].as<u32>());
      size_t at = 0;
      for (const HostQuot::Emission& e : Gr.em) {
        if (e.count == 0 || e.q_begin >= c1 || e.q_end <= c0) continue;
        u64* d_list = d_ovf_up[buf].as<u64>() + at;
        cudaMemcpyAsync(d_list, Gr.ovf + e.ovf_off, sizeof(u64) * e.count, cudaMemcpyHostToDevice, copy_st);
        bytes_h2d += sizeof(u64) * e.count;
        ++g_launches; wt_patch_kernel<<<blocks_for(e.count, 256), 256, 0, copy_st>>>(e.count, d_list, e.q_begin - c0, cnt, d_wt[buf].as<u32>());
        at += e.count;
      }
    };

    auto upload_batch = [&](int k, int buf) {
      const int64_t c0 = cuts[k], c1 = cuts[k + 1];
      const int* hc = (outer == 1) ? batch_col(k) : hq.col + c0;
      if (c1 > c0) {
        cudaMemcpyAsync(d_col[buf].p, hc, sizeof(int) * (size_t)(c1 - c0), cudaMemcpyHostToDevice, copy_st);
        bytes_h2d += sizeof(int) * (c1 - c0);
        upload_weights(k, buf, c0, c1);
      }
      const int64_t nr = r1[k] - r0[k];
      cudaMemcpyAsync(d_rp[buf].p, rp + r0[k], sizeof(int64_t) * (size_t)(nr + 1), cudaMemcpyHostToDevice, copy_st);
      bytes_h2d += sizeof(int64_t) * (nr + 1);
      cudaEventRecord(ev_up[buf], copy_st);
    };

    phase("alloc");
    // ---- Alg. 2 lines 7-12: local refinement per batch, merge (Eq. 4), boundary singletons, in node order -------------
    int64_t base_id = have_next ? next_base_id : 0;  // have_next: the whole block map was made by the previous quotient pass
    int64_t n_boundary = 0;
    auto gap = [&](int64_t g0, int64_t g1) {  // the nodes g0 .. g1 - 1 lie between two inner ranges: boundary nodes
      if (g1 <= g0) return;
      ++g_launches; gap_singletons_kernel<<<blocks_for(g1 - g0, 256), 256, 0, st>>>(g0, g1 - g0, (int)base_id, d_Hc.as<int>(), d_isrep.as<unsigned char>());
      base_id += g1 - g0;
      n_boundary += g1 - g0;
    };
    cudaStreamSynchronize(st);  // buffers of the previous iteration are free
    if (!have_next) upload_batch(0, 0);
    int64_t next_node = 0;
    for (int k = 0; k < nb && !rc && !have_next; ++k) {
      const int buf = k & 1;
      if (k + 1 < nb) upload_batch(k + 1, buf ^ 1);
      cudaStreamWaitEvent(st, ev_up[buf], 0);
      const int64_t nr = r1[k] - r0[k];
      if (outer == 1 && !(flags & WL_FLAG_NO_VALIDATE) && cuts[k + 1] > cuts[k]) {
        // S0 for the entries outside the inner rows (rows cut by a batch border are never seen by refine_core, yet the
        // quotient pass maps every stored target through the block map): range check of the WHOLE uploaded slice
        ++g_launches; slice_cols_check_kernel<<<148 * 8, 256, 0, st>>>(n_t, cuts[k + 1] - cuts[k], d_col[buf].as<int>(), (u32*)d_misc.p + 64);
      }
      gap(next_node, r0[k]);
      next_node = std::max(next_node, r1[k]);
      if (nr == 0) {  // a batch inside one cut row: nothing to refine, but its range check must have read the buffer before
                      // the upload after next reuses it (the synchronisation that ends every other batch)
        rc = check_cuda(cudaStreamSynchronize(st));
        continue;
      }
      const int64_t e0 = rp[r0[k]], e1 = rp[r1[k]];
      wl_csr lg;
      lg.n = nr;
      lg.m = e1 - e0;
      lg.row_ptr = d_rp[buf].as<int64_t>();
      lg.col_idx = d_col[buf].as<int>() - cuts[k];  // row offsets are global edge positions
      lg.weights = weighted ? d_wt[buf].as<u32>() - cuts[k] : nullptr;
      wl_options lo{};
      lo.flags = flags & (WL_FLAG_NO_VALIDATE | WL_FLAG_NO_PRUNE | WL_FLAG_EDGE_BALANCED);
      if (outer > 1) lo.flags |= WL_FLAG_NO_VALIDATE;  // a quotient made by this library is well formed and keeps row sums (L447)
      lo.max_rounds = opt ? opt->max_rounds : 0;
      lo.ring_bits = opt ? opt->ring_bits : 0;
      lo.stream_id = ((u64)outer << 32) | (u64)(u32)k;
      const Layout L = make_layout(nr, lg.m);
      CoreResult cr{};
      rc = refine_core(&lg, init_host ? d_cls.as<int>() + r0[k] : nullptr, seed, &lo, /*ranged=*/true, (int)r0[k], (int)r1[k], n_t, e0, d_ws.p, L.bytes, L, st, &cr);
      if (rc) break;
      // canonical ids inside the batch (scratch: two dead arrays of the local workspace, as wl_refine does), then Eq. 4
      char* wsb = (char*)d_ws.p;
      int* first_l = (int*)(wsb + L.o_tmp);
      launch_canonical(L, nr, cr.colour, d_Hc.as<int>() + r0[k], first_l, (int*)(wsb + L.o_rep), (int*)(wsb + L.o_bsum),
                       (u64*)(wsb + L.o_scal) + kScalCanon, st, cr.k);
      ++g_launches; merge_canon_kernel<<<blocks_for(nr, 256), 256, 0, st>>>(nr, cr.colour, first_l, (int)base_id, d_Hc.as<int>() + r0[k], d_isrep.as<unsigned char>() + r0[k]);
      base_id += cr.k;
      edges_streamed += cr.edges_streamed;
      ms_spmv += cr.ms_spmv;
      ms_relabel += cr.ms_relabel;
      ms_spmv_kernel += cr.ms_spmv_kernel;
      spmv_alg_bytes += cr.spmv_alg_bytes;
      spmv_launches += cr.spmv_launches;
      rc = check_cuda(cudaStreamSynchronize(st));  // the workspace and this buffer are reused by the next batch
    }
    if (rc) break;
    if (!have_next) gap(next_node, n_t);
    if (outer == 1) boundary_first = n_boundary;
    if (outer == 1 && !(flags & WL_FLAG_NO_VALIDATE)) {
      cudaMemcpyAsync(hs + kNumScal + 2, (u32*)d_misc.p + 64, sizeof(u32), cudaMemcpyDeviceToHost, st);
      rc = check_cuda(cudaStreamSynchronize(st));
      if (rc) break;
      if ((u32)hs[kNumScal + 2] & kErrCol) {
        rc = WL_EINVAL;
        break;
      }
      // row sums of the rows cut by a batch border (Theorem 1's precondition, L129): at most nb - 1 rows, summed on the host
      // from the caller's weight arrays (refine_core checks the inner rows on the device)
      if (weighted) {
        for (int k = 1; k < nb && !rc; ++k) {
          const int64_t r = (std::upper_bound(rp, rp + n_t + 1, cuts[k]) - rp) - 1;
          if (r < 0 || r >= n_t || rp[r] >= cuts[k]) continue;  // the cut falls on a row boundary
          u64 sum = 0;
          for (int j = 0; j < nb; ++j) {
            const int64_t a = std::max(rp[r], cuts[j]), b = std::min(rp[r + 1], cuts[j + 1]);
            const u32* w = batch_wt(j);
            for (int64_t p = a; p < b; ++p) sum += w[p - cuts[j]];
          }
          if (sum >= (1ull << 32)) rc = WL_ERANGE;
        }
        if (rc) break;
      }
    }
    phase("local refinement + merge");
    const int64_t K = base_id;  // the ids are canonical: K blocks
    nb_last = nb;
    K_final = K;
    // compose original -> current map
    if (map0_on_host) {
      // the composed map (4 bytes per ORIGINAL node) lives in the caller's out_colors between iterations and passes through
      // the device in tiles: at n = 2^30 it would take a quarter of a 16 GB cap for one use per iteration
      if (map0_identity) {
        cudaMemcpyAsync(out_colors, d_Hc.p, sizeof(int) * (size_t)n0, cudaMemcpyDeviceToHost, st);
        bytes_d2h += sizeof(int) * n0;
        map0_identity = false;
      } else {
        const int64_t tile = std::min<int64_t>(n0, 1ll << 26);
        DevBuf d_tile;
        if ((rc = d_tile.alloc(sizeof(int) * (size_t)tile, &used_iter, device_cap_bytes))) break;
        for (int64_t t0 = 0; t0 < n0; t0 += tile) {
          const int64_t cnt = std::min(tile, n0 - t0);
          cudaMemcpyAsync(d_tile.p, out_colors + t0, sizeof(int) * (size_t)cnt, cudaMemcpyHostToDevice, st);
          ++g_launches; compose_kernel<<<blocks_for(cnt, 256), 256, 0, st>>>(cnt, d_tile.as<int>(), d_Hc.as<int>());
          cudaMemcpyAsync(out_colors + t0, d_tile.p, sizeof(int) * (size_t)cnt, cudaMemcpyDeviceToHost, st);
          bytes_h2d += sizeof(int) * cnt;
          bytes_d2h += sizeof(int) * cnt;
        }
        cudaStreamSynchronize(st);
        d_tile.release(&used_iter);
      }
    } else if (map0_identity) {
      if ((rc = d_map0.alloc(sizeof(int) * (size_t)n0, &used, device_cap_bytes))) break;
      used_iter += d_map0.bytes;
      cudaMemcpyAsync(d_map0.p, d_Hc.p, sizeof(int) * (size_t)n0, cudaMemcpyDeviceToDevice, st);
      map0_identity = false;
    } else {
      ++g_launches; compose_kernel<<<blocks_for(n0, 256), 256, 0, st>>>(n0, d_map0.as<int>(), d_Hc.as<int>());
    }
    // ---- Alg. 2 line 15 (L200, Q15) -----------------------------------------------------------------------------------
    bool stop = (nb == 1) || (K == n_t);
    if (!stop && outer >= max_outer) {
      stop = true;
      hit_limit = true;
    }
    if (stop) {
      rc = check_cuda(cudaStreamSynchronize(st));
      break;
    }

    if (init_host) {  // classes of the K blocks = of the nodes of the quotient (ready before the first piece is refined)
      if ((rc = d_cls_next.alloc(sizeof(int) * (size_t)K, &used, device_cap_bytes))) break;
      used_iter += d_cls_next.bytes;
      ++g_launches; class_of_blocks_kernel<<<blocks_for(n_t, 256), 256, 0, st>>>(n_t, d_Hc.as<int>(), d_cls.as<int>(), d_cls_next.as<int>());
    }
    // the local workspace is dead: its bytes go to the quotient pass
    cudaStreamSynchronize(st);
    d_ws.release(&used_iter);
    // ---- Alg. 2 line 13: quotient (Def. 4), second streaming pass -------------------------------------------------------
    // Three streams: copy_st uploads batch k + 1 while st inserts / emits batch k and down_st returns the rows emitted for
    // batch k - 1 to the host (double buffers on both sides; one host synchronisation per batch, to learn the emitted size).
    if ((rc = hq.init(n0, rp0_edges, opt ? opt->host_workspace : nullptr, opt ? opt->host_workspace_bytes : 0,
                      consume ? const_cast<int*>(col) : nullptr, consume && wt ? const_cast<u32*>(wt) : nullptr, compress)))
      break;
    const int osel = outer & 1;  // offsets of the quotient being written; the graph being read uses the other array
    int64_t* nrp = hq.rp[osel];
    // per batch: the nodes whose row intersects it, and the number of blocks whose representative row is complete after it
    std::vector<int64_t> na(nb), nz(nb), done_nodes(nb), done_blocks(nb);
    for (int k = 0; k < nb; ++k) {
      const int64_t c0 = cuts[k], c1 = cuts[k + 1];
      na[k] = std::max<int64_t>(0, (std::upper_bound(rp, rp + n_t + 1, c0) - rp) - 1);
      nz[k] = c1 > c0 ? std::min<int64_t>(n_t, std::upper_bound(rp, rp + n_t + 1, c1 - 1) - rp) : na[k];
      done_nodes[k] = k == nb - 1 ? n_t : (std::upper_bound(rp + 1, rp + n_t + 1, c1) - (rp + 1));  // rp[i + 1] <= c1
      if (have_next) done_nodes[k] = node_cuts[k + 1];  // inherited batches: exactly their node range
    }
    WL_ALLOC(d_query, sizeof(int64_t) * (size_t)nb + sizeof(u64) * (size_t)(nb + 1));
    if (rc) break;
    {
      // blocks whose first node lies before done_nodes[k]: one pass over the representative flags
      u64* d_counts = (u64*)(d_query.as<int64_t>() + nb);
      std::vector<u64> h_counts(nb + 1);
      cudaMemcpyAsync(d_query.p, done_nodes.data(), sizeof(int64_t) * (size_t)nb, cudaMemcpyHostToDevice, st);
      cudaMemsetAsync(d_counts, 0, sizeof(u64) * (size_t)(nb + 1), st);
      ++g_launches; count_reps_kernel<<<blocks_for(n_t, 256), 256, 0, st>>>(n_t, d_isrep.as<unsigned char>(), d_query.as<int64_t>(), nb, d_counts);
      cudaMemcpyAsync(h_counts.data(), d_counts, sizeof(u64) * (size_t)(nb + 1), cudaMemcpyDeviceToHost, st);
      rc = check_cuda(cudaStreamSynchronize(st));
      if (rc) break;
      int64_t run = 0;
      for (int k = 0; k < nb; ++k) {
        run += (int64_t)h_counts[k];
        done_blocks[k] = run;
      }
    }
    int64_t longest_cut_row = 0;  // a row cut by a batch border stays in the table until its last piece arrives
    for (int k = 1; k < nb; ++k) {
      const int64_t r = (std::upper_bound(rp, rp + n_t + 1, cuts[k]) - rp) - 1;
      if (r >= 0 && r < n_t && rp[r] < cuts[k]) longest_cut_row = std::max(longest_cut_row, rp[r + 1] - rp[r]);
    }
    const int64_t out_cap = max_edges + longest_cut_row;  // entries one emission can hold
    const u64 qslots = quot_table_slots(out_cap);
    // window of per-block counters: the blocks emitted together, plus the one whose row is still open
    int64_t win = 2;
    {
      int64_t prev = 0;
      for (int k = 0; k < nb; ++k) {
        win = std::max(win, done_blocks[k] - prev + 2);
        prev = std::max(prev, done_blocks[k]);
      }
    }
    WL_ALLOC(d_cnt, sizeof(int) * (size_t)win);
    WL_ALLOC(d_cursor, sizeof(int) * (size_t)win);
    for (int b = 0; b < 2; ++b) WL_ALLOC(d_qrp[b], sizeof(int64_t) * (size_t)(win + 1));
    WL_ALLOC(d_qtab, sizeof(u64) * 2 * qslots);
    // heavy weights (>= 255) one emission may hold on the device before the call falls back to plain uint32 weights
    const u32 ovf_dev_cap = (flags & WL_FLAG_TEST_SMALL_OVERFLOW) ? 2u : (u32)std::min<int64_t>(out_cap, out_cap / 16 + 4096);
    HostQuot::Generation& Gw = hq.gen[outer & 1];                                   // overflow lists of the quotient being written
    for (int b = 0; b < 2; ++b) {
      WL_ALLOC(d_qcol[b], sizeof(int) * (size_t)out_cap);
      WL_ALLOC(d_qwt[b], sizeof(u32) * (size_t)out_cap);
      if (compress) {
        WL_ALLOC(d_qwt8[b], (size_t)out_cap);
        WL_ALLOC(d_qovf[b], sizeof(u64) * (size_t)ovf_dev_cap);
      }
    }
    if (compress && !rc) rc = hq.reserve_generation(outer & 1, (size_t)(rp0_edges / 255 + nb + 1024));
    WL_ALLOC(d_sbsum, sizeof(u64) * (size_t)((win + kScanC - 1) / kScanC + 2));
    WL_ALLOC(d_long, sizeof(int) * (size_t)(max_edges / kQuotLongRow + 2));
    if (debug) std::fprintf(stderr, "[wl_refine_batched] outer %d device memory %.2f GB (cap %.2f GB)%s\n", outer, used_iter / 1073741824.0, device_cap_bytes / 1073741824.0, rc ? " -> WL_ENOMEM" : "");
    if (rc) break;
    cudaMemsetAsync(d_cnt.p, 0, sizeof(int) * (size_t)win, st);
    cudaMemsetAsync(d_cursor.p, 0, sizeof(int) * (size_t)win, st);
    cudaMemsetAsync(d_qtab.p, 0, sizeof(u64) * 2 * qslots, st);
    // inherit: block map and workspace of the next iteration's local refinement (one "piece" per emission)
    std::vector<int64_t> next_edge_cuts(1, 0), next_node_cuts(1, 0);
    int64_t base_next = 0;
    if (inherit) {
      int64_t max_piece_rows = 1, prev = 0;
      for (int k = 0; k < nb; ++k) {
        max_piece_rows = std::max(max_piece_rows, done_blocks[k] - prev);
        prev = std::max(prev, done_blocks[k]);
      }
      WL_ALLOC(d_Hnext, sizeof(int) * (size_t)K);
      WL_ALLOC(d_isrep_next, (size_t)K);
      WL_ALLOC(d_ws2, make_layout(max_piece_rows, out_cap).bytes);
      if (rc) break;
    }
    // Re-cut mode (the default, Alg. 2 as printed), fused: the emitted rows arrive in the row order of the next graph, so they are
    // staged on the device and cut by the same greedy rule (Q13) as they come; every cut is refined at once (as the inherited
    // mode does with its pieces), and the next outer iteration starts at the merge: ONE upload pass per iteration.  Needs every
    // row of the quotient to fit a batch (then every cut falls on a row boundary and no row is ever cut): rows of a quotient
    // are no longer than the longest row of their graph (Def. 4).  Anything unexpected (staging too small, a piece with more
    // rows than prepared for, cuts that differ from the host's greedy cuts at the end) just drops the fusion for this
    // iteration: the next one then uploads its batches for the local refinement as before.
    const int64_t stage_cap_e = max_batch_edges + out_cap;     // entries a staging buffer holds
    const int64_t piece_rows_cap = 2 * max_rows + win + 1024;  // rows of one greedy batch we are prepared for
    const int64_t stage_cap_r = piece_rows_cap + win + 2;
    bool fuse = !inherit && max_row_cur <= max_batch_edges && !(flags & WL_FLAG_NO_FUSED_RECUT);
    size_t fuse_ws_bytes = 0;
    if (fuse) {
      fuse_ws_bytes = make_layout(piece_rows_cap, max_batch_edges).bytes;
      const size_t extra = 5 * (size_t)K + fuse_ws_bytes + 2 * (8 * (size_t)stage_cap_r + 8 * (size_t)stage_cap_e) + 4096;
      if (device_cap_bytes && used_iter + extra > device_cap_bytes) fuse = false;  // optional: never a reason to fail
    }
    if (fuse) {
      WL_ALLOC(d_Hnext, sizeof(int) * (size_t)K);
      WL_ALLOC(d_isrep_next, (size_t)K);
      WL_ALLOC(d_ws2, fuse_ws_bytes);
      for (int b = 0; b < 2; ++b) {
        WL_ALLOC(d_stg_rp[b], sizeof(int64_t) * (size_t)stage_cap_r);
        WL_ALLOC(d_stg_col[b], sizeof(int) * (size_t)stage_cap_e);
        WL_ALLOC(d_stg_wt[b], sizeof(u32) * (size_t)stage_cap_e);
      }
      if (rc) break;
    }
    int64_t* d_cutres = (int64_t*)(d_misc.as<u64>() + 40);  // cut_search_kernel's two results
    int* d_maxrow = (int*)(d_misc.as<u64>() + 44);          // longest row of the quotient being emitted
    cudaMemsetAsync(d_maxrow, 0, sizeof(int), st);
    int stg_cur = 0;
    int64_t stg_row0 = 0, stg_rows = 0, stg_e0 = 0, stg_e1 = 0;  // staged: rows [row0, row0 + rows), entries [e0, e1) of the quotient
    auto upload_quot = [&](int k, int buf) {
      const int64_t c0 = cuts[k], c1 = cuts[k + 1];
      if (c1 > c0) {
        const int* hc = (outer == 1) ? batch_col(k) : hq.col + c0;
        cudaMemcpyAsync(d_col[buf].p, hc, sizeof(int) * (size_t)(c1 - c0), cudaMemcpyHostToDevice, copy_st);
        bytes_h2d += sizeof(int) * (c1 - c0);
        upload_weights(k, buf, c0, c1);
        cudaMemcpyAsync(d_rp[buf].p, rp + na[k], sizeof(int64_t) * (size_t)(nz[k] - na[k] + 1), cudaMemcpyHostToDevice, copy_st);
        bytes_h2d += sizeof(int64_t) * (nz[k] - na[k] + 1);
      }
      cudaEventRecord(ev_up[buf], copy_st);
    };
    // Alg. 2 lines 7-10 of the NEXT iteration on a piece of quotient rows that is still on the device: nodes b_lo .. b_hi of
    // the quotient, whole rows.  Runs on its own stream next to the insertion of the following batch (and next to the copy
    // of the piece to the host); the host waits inside refine_core, which is why it is called after that insertion has
    // been queued.  The piece's blocks get canonical ids inside the piece, so the next block map is canonical as it is.
    struct Piece {
      bool valid;
      int64_t b_lo, b_hi, tot, q_off;
      int ob, index;
      const int64_t* rp_ptr;  // row offsets of the piece (global edge positions q_off .. q_off + tot)
      const int* col_base;    // columns, indexed by global edge position
      const u32* wt_base;     // weights, likewise
      cudaEvent_t ready, done;  // the rows are in place / the piece has been refined
    };
    Piece pending{false, 0, 0, 0, 0, 0, 0, nullptr, nullptr, nullptr, nullptr, nullptr};
    int64_t piece_launches = 0;  // kernels launched by the helper thread (g_launches is per thread)
    auto refine_piece_body = [&](const Piece pending) -> int {
      const int64_t launches0 = g_launches;
      struct Count {
        int64_t& sum;
        int64_t from;
        ~Count() { sum += g_launches - from; }
      } count{piece_launches, launches0};
      const int64_t nr = pending.b_hi - pending.b_lo;
      cudaStreamWaitEvent(side_st, pending.ready, 0);
      if (pending.tot == 0) {  // edgeless nodes only: one block (Eq. 3)
        ++g_launches; one_block_kernel<<<blocks_for(nr, 256), 256, 0, side_st>>>(nr, (int)base_next, d_Hnext.as<int>() + pending.b_lo, d_isrep_next.as<unsigned char>() + pending.b_lo);
        base_next += 1;
        cudaEventRecord(pending.done, side_st);
        return check_cuda(cudaStreamSynchronize(side_st));
      }
      wl_csr lg;
      lg.n = nr;
      lg.m = pending.tot;
      lg.row_ptr = pending.rp_ptr;  // global positions q_off .. q_off + tot
      lg.col_idx = pending.col_base;
      lg.weights = pending.wt_base;
      wl_options lo{};
      lo.flags = (flags & (WL_FLAG_NO_PRUNE | WL_FLAG_EDGE_BALANCED)) | WL_FLAG_NO_VALIDATE;
      lo.max_rounds = opt ? opt->max_rounds : 0;
      lo.ring_bits = opt ? opt->ring_bits : 0;
      lo.stream_id = ((u64)(outer + 1) << 32) | (u64)(u32)pending.index;
      const Layout L2 = make_layout(nr, pending.tot);
      CoreResult cr{};
      int prc = refine_core(&lg, init_host ? d_cls_next.as<int>() + pending.b_lo : nullptr, seed, &lo, /*ranged=*/true, (int)pending.b_lo, (int)pending.b_hi, K, pending.q_off,
                            d_ws2.p, L2.bytes, L2, side_st, &cr);
      if (prc) return prc;
      char* wsb = (char*)d_ws2.p;
      int* first_l = (int*)(wsb + L2.o_tmp);
      launch_canonical(L2, nr, cr.colour, d_Hnext.as<int>() + pending.b_lo, first_l, (int*)(wsb + L2.o_rep), (int*)(wsb + L2.o_bsum),
                       (u64*)(wsb + L2.o_scal) + kScalCanon, side_st, cr.k);
      ++g_launches; merge_canon_kernel<<<blocks_for(nr, 256), 256, 0, side_st>>>(nr, cr.colour, first_l, (int)base_next, d_Hnext.as<int>() + pending.b_lo, d_isrep_next.as<unsigned char>() + pending.b_lo);
      base_next += cr.k;
      edges_streamed += cr.edges_streamed;
      ms_spmv += cr.ms_spmv;
      ms_relabel += cr.ms_relabel;
      ms_spmv_kernel += cr.ms_spmv_kernel;
      spmv_alg_bytes += cr.spmv_alg_bytes;
      spmv_launches += cr.spmv_launches;
      // the emission buffers may be overwritten once this piece is refined (emission + 2 waits on the stream `st`)
      cudaEventRecord(pending.done, side_st);
      return check_cuda(cudaStreamSynchronize(side_st));  // d_ws2 is reused by the next piece
    };
    // joins the piece before (its ids come first, its workspace is reused) and hands the pending one to the helper thread
    auto refine_piece = [&]() -> int {
      const int prc = piece_worker.wait();
      if (prc) return prc;
      if (!pending.valid) return WL_OK;
      const Piece p = pending;
      pending.valid = false;
      piece_worker.submit([&refine_piece_body, p]() { return refine_piece_body(p); });
      return WL_OK;
    };
    int64_t q_off = 0, emitted_blocks = 0;
    int n_emit = 0;
    // compressed weights: the overflow list of an emission goes to the host one synchronisation later, when its length is known
    u32* d_ovf_cnt = (u32*)(d_misc.as<u64>() + 32);  // two counters (by emission parity)
    volatile u64* h_ovf_cnt = hs + kNumScal + 4;      // their host copies
    struct PendingOvf {
      bool valid;
      int ob;
      size_t em_index;
    } pend_ovf{false, 0, 0};
    auto flush_overflow = [&]() -> int {  // call right after a synchronisation of `st`
      if (!pend_ovf.valid) return WL_OK;
      pend_ovf.valid = false;
      const u32 cnt = (u32)h_ovf_cnt[pend_ovf.ob];
      if (cnt > ovf_dev_cap) return kCompressOverflow;
      HostQuot::Emission& e = Gw.em[pend_ovf.em_index];
      if (Gw.used + cnt > Gw.cap) return WL_ECUDA;  // unreachable: at most m / 255 weights reach 255 (L447)
      e.ovf_off = Gw.used;
      e.count = cnt;
      if (cnt) {
        cudaMemcpyAsync(Gw.ovf + Gw.used, d_qovf[pend_ovf.ob].p, sizeof(u64) * cnt, cudaMemcpyDeviceToHost, down_st);
        bytes_d2h += sizeof(u64) * cnt;
        cudaEventRecord(ev_down[pend_ovf.ob], down_st);  // the buffer is free again only after this copy
        Gw.used += cnt;
      }
      return WL_OK;
    };
    auto checkpoint = [&](const char* what, int k) {  // WL_DEBUG: find the launch that faults
      if (!debug) return;
      cudaError_t e = cudaDeviceSynchronize();
      if (e != cudaSuccess) std::fprintf(stderr, "[wl_refine_batched] outer %d batch %d: %s -> %s\n", outer, k, what, cudaGetErrorString(e));
    };
    // fused re-cut: one greedy batch of the quotient, rows [stg_row0, stg_row0 + idx) of what is staged, handed to the helper
    // thread; the rest of the staged rows moves to the other staging buffer (the piece keeps reading this one)
    auto form_piece = [&](int64_t limit, bool take_all) -> int {
      int64_t idx = stg_rows, cut_edge = stg_e1;
      if (!take_all) {
        ++g_launches; cut_search_kernel<<<1, 1, 0, st>>>(d_stg_rp[stg_cur].as<int64_t>(), stg_rows, limit, d_cutres);
        cudaMemcpyAsync(hs + kNumScal + 6, d_cutres, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, st);
        const int src = check_cuda(cudaStreamSynchronize(st));
        if (src) return src;
        idx = (int64_t)hs[kNumScal + 6];
        cut_edge = (int64_t)hs[kNumScal + 7];
      }
      if (idx <= 0 || idx > piece_rows_cap) {  // (a batch without rows cannot happen when every row fits a batch)
        fuse = false;                            // more rows than prepared for: no fusion this time
        return WL_OK;
      }
      const int prc = piece_worker.wait();  // the piece before read the other staging buffer
      if (prc) return prc;
      cudaEventRecord(ev_stage[stg_cur], st);
      pending = Piece{true, stg_row0, stg_row0 + idx, cut_edge - stg_e0, stg_e0, stg_cur, (int)next_node_cuts.size() - 1,
                      d_stg_rp[stg_cur].as<int64_t>(), d_stg_col[stg_cur].as<int>() - stg_e0, d_stg_wt[stg_cur].as<u32>() - stg_e0,
                      ev_stage[stg_cur], ev_staged[stg_cur]};
      next_edge_cuts.push_back(cut_edge);
      next_node_cuts.push_back(stg_row0 + idx);
      const int64_t rem_rows = stg_rows - idx, rem_e = stg_e1 - cut_edge;
      const int other = stg_cur ^ 1;
      cudaMemcpyAsync(d_stg_rp[other].p, d_stg_rp[stg_cur].as<int64_t>() + idx, sizeof(int64_t) * (size_t)(rem_rows + 1), cudaMemcpyDeviceToDevice, st);
      if (rem_e > 0) {
        cudaMemcpyAsync(d_stg_col[other].p, d_stg_col[stg_cur].as<int>() + (cut_edge - stg_e0), sizeof(int) * (size_t)rem_e, cudaMemcpyDeviceToDevice, st);
        cudaMemcpyAsync(d_stg_wt[other].p, d_stg_wt[stg_cur].as<u32>() + (cut_edge - stg_e0), sizeof(u32) * (size_t)rem_e, cudaMemcpyDeviceToDevice, st);
      }
      const int qrc = refine_piece();  // (nothing to join any more: submits)
      stg_row0 += idx;
      stg_rows = rem_rows;
      stg_e0 = cut_edge;
      stg_cur = other;
      return qrc;
    };
    upload_quot(0, 0);
    for (int k = 0; k < nb && !rc; ++k) {
      const int buf = k & 1;
      const int64_t c0 = cuts[k], c1 = cuts[k + 1];
      if (k + 1 < nb) {
        if (k >= 1) cudaStreamWaitEvent(copy_st, ev_ins[buf ^ 1], 0);  // batch k - 1 has been read out of that buffer
        upload_quot(k + 1, buf ^ 1);
      }
      cudaStreamWaitEvent(st, ev_up[buf], 0);
      const int64_t wb = emitted_blocks;  // window base: block wb is index 0 of the counters
      if (c1 > c0 && nz[k] > na[k]) {
        // rows that cross a cut arrive in pieces: the kernel clips every row to [c0, c1)
        launch_quot_insert(na[k], nz[k] - na[k], d_rp[buf].as<int64_t>(), c0, c1, d_col[buf].as<int>() - c0,
                           weighted ? d_wt[buf].as<u32>() - c0 : nullptr, d_Hc.as<int>(), nullptr, d_isrep.as<unsigned char>(),
                           d_qtab.as<u64>(), qslots - 1, d_cnt.as<int>() - wb, d_long.as<int>(), (u32*)(d_misc.as<u64>() + 16), st, c1 - c0);
      }
      cudaEventRecord(ev_ins[buf], st);
      checkpoint("insert", k);
      if (!fuse && (rc = refine_piece())) break;  // the previous emission, next to this insertion
      // a representative row that continues into the next batch is completed there: emit the blocks whose representative
      // row ends at or before c1 and that were not emitted yet
      const int64_t b_lo = emitted_blocks, b_hi = done_blocks[k];
      if (b_hi > b_lo) {
        const int ob = n_emit & 1;
        if (n_emit >= 2) {
          cudaStreamWaitEvent(st, ev_down[ob], 0);  // the rows emitted two emissions ago are on the host ...
          if (inherit) cudaStreamWaitEvent(st, ev_piece[ob], 0);  // ... and refined
        }
        launch_scan32(d_cnt.as<int>(), b_hi - b_lo, q_off, d_qrp[ob].as<int64_t>(), d_sbsum.as<u64>(), d_misc.as<u64>() + 8, st);
        if (!inherit) {  // row lengths of the quotient = the block counters: the longest one decides whether the NEXT pass may fuse
          ++g_launches; max_i32_kernel<<<blocks_for(b_hi - b_lo, 256), 256, 0, st>>>(b_hi - b_lo, d_cnt.as<int>(), d_maxrow);
        }
        cudaMemcpyAsync(hs + kNumScal + 1, d_misc.as<u64>() + 8, sizeof(u64), cudaMemcpyDeviceToHost, st);
        rc = check_cuda(cudaStreamSynchronize(st));
        if (rc) break;
        const int64_t tot = (int64_t)hs[kNumScal + 1];
        if ((rc = flush_overflow())) break;
        if (debug) std::fprintf(stderr, "[wl_refine_batched] outer %d batch %d: rows %lld..%lld blocks %lld..%lld entries %lld at %lld (cap %lld)\n", outer, k, (long long)na[k], (long long)nz[k], (long long)b_lo, (long long)b_hi, (long long)tot, (long long)q_off, (long long)out_cap);
        if (tot > out_cap || q_off + tot > hq.cap_edges || b_hi > hq.cap_nodes) {
          rc = WL_ECUDA;  // unreachable: a quotient has at most the entries and nodes of its graph
          break;
        }
        ++n_emit;
        ++g_launches; quot_emit_kernel<<<blocks_for((int64_t)qslots, 256), 256, 0, st>>>(d_qtab.as<u64>(), qslots, d_qrp[ob].as<int64_t>() - b_lo, q_off, d_cursor.as<int>() - b_lo, d_qcol[ob].as<int>(), d_qwt[ob].as<u32>(), (int)b_lo, (int)b_hi);
        if (compress && tot) {
          cudaMemsetAsync(d_ovf_cnt + ob, 0, sizeof(u32), st);
          ++g_launches; wt_pack_kernel<<<blocks_for(tot, 256), 256, 0, st>>>(tot, d_qwt[ob].as<u32>(), d_qwt8[ob].as<unsigned char>(), d_qovf[ob].as<u64>(), d_ovf_cnt + ob, ovf_dev_cap);
          cudaMemcpyAsync((void*)(h_ovf_cnt + ob), d_ovf_cnt + ob, sizeof(u32), cudaMemcpyDeviceToHost, st);
        }
        cudaEventRecord(ev_emit[ob], st);
        checkpoint("emit", k);
        // the window moves on: the counter of the block whose row is still open becomes index 0
        ++g_launches; window_carry_kernel<<<1, 1, 0, st>>>(d_cnt.as<int>(), b_hi - b_lo, (int*)(d_misc.as<u64>() + 24), 0);
        cudaMemsetAsync(d_cnt.p, 0, sizeof(int) * (size_t)(b_hi - b_lo + 1), st);
        cudaMemsetAsync(d_cursor.p, 0, sizeof(int) * (size_t)(b_hi - b_lo + 1), st);
        ++g_launches; window_carry_kernel<<<1, 1, 0, st>>>(d_cnt.as<int>(), b_hi - b_lo, (int*)(d_misc.as<u64>() + 24), 1);
        cudaStreamWaitEvent(down_st, ev_emit[ob], 0);
        // in place from the second quotient on: q_off + tot <= c1, and everything below c1 has been uploaded already
        if (tot) {
          if (consume) g_input_consumed = true;
          cudaMemcpyAsync(hq.col + q_off, d_qcol[ob].p, sizeof(int) * (size_t)tot, cudaMemcpyDeviceToHost, down_st);
          if (compress) {
            cudaMemcpyAsync(hq.wt8 + q_off, d_qwt8[ob].p, (size_t)tot, cudaMemcpyDeviceToHost, down_st);
            bytes_d2h += (sizeof(int) + 1) * tot;
            Gw.em.push_back(HostQuot::Emission{q_off, q_off + tot, 0, 0});
            pend_ovf = PendingOvf{true, ob, Gw.em.size() - 1};
          } else {
            cudaMemcpyAsync(hq.wt + q_off, d_qwt[ob].p, sizeof(u32) * (size_t)tot, cudaMemcpyDeviceToHost, down_st);
            bytes_d2h += (sizeof(int) + sizeof(u32)) * tot;
          }
        }
        cudaMemcpyAsync(nrp + b_lo, d_qrp[ob].p, sizeof(int64_t) * (size_t)(b_hi - b_lo + 1), cudaMemcpyDeviceToHost, down_st);
        bytes_d2h += sizeof(int64_t) * (b_hi - b_lo + 1);
        cudaEventRecord(ev_down[ob], down_st);
        if (inherit) {  // refined while the next batch is being inserted (refine_piece)
          pending = Piece{true, b_lo, b_hi, tot, q_off, ob, (int)next_node_cuts.size() - 1, d_qrp[ob].as<int64_t>(),
                          d_qcol[ob].as<int>() - q_off, d_qwt[ob].as<u32>() - q_off, ev_emit[ob], ev_piece[ob]};
          next_edge_cuts.push_back(q_off + tot);
          next_node_cuts.push_back(b_hi);
        }
        if (fuse) {  // the emitted rows join the staged ones; every greedy batch that is complete by now is cut off and refined
          const int64_t nrows_e = b_hi - b_lo;
          if (stg_rows + nrows_e + 1 > stage_cap_r || (stg_e1 - stg_e0) + tot > stage_cap_e) {
            fuse = false;
          } else {
            cudaMemcpyAsync(d_stg_rp[stg_cur].as<int64_t>() + stg_rows, d_qrp[ob].p, sizeof(int64_t) * (size_t)(nrows_e + 1), cudaMemcpyDeviceToDevice, st);
            if (tot) {
              cudaMemcpyAsync(d_stg_col[stg_cur].as<int>() + (q_off - stg_e0), d_qcol[ob].p, sizeof(int) * (size_t)tot, cudaMemcpyDeviceToDevice, st);
              cudaMemcpyAsync(d_stg_wt[stg_cur].as<u32>() + (q_off - stg_e0), d_qwt[ob].p, sizeof(u32) * (size_t)tot, cudaMemcpyDeviceToDevice, st);
            }
            stg_rows += nrows_e;
            stg_e1 = q_off + tot;
            while (fuse && !rc && stg_e1 - stg_e0 >= max_batch_edges && b_hi < K) rc = form_piece(stg_e0 + max_batch_edges, false);
            if (rc) break;
          }
        }
        q_off += tot;
        emitted_blocks = b_hi;
      }
    }
    if (fuse && !rc && emitted_blocks == K) {  // everything is staged: the last greedy batches
      while (fuse && !rc && stg_rows > 0) {
        const bool last = stg_e1 - stg_e0 <= max_batch_edges;
        rc = form_piece(stg_e0 + max_batch_edges, last);
      }
    } else if (fuse) {
      fuse = false;
    }
    if (!rc) rc = refine_piece();
    {
      const int prc = piece_worker.wait();  // (also on an error path: nothing of this iteration may outlive it)
      if (!rc) rc = prc;
    }
    g_launches += piece_launches;
    if (!rc) rc = check_cuda(cudaStreamSynchronize(side_st));
    if (!rc) rc = check_cuda(cudaStreamSynchronize(st));
    if (!rc) rc = flush_overflow();
    if (!rc) rc = check_cuda(cudaStreamSynchronize(down_st));
    if (rc) break;
    nrp[(size_t)K] = q_off;
    phase("quotient");
    // ---- next outer iteration on the quotient ---------------------------------------------------------------------------
    rp = nrp;
    n_t = K;
    weighted = true;
    if (init_host) {  // the quotient becomes the current graph
      d_cls.release(&used);
      d_cls.take(d_cls_next);
    }
    std::vector<int64_t> next_cuts;
    if (inherit) {
      next_cuts = next_edge_cuts;
      if (next_cuts.size() == 1) next_cuts.push_back(0);  // no block at all cannot happen (K >= 1); keep one batch
    } else {
      greedy_cuts(n_t, rp, max_batch_edges, next_cuts);
      // the fused cuts are used only if they are exactly the cuts the greedy rule gives on the finished quotient
      if (fuse && (next_cuts != next_edge_cuts || next_node_cuts.back() != K)) fuse = false;
      {
        int h_maxrow = 0;
        cudaMemcpy(&h_maxrow, d_maxrow, sizeof(int), cudaMemcpyDeviceToHost);  // (every stream of the pass is idle here)
        max_row_cur = h_maxrow;
      }
      if (debug) std::fprintf(stderr, "[wl_refine_batched] outer %d: %s, longest row of the quotient %lld\n", outer,
                              fuse ? "local refinement of the next iteration done on the staged rows" : "next iteration uploads its batches for the local refinement", (long long)max_row_cur);
    }
    if ((flags & WL_FLAG_AGGRESSIVE_STOP) && (int64_t)next_cuts.size() - 1 >= nb) {  // L328
      break;
    }
    cuts.swap(next_cuts);
    if (inherit || fuse) {
      node_cuts.swap(next_node_cuts);
      next_base_id = base_next;
      d_Hnext_keep.take(d_Hnext);  // survive this iteration's buffers
      d_isrep_keep.take(d_isrep_next);
      have_next = true;
    }
  }

  if (rc == WL_OK) {
    if (map0_identity) {
      rc = WL_ECUDA;  // unreachable: every iteration composes the map
    } else if (map0_on_host) {  // the result is where it belongs already
      cudaEventRecord(ev_end, st);
      rc = check_cuda(cudaStreamSynchronize(st));
    } else {
      cudaMemcpyAsync(out_colors, d_map0.p, sizeof(int) * (size_t)n0, cudaMemcpyDeviceToHost, st);
      bytes_d2h += sizeof(int) * n0;
      cudaEventRecord(ev_end, st);
      rc = check_cuda(cudaStreamSynchronize(st));
    }
  }
  if (rc == WL_OK && stats) {
    float t = 0;
    cudaEventElapsedTime(&t, ev_begin, ev_end);
    stats->outer_iters = outer;
    stats->last_num_batches = nb_last;
    stats->boundary_nodes = boundary_first;
    stats->num_colors = K_final;
    stats->edges_streamed = edges_streamed;
    stats->bytes_h2d = bytes_h2d;
    stats->bytes_d2h = bytes_d2h;
    stats->ms_total = t;
    stats->ms_spmv = ms_spmv;
    stats->ms_relabel = ms_relabel;
    stats->ms_spmv_kernel = ms_spmv_kernel;
    stats->spmv_alg_bytes = spmv_alg_bytes;
    stats->spmv_launches = spmv_launches;
    stats->kernel_launches = (int32_t)(g_launches - launches_at_entry);
  }
  cleanup();
  if (debug)
    std::fprintf(stderr, "[wl_refine_batched] result copy + clean-up %9.3f ms, whole call %9.3f ms\n", 1e3 * (wall() - t_mark),
                 std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_entry).count());
  if (rc == WL_OK && hit_limit) return WL_EMAXROUNDS;
  return rc;
}

// Rough device budget of batched_run for a batch cap M_b (DESIGN.md §8 "Device budget"): node arrays, two input and two
// output buffers of 8 bytes per edge, the quotient table, the local workspace of a batch with its share of the rows.
static double batched_budget(int64_t n, int64_t m, int64_t mb, size_t cap, bool inherit, bool with_init) {
  double slots = 1024;
  while (slots < 2.0 * (double)mb) slots *= 2;
  const double rows = m > 0 ? (double)n * (double)mb / (double)m + 1 : (double)n;
  // per node: block map + representative flag; the composed map unless it stays on the host; the next block map (inherit)
  // The default mode can refine the next iteration's batches on staged quotient rows (next block map + two staging buffers:
  // one upload pass per iteration).  That is budgeted for only while the extra per-node array is small against the cap: at
  // configs[4] (n = 2^30 under 16 GB) it would take a third of the cap from the batches, M_b would drop fourfold, and the finer
  // batching costs more colours and iterations than the saved uploads buy (measured: 516 batches, 7 iterations, 28.1 s
  // against 136 batches, 6 iterations, 27-28 s).  Without the budget the staging simply does not fit and the pass uploads twice.
  const bool fused = !inherit && 5.0 * (double)n < 0.1 * (double)cap;
  const double per_node = 5.0 + ((size_t)n * 32 > cap ? 0.25 : 4.0) + (inherit ? 4.0 : 0.0) + (fused ? 5.0 : 0.0) +
                          (with_init ? 8.0 : 0.0);  // initial classes of the current graph and of its quotient
  return per_node * (double)n + (fused ? 64.0 : 32.0) * (double)mb + 16.0 * slots + (fused ? 300.0 : 100.0) * rows + (double)(1 << 20);
}

extern "C" {

int wl_refine_batched(int64_t n, int32_t num_batches, const wl_edge_batch* batches, const wl_csr* whole, uint64_t seed,
                      size_t device_cap_bytes, int64_t max_batch_edges, int32_t* out_colors, wl_stats* stats,
                      const wl_options* opt, void* cuda_stream) {
  // compressed quotient weights are tried first; a batch with too many heavy weights for the device-side overflow list makes the
  // call start over with plain uint32 weights (impossible once the input has been consumed: WL_ENOMEM then)
  g_input_consumed = false;
  auto run = [&](int64_t mb) -> int {
    const auto t0 = std::chrono::steady_clock::now();
    struct Trace {
      std::chrono::steady_clock::time_point t0;
      ~Trace() {
        if (debug_enabled())
          std::fprintf(stderr, "[wl_refine_batched] back in the entry point after %9.3f ms\n",
                       std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count());
      }
    } trace{t0};
    int rc = batched_run(n, num_batches, batches, whole, seed, device_cap_bytes, mb, out_colors, stats, opt, cuda_stream, true);
    if (rc == kCompressOverflow) {
      if (g_input_consumed) return WL_ENOMEM;
      rc = batched_run(n, num_batches, batches, whole, seed, device_cap_bytes, mb, out_colors, stats, opt, cuda_stream, false);
    }
    return rc;
  };
  if (max_batch_edges > 0) return run(max_batch_edges);
  // M_b <= 0: derive it from the device cap (BASELINE.json configs[4]: "a device working-set cap forces the batching").
  // The largest M_b whose estimated budget fits 90 % of the cap; an estimate that turns out too low is answered by WL_ENOMEM
  // from the checked allocations, and M_b shrinks until the run fits.
  if (device_cap_bytes == 0 || num_batches != 0 || !whole || n <= 0) return WL_EINVAL;
  const int64_t m = whole->m;
  int64_t mb = m > 0 ? m : 1;
  const bool inh = opt && (opt->flags & WL_FLAG_INHERIT_BATCHES);
  while (mb > 1024 && batched_budget(n, m, mb, device_cap_bytes, inh, opt && opt->batched_init_colors) > 0.9 * (double)device_cap_bytes) mb = (int64_t)((double)mb * 0.8);
  for (int attempt = 0; attempt < 12; ++attempt) {
    const int rc = run(mb);
    if (rc != WL_ENOMEM || mb <= 1024 || g_input_consumed) return rc;  // a consumed input cannot be read a second time
    mb = (int64_t)((double)mb * 0.7);
  }
  return WL_ENOMEM;
}

}  // extern "C"
