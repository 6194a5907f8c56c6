// Host side of the single-batch engine: workspace layout, the round loop of Algorithm 1 and the
// step-level entry points declared in include/wl_refine.h.  Every step of the path runs in the kernels of wl_kernels.cuh.
#include "wl_host.h"

#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "wl_deep.cuh"
#include "wl_kernels.cuh"

namespace wl {

static_assert(kCanonChunk == kScanChunk, "wl_batched.cu sizes the scan scratch with kCanonChunk");
thread_local int g_last_cuda_error = 0;
thread_local int64_t g_launches = 0;



static inline u32 table_slots_for(int64_t n) {
  // power of two >= 2n, at least 1024, at most 2^31 (slot indices share a word with the winner bit)
  u64 s = 1024;
  while (s < 2ull * (u64)n && s < (1ull << 31)) s <<= 1;
  return (u32)(s - 1);  // returned as mask
}

Layout make_layout(int64_t n, int64_t m) {
  Layout L{};
  L.n = n;
  L.m = m;
  L.ntiles = (n + m + kSpmvTile - 1) / kSpmvTile;
  L.table_mask = table_slots_for(n);
  L.nscan = (n + kScanChunk - 1) / kScanChunk;
  size_t off = 0;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off = align_up(off + bytes);
    return o;
  };
  L.o_scal = take(sizeof(u64) * kNumScal);
  L.o_colour = take(sizeof(int) * (size_t)n);
  L.o_rep = take(sizeof(int) * (size_t)n);
  L.o_stamp = take(sizeof(int) * (size_t)n);
  L.o_tmp = take(sizeof(u32) * (size_t)n);
  L.o_y = take(sizeof(u64) * (size_t)n);
  L.o_tile_row = take(sizeof(int) * (size_t)(L.ntiles + 1));
  L.o_table = take(sizeof(Slot) * ((size_t)L.table_mask + 1));
  L.o_colour16 = take(sizeof(unsigned short) * (size_t)n);
  L.o_act0 = take(sizeof(int) * (size_t)n);
  L.o_act1 = take(sizeof(int) * (size_t)n);
  L.hub_cap = m / kHubChunk + m / (kHubThreshold + 1) + 1;
  L.o_hub = take(sizeof(int2) * (size_t)L.hub_cap);
  L.o_chunk_row = take(sizeof(int) * (size_t)(m / kEbSuper + 4));
  L.o_tag64 = take(sizeof(u64) * kTagSlots);
  L.o_tag32 = take(sizeof(u32) * kTagSlots);
  L.o_y2 = take(sizeof(u64) * (size_t)n);
  L.o_bsum = take(sizeof(int) * canon_scratch_ints(n));  // (last: the arrays the gathers read keep their place)
  L.bytes = off;
  return L;
}



DeepLayout make_deep_layout(const Layout& L) {
  DeepLayout D{};
  size_t off = L.bytes;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off = align_up(off + bytes);
    return o;
  };
  const size_t n = (size_t)L.n, m = (size_t)L.m;
  D.o_scal = take(sizeof(u64) * kNumDeep);
  D.o_tp_ptr = take(sizeof(int64_t) * (n + 1));
  D.o_tp_src = take(sizeof(int) * m);
  D.o_size = take(sizeof(int) * n);
  D.o_inherit = take(sizeof(int) * n);
  D.o_mark = take(sizeof(int) * n);
  D.o_slots = take(sizeof(u32) * n);
  for (int b = 0; b < 2; ++b) {  // double-buffered by round parity
    D.o_lcount[b] = take(sizeof(int) * n);
    D.o_leavers[b] = take(sizeof(int) * n);
    D.o_leaver_block[b] = take(sizeof(int) * n);
    D.o_changed[b] = take(sizeof(int) * n);
  }
  D.o_bsum = take(sizeof(u64) * (n / kScan32Chunk + 3));
  D.bytes = off;
  return D;
}

// ---- step launchers -----------------------------------------------------------------------------------------------
void launch_tile_search(const Layout& L, const wl_csr& g, int* tile_row, cudaStream_t st) {
  ++g_launches; tile_search_kernel<<<blocks_for(L.ntiles + 1, 256), 256, 0, st>>>(g.n, g.m, g.row_ptr, L.ntiles, tile_row);
}

// S1+S2 over all rows or an active row list.  merge: the merge-path kernel (all rows; y must be zero before it).
// Otherwise warp-per-row over `rows` (NULL: all) followed by the hub-chunk kernel.  narrow: gather 16-bit colour ids.
struct SpmvArgs {
  const int* rows;       // active row list or NULL
  int64_t nrows;         // rows to process (n when rows == NULL)
  const int* colour;     // int32 colours
  const unsigned short* colour16;  // valid when narrow
  bool narrow;
  const int2* hub_chunks;
  int64_t num_hub_chunks;
  const int* stamp;      // hub activity test (NULL: all hubs)
  int live_stamp;
  bool ranged;           // batched local RSC: targets outside [lo, hi) are implicit singletons
  int lo, hi;
  bool eb = false;       // edge-balanced kernel over ALL rows (rows / hub_chunks ignored)
  bool validate = false; // fold the column range check of S0 into this pass (it must read every column: no row list)
  int* chunk_row = nullptr;
  int64_t e_first = 0;   // row_ptr[0]
  int64_t n_targets = 0;
  u32* err = nullptr;
  const u32* tag32 = nullptr;  // hot-id table (16-bit ids, plain RSC only) or NULL
  u32 idmask = 0;
  u64* ticket = nullptr;       // zeroed device counter of the persistent kernel
  u64 key2 = 0;                // DUAL rows: second key and second sum (finality test of the coming compaction)
  u64* y2 = nullptr;
  bool hubs_only = false;      // the row kernel has been launched piece by piece (ColumnFeed): only the hub chunks are left
  cudaStream_t hub_stream = nullptr;  // not NULL: the hub kernel runs on this stream NEXT TO the row kernel (it fills the row
  cudaEvent_t hub_fork = nullptr, hub_join = nullptr;  // kernel's tail: 4 % of its time on the headline round)
};

// edge-balanced S1+S2 over all rows of g (see spmv_eb_kernel)
template <bool W, typename CT, bool R, bool V>
static void launch_eb3(const wl_csr& g, const SpmvArgs& a, const CT* colour, u64 key, u64* y, cudaStream_t st) {
  const int64_t e_first = a.e_first, e_last = e_first + g.m;
  const int64_t e_anchor = e_first;
  const int64_t nchunks = (e_last - e_anchor + kEbSuper - 1) / kEbSuper;
  ++g_launches; eb_setup_kernel<<<blocks_for(nchunks, 256), 256, 0, st>>>(g.n, g.row_ptr, e_anchor, nchunks, a.chunk_row, y);
  ++g_launches; spmv_eb_kernel<W, CT, R, V><<<blocks_for(nchunks * 32, 256), 256, 0, st>>>(g.n, g.row_ptr, g.col_idx, g.weights, colour, key, y, a.chunk_row, e_anchor, e_first, e_last, a.lo, a.hi, a.n_targets, a.err);
}
template <bool W, typename CT>
static void launch_eb(const wl_csr& g, const SpmvArgs& a, const CT* colour, u64 key, u64* y, cudaStream_t st) {
  if (a.ranged) {
    if (a.validate) launch_eb3<W, CT, true, true>(g, a, colour, key, y, st);
    else launch_eb3<W, CT, true, false>(g, a, colour, key, y, st);
  } else {
    if (a.validate) launch_eb3<W, CT, false, true>(g, a, colour, key, y, st);
    else launch_eb3<W, CT, false, false>(g, a, colour, key, y, st);
  }
}

constexpr int kRowsCta = 64;  // two warps per CTA: a warp stuck on long rows does not hold six finished ones' slots (measured)

// the row kernel through the hot-id table: one persistent CTA per SM (128 KB of shared memory each)
template <bool V>
static void launch_rows_tag(const wl_csr& g, const SpmvArgs& a, u64 key, u64* y, cudaStream_t st) {
  static thread_local bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(spmv_rows32_tag_kernel<false, V>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(u32) * kTagSlots));
    attr_set = true;
  }
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaMemsetAsync(a.ticket, 0, sizeof(u64), st);
  ++g_launches; spmv_rows32_tag_kernel<false, V><<<(unsigned)sms, kTagThreads, sizeof(u32) * kTagSlots, st>>>(a.nrows, a.rows, g.row_ptr, g.col_idx, g.weights, a.colour16, key, y, kHubThreshold, a.n_targets, a.err, a.tag32, a.idmask, a.ticket, kTagRun);
}

template <bool W, typename CT, bool R, bool V>
static void launch_row_hub2(const wl_csr& g, const SpmvArgs& a, const CT* colour, u64 key, u64* y, cudaStream_t st) {
  unsigned grid = blocks_for(a.nrows, kRowsCta);
  // side by side: y of the hub rows is zeroed first, the row kernel leaves those rows alone, the hub kernel is queued on the
  // second stream right behind the row kernel's launch: its CTAs get the SMs the row kernel no longer fills
  const bool beside = a.hub_stream && a.num_hub_chunks > 0 && !a.hubs_only && !(!W && !R && a.tag32 && a.narrow);
  if (beside) {
    ++g_launches; hub_zero_kernel<<<blocks_for(a.num_hub_chunks, 256), 256, 0, st>>>(a.num_hub_chunks, a.hub_chunks, y);
    cudaEventRecord(a.hub_fork, st);
    cudaStreamWaitEvent(a.hub_stream, a.hub_fork, 0);
  }
  const int hub_store = beside ? 0 : 1;
  if (a.hubs_only) {
  } else if (!W && !R && a.tag32 && a.narrow) {
    launch_rows_tag<V>(g, a, key, y, st);
  } else if (!W && !R && !V && a.y2 && sizeof(CT) == 4) {
    ++g_launches; spmv_rows32_kernel<false, int, false, false, true><<<grid, kRowsCta, 0, st>>>(a.nrows, a.rows, g.row_ptr, g.col_idx, g.weights, a.colour, key, y, kHubThreshold, a.lo, a.hi, a.n_targets, a.err, a.key2, a.y2, hub_store);
  } else {
    ++g_launches; spmv_rows32_kernel<W, CT, R, V><<<grid, kRowsCta, 0, st>>>(a.nrows, a.rows, g.row_ptr, g.col_idx, g.weights, colour, key, y, kHubThreshold, a.lo, a.hi, a.n_targets, a.err, 0, nullptr, hub_store);
  }
  if (a.num_hub_chunks > 0) {
    cudaStream_t hs = beside ? a.hub_stream : st;
    ++g_launches; spmv_hub_kernel<W, CT, R, V><<<(unsigned)a.num_hub_chunks, kHubThreads, 0, hs>>>(a.hub_chunks, g.row_ptr, g.col_idx, g.weights, colour, key, y, a.colour, a.stamp, a.live_stamp, a.lo, a.hi, a.n_targets, a.err);
    if (beside) {
      cudaEventRecord(a.hub_join, a.hub_stream);
      cudaStreamWaitEvent(st, a.hub_join, 0);
    }
  }
}
template <bool W, typename CT>
static void launch_row_hub(const wl_csr& g, const SpmvArgs& a, const CT* colour, u64 key, u64* y, cudaStream_t st) {
  if (a.ranged) launch_row_hub2<W, CT, true, false>(g, a, colour, key, y, st);
  else if (a.validate) launch_row_hub2<W, CT, false, true>(g, a, colour, key, y, st);
  else launch_row_hub2<W, CT, false, false>(g, a, colour, key, y, st);
}

void launch_spmv(const Layout& L, const wl_csr& g, const SpmvArgs& a, u64 key, const int* tile_row, u64* y, bool merge,
                 cudaStream_t st) {
  if (g.n == 0 || a.nrows == 0) return;
  if (merge) {
    if (g.weights) {
      ++g_launches; spmv_merge_kernel<true><<<(unsigned)L.ntiles, kSpmvThreads, 0, st>>>(g.n, g.m, g.row_ptr, g.col_idx, g.weights, a.colour, key, tile_row, y);
    } else {
      ++g_launches; spmv_merge_kernel<false><<<(unsigned)L.ntiles, kSpmvThreads, 0, st>>>(g.n, g.m, g.row_ptr, g.col_idx, g.weights, a.colour, key, tile_row, y);
    }
    return;
  }
  if (a.eb) {
    if (g.weights) {
      if (a.narrow) launch_eb<true, unsigned short>(g, a, a.colour16, key, y, st);
      else launch_eb<true, int>(g, a, a.colour, key, y, st);
    } else {
      if (a.narrow) launch_eb<false, unsigned short>(g, a, a.colour16, key, y, st);
      else launch_eb<false, int>(g, a, a.colour, key, y, st);
    }
    return;
  }
  if (g.weights) {
    if (a.narrow) launch_row_hub<true, unsigned short>(g, a, a.colour16, key, y, st);
    else launch_row_hub<true, int>(g, a, a.colour, key, y, st);
  } else {
    if (a.narrow) launch_row_hub<false, unsigned short>(g, a, a.colour16, key, y, st);
    else launch_row_hub<false, int>(g, a, a.colour, key, y, st);
  }
}

// hub chunk list (rows with degree > kHubThreshold); *counter (device u64) must be zero
void launch_hub_collect(const Layout& L, const wl_csr& g, int2* chunks, u64* counter, cudaStream_t st) {
  if (g.n == 0) return;
  ++g_launches; hub_collect_kernel<<<blocks_for(g.n, 256), 256, 0, st>>>(g.n, g.row_ptr, kHubThreshold, chunks, counter);
}

// One relabel step (S3+S4) over `nodes` (NULL: all): scal[kScalK] is the current colour count, scal[kScalNew] must be
// zero; on completion scal[kScalK] has grown by the number of new ids (logged to log[log_slot] if log != NULL), the slots
// [0, table_mask] of the table are empty again and colour16 (may be NULL) mirrors the new ids as 16 bits.
// clean == false: the claimed slots stay (the caller empties them with clean_table once it knows the new colour count).
void launch_relabel(u32 table_mask, int64_t count, const int* nodes, int* colour, unsigned short* colour16, const u64* y,
                    int* rep, int* stamp, int round, Slot* table, u32* slot_of, u64* scal, u64* log, int log_slot,
                    bool clean, cudaStream_t st, int* changed = nullptr, u64* n_changed = nullptr, u64 ymask = ~0ull) {
  if (count > 0) {
    unsigned grid = blocks_for(count, kRelabelThreads);
    ++g_launches; relabel_kernel<<<grid, kRelabelThreads, 0, st>>>(count, nodes, colour, colour16, y, rep, stamp, round, table, table_mask, slot_of, scal + kScalK, scal + kScalNew, changed, n_changed, ymask);
  }
  const unsigned fgrid = clean ? (unsigned)std::max<int64_t>(1, std::min<int64_t>(blocks_for(count, 256), 148 * 8)) : 1u;
  ++g_launches; relabel_finish_kernel<<<fgrid, 256, 0, st>>>(table, slot_of, scal, log, log_slot, clean ? 1 : 0);
}

// Re-empty the slots claimed by the ids [first_id, first_id + count) of a relabel step run with clean == false:
// one scattered 16-byte store per id, or a memset of the slot range when that is cheaper (measured on B200: a scattered
// store costs about as much as 16 slots of memset).
void clean_table(Slot* table, u32 table_mask, const u32* slot_of, int64_t first_id, int64_t count, cudaStream_t st) {
  if (count <= 0) return;
  if (count * 16 >= (int64_t)table_mask + 1) {
    cudaMemsetAsync(table, 0xff, sizeof(Slot) * ((size_t)table_mask + 1), st);
  } else {
    ++g_launches; relabel_clean_kernel<<<blocks_for(count, 256), 256, 0, st>>>(table, slot_of, first_id, count);
  }
}

static u32 round_table_mask(const Layout& L, int64_t n_active) {
  u64 s = 1024;
  while (s < 2ull * (u64)n_active && s < (u64)L.table_mask + 1) s <<= 1;
  return (u32)(s - 1);
}

// canonical ids: uses `first` (int[n], first node per colour) and `cid` (int[n], canonical id per colour) as scratch, bsum =
// canon_scratch_ints(n) ints (chunk sums + one flag bit per node), total -> scal slot.  k > 0: the colour ids are < k (only that
// much of `first` is initialised and meaningful afterwards).
void launch_canonical(const Layout& L, int64_t n, const int* colour, int* out, int* first, int* cid, int* bsum,
                      u64* total, cudaStream_t st, int64_t k) {
  if (n == 0) return;
  const int64_t kk = k > 0 && k < n ? k : n;
  u32* flags = (u32*)(bsum + L.nscan + 1);
  ++g_launches; fill_i32_kernel<<<blocks_for(kk, 256), 256, 0, st>>>(kk, first, kNoNode);
  ++g_launches; first_node_kernel<<<blocks_for(n, 256 * kFirstItems), 256, 0, st>>>(n, colour, first);
  ++g_launches; canon_count_kernel<<<(unsigned)L.nscan, kScanThreads, 0, st>>>(n, colour, first, bsum, flags);
  ++g_launches; scan_bsum_kernel<<<1, 1024, 0, st>>>(L.nscan, bsum, total);
  ++g_launches; canon_rank_kernel<<<(unsigned)L.nscan, kScanThreads, 0, st>>>(n, colour, flags, bsum, cid);
  ++g_launches; canon_apply_kernel<<<(unsigned)L.nscan, kScanThreads, 0, st>>>(n, colour, cid, flags, bsum, out);
}

// WL_DEBUG (per-round trace on stderr) is read once per process, not per call
bool debug_enabled() {
  static const bool on = std::getenv("WL_DEBUG") != nullptr;
  return on;
}

int check_cuda(cudaError_t e) {
  if (e == cudaSuccess) return WL_OK;
  g_last_cuda_error = (int)e;
  return WL_ECUDA;
}

int basic_csr_check(const wl_csr* g) {
  if (!g) return WL_EINVAL;
  if (g->n < 0 || g->m < 0) return WL_EINVAL;
  if (g->n > 0 && !g->row_ptr) return WL_EINVAL;
  if (g->m > 0 && !g->col_idx) return WL_EINVAL;
  if (g->n > kMaxNodes) return WL_ERANGE;
  if (g->n == 0 && g->m != 0) return WL_EINVAL;
  return WL_OK;
}

// pinned host mirror of the device scalars (one per host thread; released when the thread ends: the batched path runs
// refinements on a helper thread of its own per call)
u64* host_scal() {
  // a block goes back to a process-wide list when its thread ends and is handed to the next new thread: the batched path starts
  // a helper thread per call, and cudaHostAlloc / cudaFreeHost cost up to hundreds of milliseconds now and then
  struct Spare {
    std::mutex mu;
    std::vector<u64*> blocks;
  };
  static Spare* spare = new Spare;  // (never destroyed: threads may end after the statics of this library)
  struct Holder {
    u64* p = nullptr;
    ~Holder() {
      if (!p) return;
      std::lock_guard<std::mutex> lock(spare->mu);
      spare->blocks.push_back(p);
    }
  };
  static thread_local Holder h;
  if (!h.p) {
    {
      std::lock_guard<std::mutex> lock(spare->mu);
      if (!spare->blocks.empty()) {
        h.p = spare->blocks.back();
        spare->blocks.pop_back();
      }
    }
    if (!h.p && cudaHostAlloc((void**)&h.p, sizeof(u64) * (kNumScal + 8), cudaHostAllocDefault) != cudaSuccess) h.p = nullptr;
  }
  return h.p;
}

}  // namespace wl

using namespace wl;

extern "C" {

size_t wl_refine_workspace_bytes(int64_t n, int64_t m) {
  if (n < 0 || m < 0 || n > kMaxNodes) return 0;
  return make_layout(n, m).bytes;
}

size_t wl_refine_deep_workspace_bytes(int64_t n, int64_t m) {
  if (n < 0 || m < 0 || n > kMaxNodes) return 0;
  return make_deep_layout(make_layout(n, m)).bytes;
}

uint64_t wl_round_key(uint64_t seed, uint64_t stream_id, uint64_t round) { return round_key(seed, stream_id, round); }
uint64_t wl_weight(uint64_t key, uint64_t color) { return weight_of(key, color); }

}  // extern "C"

namespace wl {

// Side stream of refine_core: the bulk of the table memset runs next to S0 and round 1 when that round needs only a small
// prefix of the table (uniform start: y = outdeg * w(0), at most sqrt(2m) distinct keys).  It is cut in two pieces so that
// a round whose table fits the lower half does not wait for the upper one.
struct AuxStream {
  cudaStream_t s = nullptr;
  cudaEvent_t fork = nullptr, done_a = nullptr, done_b = nullptr, hub_fork = nullptr, hub_join = nullptr;
  u64 slots_a = 0, slots_b = 0;  // slots [0, slots_a) are empty after done_a, [0, slots_b) after done_b
  bool active = false;
  int init() {
    if (cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess) return WL_ECUDA;
    cudaEventCreateWithFlags(&fork, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&done_a, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&done_b, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&hub_fork, cudaEventDisableTiming);
    cudaEventCreateWithFlags(&hub_join, cudaEventDisableTiming);
    return WL_OK;
  }
  Slot* table = nullptr;
  bool b_issued = false;  // the upper piece is only emptied if a round ever needs it (R-MAT: never, half the memset saved)
  // make `st` wait until slots [0, slots) are empty
  void need(cudaStream_t st, u64 slots, u64 prefix) {
    if (!active || slots <= prefix) return;
    if (slots > slots_a && !b_issued) {
      cudaMemsetAsync(table + slots_a, 0xff, sizeof(Slot) * (slots_b - slots_a), s);
      cudaEventRecord(done_b, s);
      b_issued = true;
    }
    cudaStreamWaitEvent(st, slots <= slots_a ? done_a : done_b, 0);
  }
  ~AuxStream() {
    if (s) cudaStreamSynchronize(s);  // the workspace belongs to the caller again once refine_core returns
    if (fork) cudaEventDestroy(fork);
    if (done_a) cudaEventDestroy(done_a);
    if (done_b) cudaEventDestroy(done_b);
    if (hub_fork) cudaEventDestroy(hub_fork);
    if (hub_join) cudaEventDestroy(hub_join);
    if (s) cudaStreamDestroy(s);
  }
};

// Algorithm 1 (L106-L127) on the rows of `g` (local nodes 0..g.n-1).  ranged: batched local RSC, targets outside [lo, hi)
// are implicit singletons and targets inside map to local node j - lo (Eq. 3).  On success the dense (non canonical)
// colours are in the workspace's colour array and *k_out is their number.  Synchronises `st` once per round.
int refine_core(const wl_csr* g, const int32_t* init_colors, uint64_t seed, const wl_options* opt, bool ranged, int lo,
                int hi, int64_t n_targets, int64_t edge_first, void* workspace, size_t workspace_bytes, const Layout& L,
                cudaStream_t st, CoreResult* res, const ColumnFeed* feed) {
  const int64_t n = g->n, m = g->m;
  int rc = WL_OK;
  const auto t_entry = std::chrono::steady_clock::now();  // (WL_DEBUG trace only)
  const uint32_t flags = opt ? opt->flags : 0u;
  const int64_t max_rounds = (opt && opt->max_rounds > 0) ? opt->max_rounds : n + 1;
  const uint64_t stream_id = opt ? opt->stream_id : 0;
  const u64 ymask = ring_mask(opt ? opt->ring_bits : 0);  // Z/2^q (Alg. 1's precision parameter); all ones for q = 64
  u64* hs = host_scal();
  if (!hs) return check_cuda(cudaErrorMemoryAllocation);

  char* ws = (char*)workspace;
  u64* scal = (u64*)(ws + L.o_scal);
  int* colour = (int*)(ws + L.o_colour);
  int* rep = (int*)(ws + L.o_rep);
  int* stamp = (int*)(ws + L.o_stamp);
  u32* slot_of = (u32*)(ws + L.o_tmp);
  u64* y = (u64*)(ws + L.o_y);
  int* tile_row = (int*)(ws + L.o_tile_row);
  int* chunk_row = (int*)(ws + L.o_chunk_row);
  Slot* table = (Slot*)(ws + L.o_table);
  unsigned short* colour16 = (unsigned short*)(ws + L.o_colour16);
  int* act[2] = {(int*)(ws + L.o_act0), (int*)(ws + L.o_act1)};
  int2* hub_chunks = (int2*)(ws + L.o_hub);
  u64* tag64 = (u64*)(ws + L.o_tag64);
  u32* tag32 = (u32*)(ws + L.o_tag32);
  u64* y2 = (u64*)(ws + L.o_y2);
  const int64_t launches_at_entry = g_launches;
  EventPool evp;
  const bool merge = (flags & WL_FLAG_MERGE_KERNEL) != 0 && !ranged;
  const bool prune = !merge && !(flags & WL_FLAG_NO_PRUNE);
  const bool validate = !(flags & WL_FLAG_NO_VALIDATE);

  // ---- S0: setup ---------------------------------------------------------------------------------------------------
  cudaMemsetAsync(scal, 0, sizeof(u64) * kNumScal, st);
  u32* d_err = (u32*)(scal + kScalErr);
  // Round 1 from a uniform start with unit weights is y = outdeg * w(0): no column is read and at most sqrt(2m) + 1
  // distinct keys exist (distinct degrees d_1 < d_2 < ... sum to at most m), so it runs in a small prefix of the table
  // while the side stream empties the rest; one kernel validates the offsets, sets the initial colour, computes that y
  // and collects the hub chunks.  The column range check is folded into the first kernel that reads the columns.
  const bool uniform_start = !init_colors && !g->weights && !ranged && !merge;
  const bool force_eb = (flags & WL_FLAG_EDGE_BALANCED) != 0 && !merge && m > 0;
  constexpr int64_t kSyncRounds = 6;
  // deep-round (worklist) regime, wl_deep.cuh: needs the larger workspace
  const DeepLayout DL = make_deep_layout(L);
  // (wl_refine_host lets the engine allocate that part itself, and only once the loop gets there: kFlagLazyDeep)
  const bool deep_wanted = !(flags & WL_FLAG_NO_DEEP) && !ranged && !merge && !force_eb && m > 0;
  struct LazyDeep {
    char* p = nullptr;
    ~LazyDeep() {
      if (p) cudaFree(p);
    }
  } lazy_deep;
  char* dws = ws;  // base the deep offsets are relative to
  bool deep_ok = deep_wanted && (workspace_bytes >= DL.bytes || (flags & kFlagLazyDeep));
  const int64_t deep_start = (flags & WL_FLAG_DEEP_EARLY) ? 2 : kSyncRounds + 1;
  u64* deep = nullptr;
  int* changed[2] = {nullptr, nullptr};
  auto bind_deep = [&]() {
    deep = (u64*)(dws + DL.o_scal);
    changed[0] = (int*)(dws + DL.o_changed[0]);
    changed[1] = (int*)(dws + DL.o_changed[1]);
  };
  if (workspace_bytes >= DL.bytes) bind_deep();
  bool cols_checked = !validate || m == 0;
  bool dropped_checked = false;  // the rows outside the active list have had their columns range-checked
  // wl_refine_host (ColumnFeed): row_ptr is needed from here on; the columns arrive piece by piece behind it
  bool feed_pending = feed != nullptr && feed->pieces > 0;
  if (feed) cudaStreamWaitEvent(st, feed->rows_ready, 0);
  auto cols_wait_all = [&]() {  // before any launch that may read any column
    if (!feed_pending) return;
    cudaStreamWaitEvent(st, feed->ready[feed->pieces - 1], 0);  // the pieces are copied in order on one stream
    feed_pending = false;
  };
  if (validate && !uniform_start) {
    // the kernels below walk row_ptr: make sure it is well formed first
    ++g_launches; validate_rows_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, g->row_ptr, g->weights, edge_first, edge_first + m, d_err);
    cudaMemcpyAsync(hs + kScalErr, scal + kScalErr, sizeof(u64), cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    const u32 e = (u32)hs[kScalErr];
    if (e & kErrRowPtr) return WL_EINVAL;
    if (e & kErrRowSum) return WL_ERANGE;
  }
  const u64 table_slots = (u64)L.table_mask + 1;
  u64 prefix_slots = table_slots;
  if (uniform_start) {
    u64 keys = 2;
    while (keys * keys < 2ull * (u64)m + 4) keys <<= 1;  // power of two >= sqrt(2m)
    u64 want = std::max<u64>(1024, 4 * keys);
    if (want < prefix_slots) prefix_slots = want;
  }
  const bool overlap = uniform_start && prefix_slots < table_slots && n >= (1 << 16);
  AuxStream aux;
  cudaMemsetAsync(table, 0xff, sizeof(Slot) * (overlap ? prefix_slots : table_slots), st);
  cudaMemsetAsync(stamp, 0xff, sizeof(int) * (size_t)n, st);
  if (overlap) {
    if ((rc = aux.init())) return check_cuda(cudaGetLastError());
    cudaEventRecord(aux.fork, st);
    cudaStreamWaitEvent(aux.s, aux.fork, 0);
    aux.slots_a = std::max<u64>(prefix_slots, table_slots / 2);
    aux.slots_b = table_slots;
    if (aux.slots_a > prefix_slots) cudaMemsetAsync(table + prefix_slots, 0xff, sizeof(Slot) * (aux.slots_a - prefix_slots), aux.s);
    cudaEventRecord(aux.done_a, aux.s);
    aux.table = table;
    aux.active = true;
  }
  // rep[0] = node 0; stamp[0] = 0 marks block 0 as non-singleton; one colour
  cudaMemsetAsync(rep, 0, sizeof(int), st);
  cudaMemsetAsync(stamp, 0, sizeof(int), st);
  hs[kNumScal] = 1;
  cudaMemcpyAsync(scal + kScalK, hs + kNumScal, sizeof(u64), cudaMemcpyHostToDevice, st);
  // hot-id table of the 16-bit rounds (WL_FLAG_TAG_TABLE, wl_kernels.cuh): candidates = nodes of at least 8 times the average
  // out-degree, collected by the round-1 kernel
  u32 idmask = 1;
  while ((int64_t)idmask + 1 < n) idmask = (idmask << 1) | 1u;
  const bool tag_possible = uniform_start && (flags & WL_FLAG_TAG_TABLE) && n <= (1ll << 30) && !force_eb;
  if (tag_possible) cudaMemsetAsync(tag64, 0, sizeof(u64) * kTagSlots, st);
  if (uniform_start) {
    // S0 and round 1 in one pass over row_ptr (round1_uniform_kernel); the loop below only closes the round
    const u64 w0 = weight_of(round_key(seed, stream_id, 1), 0);
    const u32 mask1 = overlap ? (u32)(prefix_slots - 1) : L.table_mask;
    ++g_launches; round1_uniform_kernel<<<blocks_for(n, kRelabelThreads * kR1Sub), kRelabelThreads, 0, st>>>(n, g->row_ptr, edge_first, edge_first + m, w0, colour, colour16, rep, stamp, table, mask1, slot_of, scal + kScalNew, kHubThreshold, hub_chunks, L.hub_cap, scal + kScalHub, act[0], scal + kScalActive, scal + kScalActiveHub, d_err, ymask, tag_possible ? tag64 : nullptr,
                                                                                                  std::max<int64_t>(64, 8 * (m / std::max<int64_t>(n, 1))), idmask);
  } else {
    if (!cols_checked) {
      cols_wait_all();
      ++g_launches; validate_cols_kernel<<<148 * 8, 256, 0, st>>>(n_targets, edge_first, edge_first + m, g->col_idx, d_err);
      cols_checked = true;
    }
    if (merge) launch_tile_search(L, *g, tile_row, st);
    else launch_hub_collect(L, *g, hub_chunks, scal + kScalHub, st);
    // initial partition: colour 0 everywhere; a given init is densified by one relabel step keyed on the label (L94)
    ++g_launches; init_labels_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, init_colors, colour, colour16, y, d_err);
  }
  int64_t k = 1;
  int64_t num_hub_chunks = 0;
  if (!uniform_start) {
    if (init_colors)
      launch_relabel(L.table_mask, n, nullptr, colour, colour16, y, rep, stamp, /*round=*/0, table, slot_of, scal, nullptr, 0, /*clean=*/false, st,
                     nullptr, nullptr, /*ymask=*/~0ull);  // the key is the caller's label, not a ring element
    cudaMemcpyAsync(hs, scal, sizeof(u64) * kNumScal, cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    const u32 e = (u32)hs[kScalErr];
    if (e & kErrCol) return WL_EINVAL;
    if (e & kErrInit) return WL_EINVAL;
    k = (int64_t)hs[kScalK];
    num_hub_chunks = merge ? 0 : (int64_t)hs[kScalHub];
  }
  // slots still claimed by the previous relabel step (emptied before the next one, when the host knows their number)
  int64_t dirty_first = 1, dirty_count = init_colors ? k - 1 : 0;
  u32 dirty_mask = L.table_mask;
  int64_t active_hubs = num_hub_chunks;  // > 0: some hub row may still be in a splittable block

  // ---- S1-S5: rounds -------------------------------------------------------------------------------------------------
  int64_t edges_streamed = 0, spmv_alg_bytes = 0, last_alg_bytes = 0, last_edges = 0;
  int64_t top_alg_bytes = 0, top_edges = 0;
  double ms_spmv = 0, ms_relabel = 0, ms_spmv_kernel = 0, ms_spmv_top = 0, ms_rest_top = 0;
  int64_t rows_top = 0, last_rows = 0;
  int32_t rounds = 0, spmv_launches = 0;
  bool converged = false;
  const bool debug = debug_enabled();
  auto wall_ms = [&]() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_entry).count(); };
  constexpr double list_frac = 0.75;  // an active list pays once a quarter of the rows has left (measured, scale 27)
  const bool no_runahead = (flags & WL_FLAG_SYNC_EVERY_ROUND) != 0;
  const int* cur_list = nullptr;  // NULL: every node is active
  int64_t n_active = n, active_edges = m, pending_new = 0;
  int cur = 0;
  // One refinement round queued on the stream (S1-S4); no host decision inside.
  auto queue_round = [&](int64_t r, bool narrow, bool mirror, bool clean, u64* log, int log_slot, cudaEvent_t ek0,
                         cudaEvent_t ek1, bool list_changed = false, bool dual = false) -> bool {
    const u64 key = round_key(seed, stream_id, (u64)r);
    bool streamed = false;
    u32 mask_r = round_table_mask(L, n_active);
    const bool round1_done = uniform_start && r == 1;  // round1_uniform_kernel did S1-S3 (R2); only S4 is left
    if (round1_done) {
      mask_r = aux.active ? (u32)(prefix_slots - 1) : L.table_mask;  // the slots its keys may have claimed
    } else {
      if (merge) cudaMemsetAsync(y, 0, sizeof(u64) * (size_t)n, st);
      // row kernels over the active list by default; WL_FLAG_EDGE_BALANCED: the edge-balanced kernel over all rows
      const bool eb = force_eb;
      SpmvArgs a{cur_list, n_active, colour, colour16, narrow, hub_chunks, active_hubs > 0 ? num_hub_chunks : 0,
                 cur_list ? stamp : nullptr, (int)r - 1, ranged, lo, hi};
      a.eb = eb;
      if (aux.active && !(flags & WL_FLAG_SYNC_EVERY_ROUND)) {  // (the side stream exists for large uniform starts)
        a.hub_stream = aux.s;
        a.hub_fork = aux.hub_fork;
        a.hub_join = aux.hub_join;
      }
      a.chunk_row = chunk_row;
      a.e_first = edge_first;
      a.n_targets = n_targets;
      a.err = d_err;
      if (dual && !narrow && !eb && !a.validate) {  // second, independent sum for the finality test that follows this round
        a.key2 = round_key(seed, stream_id ^ 0x5ec0dd5ec0dd5ec0ull, (u64)r);
        a.y2 = y2;
      }
      if (tag_possible && narrow && !eb) {
        // the table carries the colours of THIS round: rebuilt from the slot winners (32 K threads)
        ++g_launches; tag_finalize_kernel<<<kTagSlots / 256, 256, 0, st>>>(tag64, colour16, idmask, tag32);
        a.tag32 = tag32;
        a.idmask = idmask;
        a.ticket = scal + kScalRowTicket;
      }
      bool all_rows = eb;
      if (!cols_checked) {  // S0's column range check rides on the first pass over the columns, which then takes every row
        if (merge || ranged) {
          ++g_launches; validate_cols_kernel<<<148 * 8, 256, 0, st>>>(n_targets, edge_first, edge_first + m, g->col_idx, d_err);
        } else {
          a.validate = true;
          a.num_hub_chunks = num_hub_chunks;  // every hub chunk: pruned hub rows are only range-checked
          if (!eb && cur_list && !dropped_checked) {  // cannot happen with the current round order; kept for safety
            a.rows = nullptr, a.nrows = n, a.stamp = nullptr;
            all_rows = true;
          }
        }
        cols_checked = true;
      }
      cudaEventRecord(ek0, st);
      if (feed_pending && !merge && !eb && !ranged && !a.tag32) {
        // the first pass over the columns of a wl_refine_host call: the row kernel takes the rows piece by piece as their
        // columns land (every row of a piece, empty rows cost one lane-step: no list), the hub chunks follow the last piece
        int64_t node0 = 0;
        for (int j = 0; j < feed->pieces; ++j) {
          cudaStreamWaitEvent(st, feed->ready[j], 0);
          const int64_t node1 = feed->node_end[j];
          if (node1 > node0) {
            SpmvArgs aj = a;
            aj.rows = nullptr;
            aj.nrows = node1 - node0;
            aj.num_hub_chunks = 0;
            if (aj.y2) aj.y2 += node0;
            wl_csr gj = *g;
            gj.row_ptr += node0;
            launch_spmv(L, gj, aj, key, tile_row, y + node0, merge, st);
          }
          node0 = node1;
        }
        feed_pending = false;
        if (a.num_hub_chunks > 0) {
          a.hubs_only = true;
          launch_spmv(L, *g, a, key, tile_row, y, merge, st);
        }
      } else {
        cols_wait_all();
        launch_spmv(L, *g, a, key, tile_row, y, merge, st);
      }
      cudaEventRecord(ek1, st);
      const int64_t e_r = all_rows ? m : active_edges, n_r = all_rows ? n : n_active;
      edges_streamed += e_r;
      last_alg_bytes = (int64_t)(4 + (narrow ? 2 : 4) + (g->weights ? 4 : 0)) * e_r + 16 * n_r;
      last_edges = e_r;
      last_rows = n_r;
      spmv_alg_bytes += last_alg_bytes;
      streamed = true;
    }
    aux.need(st, (u64)mask_r + 1, prefix_slots);
    clean_table(table, dirty_mask, slot_of, dirty_first, dirty_count, st);
    dirty_count = 0;
    dirty_mask = mask_r;
    launch_relabel(mask_r, round1_done ? 0 : n_active, cur_list, colour, mirror ? colour16 : nullptr, y, rep, stamp, (int)r, table, slot_of,
                   scal, log, log_slot, clean, st, list_changed ? changed[(r + 1) & 1] : nullptr,
                   list_changed ? deep + kDeepChanged0 + ((r + 1) & 1) : nullptr, ymask);
    return streamed;
  };
  // final_test: also drop the blocks whose neighbourhood can no longer change (R5); k_prev = colours before round r
  auto queue_compaction = [&](int64_t r, bool final_test = false, int64_t k_prev = 0) {
    if (uniform_start && r == 1) {  // round1_uniform_kernel listed every row with an out-edge and counted them
      dropped_checked = true;       // the rows it dropped have no columns
      return;
    }
    cudaMemsetAsync(scal + kScalActive, 0, 2 * sizeof(u64), st);
    cudaMemsetAsync(scal + kScalActiveHub, 0, sizeof(u64), st);
    // while the column range check is pending the rows dropped here are checked here (a row kernel never reads them)
    const bool check = !cols_checked && !merge && !ranged;
    if (check || final_test) cols_wait_all();
    ++g_launches; compact_active_kernel<<<blocks_for(n_active, 256), 256, 0, st>>>(n_active, cur_list, colour, stamp, rep, (int)r, g->row_ptr, kHubThreshold, act[cur], scal + kScalActive, scal + kScalActiveHub, check ? g->col_idx : nullptr, n_targets, d_err, final_test ? g->col_idx : nullptr, (int)k_prev, y2);
    if (check) dropped_checked = true;
  };
  // host side of a compaction whose counters have been read back; returns true when nothing is left to refine
  auto adopt_compaction = [&]() -> bool {
    pending_new = 0;
    n_active = (int64_t)hs[kScalActive];
    active_edges = (int64_t)hs[kScalActiveDeg];
    active_hubs = (int64_t)hs[kScalActiveHub];
    if ((double)n_active < list_frac * (double)n) {
      cur_list = act[cur];
      cur ^= 1;
    } else {  // nearly everything is still active: keep the list-free kernels
      cur_list = nullptr;
      n_active = n;
      active_edges = m;
      active_hubs = num_hub_chunks;
    }
    return n_active == 0;
  };
  auto log_round = [&](int64_t r, int64_t k_new) {
    if (opt && opt->round_colors && r <= opt->round_colors_cap) opt->round_colors[r - 1] = k_new;
  };

  int64_t r = 1;
  bool deep_entered = false;
  int64_t deep_start_cur = deep_start;  // the round at which the worklist regime is (re-)entered
  bool tp_built = false;            // the in-neighbour lists exist (first entry into the worklist regime)
  while (true) {  // plain rounds -> worklist rounds under one key -> one plain confirming round under a fresh key -> ...
  deep_entered = false;
  while (r <= max_rounds && !converged && !deep_entered) {
    // Rounds 1..kSyncRounds: one host synchronisation per round (the host picks kernels from k and the active count).
    // Deep-round regime (S5): up to kRunAhead rounds are queued back to back; the device keeps k, logs it per round,
    // and the host looks at the log once per window.  A round after the fixed point changes nothing, so running past
    // it is harmless; `rounds` and the trajectory stop at the first repeated count exactly as in the per-round mode.
    // the round at which the worklist regime starts is an ordinary round that also lists the nodes it moved; its key
    // stays the key of every later round
    if (deep_ok && r == deep_start_cur && !deep) {  // the deep part of the workspace is allocated now (wl_refine_host)
      if (cudaMalloc((void**)&lazy_deep.p, DL.bytes - L.bytes) == cudaSuccess) {
        dws = lazy_deep.p - L.bytes;
        bind_deep();
      } else {
        cudaGetLastError();
        deep_ok = false;  // no room: every round keeps recomputing every active row
      }
    }
    const bool switch_round = deep_ok && r == deep_start_cur;
    if (switch_round) cudaMemsetAsync(deep, 0, sizeof(u64) * kNumDeep, st);
    if (switch_round && tp_built) {
      // the worklist rounds do not maintain the representatives the plain relabel compares with: any member will do
      ++g_launches; set_rep_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, colour, rep);
    }
    const int64_t k_before = k;
    const bool window = !no_runahead && r > kSyncRounds && !switch_round;
    const int R = window ? (int)std::min<int64_t>(kRunAhead, max_rounds - r + 1) : 1;
    cudaEvent_t e0 = evp.get(2), e2 = evp.get(4);
    cudaEventRecord(e0, st);
    bool streamed[kRunAhead];
    // 16-bit ids: gathered while k <= 65536; the mirror is kept up to date by the relabel kernel as long as that holds
    // (the worklist rounds do not maintain the mirror: after them the 32-bit ids are gathered)
    const bool narrow = !merge && !tp_built && (window ? n <= 65536 : k <= 65536);
    // the finality test (R5) needs the colour count before the round (host-known in the one-round-per-sync regime only), a
    // column check that is over and 32-bit ids (the DUAL rows of the row kernel); it pays when the rows that are left are short
    // (unit weights only: there the members of a block have the same number of entries, so the row-length limit of the
    // test treats them alike and a block leaves as a whole; its representative's y is never read again)
    const bool final_test = !window && !switch_round && !ranged && !g->weights && !(flags & WL_FLAG_NO_FINAL) && r >= 2 &&
                            cols_checked && !narrow && !force_eb && !merge && cur_list != nullptr && active_edges <= 8 * n_active;
    for (int j = 0; j < R; ++j)
      streamed[j] = queue_round(r + j, narrow, narrow, /*clean=*/window, scal + kScalLog, j, evp.get(8 + 2 * j), evp.get(9 + 2 * j), switch_round, final_test);
    const int64_t r_last = r + R - 1;
    // compaction rides behind rounds 1-2 and behind every window; in between it is decided after the round, when the host
    // knows how many colours the round made (below)
    const bool compact_now = prune && !switch_round && (window || r <= 2);
    if (compact_now) queue_compaction(r_last, final_test, k);
    cudaEventRecord(e2, st);
    cudaMemcpyAsync(hs, scal, sizeof(u64) * kNumScal, cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    {
      const u32 e = (u32)hs[kScalErr];  // verdicts of the checks folded into S0 / the first column pass
      if (e & (kErrRowPtr | kErrCol)) return WL_EINVAL;
      if (e & kErrRowSum) return WL_ERANGE;
    }
    if (uniform_start && r == 1) {
      num_hub_chunks = (int64_t)hs[kScalHub];
      active_hubs = num_hub_chunks;
    }
    float t_all = 0, t_spmv = 0;
    cudaEventElapsedTime(&t_all, e0, e2);
    for (int j = 0; j < R; ++j)
      if (streamed[j]) {
        float tc = 0;
        cudaEventElapsedTime(&tc, evp.get(8 + 2 * j), evp.get(9 + 2 * j));
        t_spmv += tc;
        ++spmv_launches;
        if (R == 1 && tc > ms_spmv_top) {  // (per-round bytes are only kept in the one-round-per-sync regime)
          ms_spmv_top = tc;
          top_alg_bytes = last_alg_bytes;
          top_edges = last_edges;
          ms_rest_top = t_all - tc;
          rows_top = last_rows;
        }
      }
    ms_spmv_kernel += t_spmv;
    ms_spmv += t_spmv;
    ms_relabel += t_all - t_spmv;
    for (int j = 0; j < R && !converged; ++j) {
      const int64_t k_new = (int64_t)hs[kScalLog + j];
      rounds = (int32_t)(r + j);
      log_round(r + j, k_new);
      if (debug)
        std::fprintf(stderr, "[wl_refine] round %lld: k %lld -> %lld, rows %lld, edges %lld%s\n", (long long)(r + j),
                     (long long)k, (long long)k_new, (long long)n_active, (long long)active_edges,
                     window ? " (queued)" : "");
      if (k_new == k) converged = true;  // the partition did not change (Q1, Q2): fixed point
      if (!window) {
        dirty_first = k;
        dirty_count = k_new - k;
      }
      pending_new += k_new - k;
      k = k_new;
    }
    if (debug) std::fprintf(stderr, "[wl_refine]   %d round(s): spmv %.3f ms, rest %.3f ms; host clock %.3f ms since the rounds began\n", R, t_spmv, t_all - t_spmv, wall_ms());
    r += R;
    if (converged) break;
    if (switch_round) {
      deep_entered = true;
      break;
    }
    bool late_compact = false;
    if (!compact_now && prune && !window && pending_new * 16 >= n_active) {
      queue_compaction(r_last, final_test, k_before);
      cudaMemcpyAsync(hs, scal, sizeof(u64) * kNumScal, cudaMemcpyDeviceToHost, st);
      rc = check_cuda(cudaStreamSynchronize(st));
      if (rc) return rc;
      late_compact = true;
    }
    if ((compact_now || late_compact) && adopt_compaction()) {
      // every block is a singleton (or can never split again): the next round cannot change anything and only
      // confirms (same trajectory as the un-pruned algorithm)
      if (r <= max_rounds) {
        rounds = (int32_t)r;
        log_round(r, k);
        converged = true;
      }
      break;
    }
  }
  // ---- S5, deep-round regime (wl_deep.cuh): only the rows with a changed out-neighbour are recomputed ---------------------
  if (!(deep_entered && !converged && r <= max_rounds)) break;
  {
    const u64 key = round_key(seed, stream_id, (u64)deep_start_cur);  // the key of the switch round, kept until the fixed point
    int64_t* tp_ptr = (int64_t*)(dws + DL.o_tp_ptr);
    int* tp_src = (int*)(dws + DL.o_tp_src);
    int* size = (int*)(dws + DL.o_size);
    int* inherit = (int*)(dws + DL.o_inherit);
    int* mark = (int*)(dws + DL.o_mark);
    int* lcount[2] = {(int*)(dws + DL.o_lcount[0]), (int*)(dws + DL.o_lcount[1])};
    int* leavers[2] = {(int*)(dws + DL.o_leavers[0]), (int*)(dws + DL.o_leavers[1])};
    int* leaver_block[2] = {(int*)(dws + DL.o_leaver_block[0]), (int*)(dws + DL.o_leaver_block[1])};
    u32* slots = (u32*)(dws + DL.o_slots);
    u64* bsum = (u64*)(dws + DL.o_bsum);
    cudaEvent_t d0 = evp.get(2), d1 = evp.get(4);
    cudaEventRecord(d0, st);
    // the table is empty between deep rounds; every slot may be used
    clean_table(table, dirty_mask, slot_of, dirty_first, dirty_count, st);
    dirty_count = 0;
    aux.need(st, table_slots, prefix_slots);
    cudaMemsetAsync(size, 0, sizeof(int) * (size_t)n, st);
    cols_wait_all();
    if (!tp_built) {
      // in-neighbour lists: in-degrees -> offsets -> fill (the in-degree array counts down to zero and becomes `mark`)
      cudaMemsetAsync(mark, 0, sizeof(int) * (size_t)n, st);
      cudaMemsetAsync(lcount[0], 0, sizeof(int) * (size_t)n, st);
      cudaMemsetAsync(lcount[1], 0, sizeof(int) * (size_t)n, st);
      cudaMemsetAsync(inherit, 0, sizeof(int) * (size_t)n, st);
      ++g_launches; deep_indegree_kernel<<<148 * 8, 256, 0, st>>>(m, g->col_idx + edge_first, mark);
      launch_scan32(mark, n, 0, tp_ptr, bsum, bsum + (n / kScan32Chunk + 2), st);
      ++g_launches; deep_fill_kernel<<<blocks_for(n * 32, 256), 256, 0, st>>>(n, g->row_ptr, g->col_idx, tp_ptr, mark, tp_src);
      tp_built = true;  // (on a re-entry mark / inherit hold stamps of earlier rounds and the leaver counts are zero again)
    }
    ++g_launches; deep_sizes_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, colour, size);
    constexpr unsigned kDeepGrid = 148 * 4, kDeepFinGrid = 148;
    auto front = [&](const DeepFinishArgs& fin, int do_front, int round) {
      const int in = round & 1;
      const unsigned grid = fin.fin_ctas + (do_front ? kDeepGrid : 0);
      ++g_launches;
      if (g->weights)
        deep_front_kernel<true><<<grid, 256, 0, st>>>(fin, do_front, changed[in], deep + kDeepChanged0 + in, tp_ptr, tp_src, mark, round, g->row_ptr, g->col_idx, g->weights, colour, key, y, size, lcount[in], leavers[in], leaver_block[in], deep + kDeepLeavers0 + in, table, slots, deep, scal, ymask);
      else
        deep_front_kernel<false><<<grid, 256, 0, st>>>(fin, do_front, changed[in], deep + kDeepChanged0 + in, tp_ptr, tp_src, mark, round, g->row_ptr, g->col_idx, g->weights, colour, key, y, size, lcount[in], leavers[in], leaver_block[in], deep + kDeepLeavers0 + in, table, slots, deep, scal, ymask);
    };
    // the bookkeeping that closes `round` (rides in the launch that opens the next round, or alone at the end of a window)
    auto closing = [&](int round, int log_slot) {
      const int in = round & 1;
      DeepFinishArgs f{kDeepFinGrid, leavers[in], leaver_block[in], lcount[in], kDeepLeavers0 + in, kDeepChanged0 + in, log_slot,
                       scal + kScalLog};
      return f;
    };
    // The worklist rounds stop at the fixed point UNDER THIS KEY; a pair that collides under it would stay merged for good.
    // The confirming round of Algorithm 1 is therefore run as a plain round with a fresh key over every active row (the loop
    // above, as a new switch round): if it changes nothing the paper's terminal argument applies as it stands (L408-L414), else
    // the worklist rounds go on under the new key.
    bool fixed_point = false;
    // Launch shape of a window: two kernels per round over the whole GPU (default), or ONE launch by one thread-block cluster that
    // runs all rounds of the window with cluster barriers between the phases (deep_cluster_kernel, WL_FLAG_DEEP_CLUSTER: measured
    // and not the default: a round is two dependent chains of about ten L2 accesses whatever separates them, and eight SMs are too
    // few for the 26 k leavers per round of the 2048^2 grid: 75 us per round against 21, 17 against 10.5 on its last, small rounds;
    // profiles/r2b_deep_cluster.md).
    bool cluster_ok = (flags & WL_FLAG_DEEP_CLUSTER) != 0 && !no_runahead;
    double us_round[2] = {-1.0, -1.0};  // [0] two kernels per round, [1] cluster (WL_DEBUG trace)
    int64_t frontier = -1;
    while (r <= max_rounds && !fixed_point) {
      const int R = no_runahead ? 1 : (int)std::min<int64_t>(kRunAhead, max_rounds - r + 1);
      int shape = cluster_ok ? 1 : 0;
      cudaMemsetAsync(scal + kScalFrontier, 0, sizeof(u64), st);
      if (shape == 1) {
        DeepClusterArgs ca{};
        for (int b = 0; b < 2; ++b) {
          ca.changed[b] = changed[b];
          ca.lcount[b] = lcount[b];
          ca.leavers[b] = leavers[b];
          ca.leaver_block[b] = leaver_block[b];
        }
        ca.tp_ptr = tp_ptr, ca.tp_src = tp_src, ca.mark = mark, ca.row_ptr = g->row_ptr, ca.col = g->col_idx, ca.wt = g->weights;
        ca.colour = colour, ca.key = key, ca.y = y, ca.size = size, ca.inherit = inherit, ca.table = table;
        ca.table_mask = L.table_mask, ca.slots = slots, ca.deep = deep, ca.scal = scal, ca.ymask = ymask;
        ca.round0 = (int)r, ca.rounds = R;
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(kDeepClusterCtas), cfg.blockDim = dim3(kDeepClusterThreads), cfg.dynamicSmemBytes = 0, cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = kDeepClusterCtas, attr[0].val.clusterDim.y = 1, attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr, cfg.numAttrs = 1;
        const cudaError_t le = g->weights ? cudaLaunchKernelEx(&cfg, deep_cluster_kernel<true>, ca)
                                          : cudaLaunchKernelEx(&cfg, deep_cluster_kernel<false>, ca);
        if (le != cudaSuccess) {  // no room for the cluster on this device: the two-kernel shape always works
          cudaGetLastError();
          cluster_ok = false;
          shape = 0;
        } else {
          ++g_launches;
        }
      }
      if (shape == 0) {
        for (int j = 0; j < R; ++j) {
          const int round = (int)(r + j), in = round & 1, out = (round + 1) & 1;
          front(j == 0 ? DeepFinishArgs{0, nullptr, nullptr, nullptr, 0, 0, 0, nullptr} : closing(round - 1, j - 1), 1, round);
          ++g_launches; deep_relabel_kernel<<<kDeepGrid, 256, 0, st>>>(leavers[in], leaver_block[in], deep + kDeepLeavers0 + in, colour, y, size, lcount[in], inherit, round, table, L.table_mask, slots, deep + kDeepSlots, scal + kScalK, deep + kDeepNew, changed[out], deep + kDeepChanged0 + out, ymask);
        }
        front(closing((int)(r + R - 1), R - 1), 0, (int)(r + R));
      }
      cudaEventRecord(d1, st);
      cudaMemcpyAsync(hs, scal, sizeof(u64) * kNumScal, cudaMemcpyDeviceToHost, st);
      rc = check_cuda(cudaStreamSynchronize(st));
      if (rc) return rc;
      float t_win = 0;
      cudaEventElapsedTime(&t_win, d0, d1);
      ms_relabel += t_win;
      cudaEventRecord(d0, st);
      frontier = (int64_t)hs[kScalFrontier];
      us_round[shape] = 1e3 * (double)t_win / R;
      if (debug)
        std::fprintf(stderr, "[wl_refine]   worklist window of %d rounds, %s: %.1f us per round, largest |L| %lld\n", R,
                     shape ? "one cluster launch" : "two kernels per round", us_round[shape], (long long)frontier);
      int done = R;
      for (int j = 0; j < R; ++j) {
        const int64_t k_new = (int64_t)hs[kScalLog + j];
        if (k_new == k) {  // nothing moved in round r + j: that round is re-run as the plain confirming round
          fixed_point = true;
          done = j;
          break;
        }
        rounds = (int32_t)(r + j);
        log_round(r + j, k_new);
        if (debug)
          std::fprintf(stderr, "[wl_refine] round %lld: k %lld -> %lld (worklist)\n", (long long)(r + j), (long long)k, (long long)k_new);
          k = k_new;
      }
      r += done;
    }
    deep_start_cur = r;
  }
  }  // while (true)
  cols_wait_all();  // (a call that never read a column still has to see the uploads finished before its buffers go)
  if (!cols_checked) {  // no round read a column (everything was settled by the degrees): check them now
    ++g_launches; validate_cols_kernel<<<148 * 8, 256, 0, st>>>(n_targets, edge_first, edge_first + m, g->col_idx, d_err);
    cudaMemcpyAsync(hs + kScalErr, scal + kScalErr, sizeof(u64), cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    if ((u32)hs[kScalErr] & kErrCol) return WL_EINVAL;
  }
  res->k = k;
  res->rounds = rounds;
  res->edges_streamed = edges_streamed;
  res->spmv_alg_bytes = spmv_alg_bytes;
  res->ms_spmv = ms_spmv;
  res->ms_relabel = ms_relabel;
  res->ms_spmv_kernel = ms_spmv_kernel;
  res->spmv_launches = spmv_launches;
  res->ms_spmv_top = ms_spmv_top;
  res->spmv_top_alg_bytes = top_alg_bytes;
  res->spmv_top_edges = top_edges;
  res->ms_rest_top = ms_rest_top;
  res->rows_top = rows_top;
  res->kernel_launches = (int32_t)(g_launches - launches_at_entry);
  res->colour = colour;
  return converged ? WL_OK : WL_EMAXROUNDS;
}

}  // namespace wl

extern "C" {

// wl_refine with an optional column feed (wl_refine_host uploads the columns while the first rounds run)
static int refine_device(const wl_csr* g, const int32_t* init_colors, uint64_t seed, int32_t* out_colors, wl_stats* stats,
                         const wl_options* opt, void* workspace, size_t workspace_bytes, void* cuda_stream,
                         const wl::ColumnFeed* feed) {
  int rc = basic_csr_check(g);
  if (rc) return rc;
  const int64_t n = g->n, m = g->m;
  if (stats) std::memset(stats, 0, sizeof(*stats));
  if (n == 0) return WL_OK;
  if (!out_colors || !workspace) return WL_EINVAL;
  const Layout L = make_layout(n, m);
  if (workspace_bytes < L.bytes) return WL_ENOMEM;
  if ((uintptr_t)workspace % 256) return WL_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const uint32_t flags = opt ? opt->flags : 0u;
  const int64_t launches_at_entry = g_launches;
  EventPool evp;
  cudaEvent_t ev_begin = evp.get(0), ev_end = evp.get(1);
  cudaEventRecord(ev_begin, st);
  CoreResult cr{};
  const int core_rc = refine_core(g, init_colors, seed, opt, /*ranged=*/false, 0, 0, n, /*edge_first=*/0, workspace, workspace_bytes, L, st, &cr, feed);
  if (core_rc != WL_OK && core_rc != WL_EMAXROUNDS) return core_rc;
  char* ws = (char*)workspace;
  cudaEvent_t ev_s6 = evp.get(2);
  cudaEventRecord(ev_s6, st);
  // ---- S6: canonical ids ---------------------------------------------------------------------------------------------
  if (flags & WL_FLAG_NO_CANONICAL) {
    cudaMemcpyAsync(out_colors, cr.colour, sizeof(int) * (size_t)n, cudaMemcpyDeviceToDevice, st);
  } else {
    // scratch: tmp -> first node per colour, rep -> canonical id per colour (both dead now)
    launch_canonical(L, n, cr.colour, out_colors, (int*)(ws + L.o_tmp), (int*)(ws + L.o_rep), (int*)(ws + L.o_bsum),
                     (u64*)(ws + L.o_scal) + kScalCanon, st, cr.k);
  }
  cudaEventRecord(ev_end, st);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  rc = check_cuda(cudaGetLastError());
  if (rc) return rc;
  if (stats) {
    float t = 0;
    cudaEventElapsedTime(&t, ev_begin, ev_end);
    if (debug_enabled()) {
      float t6 = 0;
      cudaEventElapsedTime(&t6, ev_s6, ev_end);
      std::fprintf(stderr, "[wl_refine] total %.3f ms on the stream, of which S6 %.3f ms\n", t, t6);
    }
    stats->rounds = cr.rounds;
    stats->num_colors = cr.k;
    stats->edges_streamed = cr.edges_streamed;
    stats->ms_total = t;
    stats->ms_spmv = cr.ms_spmv;
    stats->ms_relabel = cr.ms_relabel;
    stats->ms_spmv_kernel = cr.ms_spmv_kernel;
    stats->spmv_launches = cr.spmv_launches;
    stats->spmv_alg_bytes = cr.spmv_alg_bytes;
    stats->ms_spmv_top = cr.ms_spmv_top;
    stats->spmv_top_alg_bytes = cr.spmv_top_alg_bytes;
    stats->spmv_top_edges = cr.spmv_top_edges;
    stats->ms_rest_top = cr.ms_rest_top;
    stats->rows_top = cr.rows_top;
    stats->kernel_launches = (int32_t)(g_launches - launches_at_entry);
  }
  return core_rc;
}

int wl_refine(const wl_csr* g, const int32_t* init_colors, uint64_t seed, int32_t* out_colors, wl_stats* stats,
              const wl_options* opt, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  return refine_device(g, init_colors, seed, out_colors, stats, opt, workspace, workspace_bytes, cuda_stream, nullptr);
}

// device arena of one wl_refine_host call
struct HostArena {
  size_t o_rp, o_col, o_wt, o_init, o_out, o_ws, bytes;
};
static HostArena host_arena(int64_t n, int64_t m, bool weighted, bool with_init) {
  HostArena A{};
  size_t off = 0;
  auto take = [&](size_t b) {
    size_t o = off;
    off = align_up(off + b);
    return o;
  };
  A.o_rp = take(sizeof(int64_t) * (size_t)(n + 1));
  A.o_col = take(sizeof(int) * (size_t)m);
  A.o_wt = take(weighted ? sizeof(u32) * (size_t)m : 0);
  A.o_init = take(with_init ? sizeof(int) * (size_t)n : 0);
  A.o_out = take(sizeof(int) * (size_t)n);
  A.o_ws = take(wl_refine_workspace_bytes(n, m));
  A.bytes = off;
  return A;
}
size_t wl_refine_host_device_bytes(int64_t n, int64_t m, int weighted, int with_init) {
  if (n < 0 || m < 0) return 0;
  return host_arena(n, m, weighted != 0, with_init != 0).bytes;
}

int wl_refine_host(const wl_csr* g, const int32_t* init_colors, uint64_t seed, int32_t* out_colors, wl_stats* stats,
                   const wl_options* opt, void* cuda_stream) {
  int rc = basic_csr_check(g);
  if (rc) return rc;
  if (stats) std::memset(stats, 0, sizeof(*stats));
  const int64_t n = g->n, m = g->m;
  if (n == 0) return WL_OK;
  if (!out_colors) return WL_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t wsb = wl_refine_workspace_bytes(n, m);  // the deep-round part is allocated by the engine if the loop gets there
  char* d_all = nullptr;
  const HostArena A = host_arena(n, m, g->weights != nullptr, init_colors != nullptr);
  const size_t o_rp = A.o_rp, o_col = A.o_col, o_wt = A.o_wt, o_init = A.o_init, o_out = A.o_out, o_ws = A.o_ws, off = A.bytes;
  const auto t_host0 = std::chrono::steady_clock::now();  // (WL_DEBUG trace only)
  auto host_ms = [&]() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t_host0).count(); };
  const bool own_arena = !(opt && opt->device_workspace);
  if (!own_arena) {
    if (opt->device_workspace_bytes < off) return WL_ENOMEM;
    if ((uintptr_t)opt->device_workspace % 256) return WL_EINVAL;
    d_all = (char*)opt->device_workspace;
  } else if (cudaMalloc((void**)&d_all, off) != cudaSuccess) {
    cudaGetLastError();
    return WL_ENOMEM;
  }
  const double t_malloc = host_ms();
  // Uploads run on a stream of their own, in the order the rounds need them: row offsets (+ the initial partition), then the
  // columns (+ weights) in pieces of whole rows.  The compute stream waits piece by piece (ColumnFeed), so S0, round 1 and the
  // first pass over the columns overlap the link; what is left after the last piece lands is the tail of that pass.
  constexpr int kMaxPieces = 32;
  cudaStream_t copy_st = nullptr;
  if (cudaStreamCreateWithFlags(&copy_st, cudaStreamNonBlocking) != cudaSuccess) {
    if (own_arena) cudaFree(d_all);
    return check_cuda(cudaGetLastError());
  }
  cudaEvent_t e0, e1, rows_ready, ready[kMaxPieces];
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  cudaEventCreateWithFlags(&rows_ready, cudaEventDisableTiming);
  const int pieces = (opt && opt->host_pieces > 0) ? std::min<int>(opt->host_pieces, kMaxPieces)
                                                   : (int)std::max<int64_t>(1, std::min<int64_t>(kMaxPieces, m / (64ll << 20)));
  for (int j = 0; j < pieces; ++j) cudaEventCreateWithFlags(&ready[j], cudaEventDisableTiming);
  cudaEventRecord(e0, st);
  cudaStreamWaitEvent(copy_st, e0, 0);  // whatever the caller queued before this call may still own nothing here, but keep order
  int64_t h2d = 0;
  cudaMemcpyAsync(d_all + o_rp, g->row_ptr, sizeof(int64_t) * (size_t)(n + 1), cudaMemcpyHostToDevice, copy_st);
  h2d += sizeof(int64_t) * (n + 1);
  if (init_colors) {
    cudaMemcpyAsync(d_all + o_init, init_colors, sizeof(int) * (size_t)n, cudaMemcpyHostToDevice, copy_st);
    h2d += sizeof(int) * n;
  }
  cudaEventRecord(rows_ready, copy_st);
  int64_t node_end[kMaxPieces];
  {
    // piece borders on row boundaries, read from the caller's offsets (still unvalidated: clamped and kept monotone, so the
    // copies stay inside the arrays whatever the offsets say; S0 on the device rejects a malformed row_ptr before any column
    // is used)
    int64_t node0 = 0, e_prev = 0;
    for (int j = 0; j < pieces; ++j) {
      int64_t node1 = n;
      if (j + 1 < pieces) {
        const int64_t target = (int64_t)((__int128)m * (j + 1) / pieces);
        node1 = (std::upper_bound(g->row_ptr, g->row_ptr + n + 1, target) - g->row_ptr) - 1;
        node1 = std::max(node0, std::min(node1, n));
      }
      int64_t e_next = j + 1 < pieces ? g->row_ptr[node1] : m;
      e_next = std::max(e_prev, std::min(e_next, m));
      if (e_next > e_prev) {
        cudaMemcpyAsync(d_all + o_col + sizeof(int) * (size_t)e_prev, g->col_idx + e_prev, sizeof(int) * (size_t)(e_next - e_prev),
                        cudaMemcpyHostToDevice, copy_st);
        if (g->weights)
          cudaMemcpyAsync(d_all + o_wt + sizeof(u32) * (size_t)e_prev, g->weights + e_prev, sizeof(u32) * (size_t)(e_next - e_prev),
                          cudaMemcpyHostToDevice, copy_st);
      }
      cudaEventRecord(ready[j], copy_st);
      node_end[j] = node1;
      node0 = node1;
      e_prev = e_next;
    }
    h2d += sizeof(int) * m + (g->weights ? sizeof(u32) * m : 0);
  }
  const ColumnFeed feed{pieces, node_end, ready, rows_ready};
  wl_csr dg = {n, m, (const int64_t*)(d_all + o_rp), (const int*)(d_all + o_col),
               g->weights ? (const u32*)(d_all + o_wt) : nullptr};
  wl_stats inner;
  wl_options hopt{};
  if (opt) hopt = *opt;
  hopt.flags |= kFlagLazyDeep;
  rc = refine_device(&dg, init_colors ? (const int*)(d_all + o_init) : nullptr, seed, (int*)(d_all + o_out), &inner, &hopt,
                     d_all + o_ws, wsb, cuda_stream, &feed);
  if (rc == WL_OK || rc == WL_EMAXROUNDS) {
    cudaMemcpyAsync(out_colors, d_all + o_out, sizeof(int) * (size_t)n, cudaMemcpyDeviceToHost, st);
    cudaEventRecord(e1, st);
    int rc2 = check_cuda(cudaStreamSynchronize(st));
    if (rc2) rc = rc2;
    if (stats) {
      *stats = inner;
      float t = 0;
      cudaEventElapsedTime(&t, e0, e1);
      stats->ms_total = t;
      stats->bytes_h2d = h2d;
      stats->bytes_d2h = sizeof(int) * n;
    }
  }
  cudaStreamSynchronize(copy_st);  // (an early error return leaves uploads in flight: they must be over before the buffers go)
  cudaStreamSynchronize(st);
  const double t_done = host_ms();
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaEventDestroy(rows_ready);
  for (int j = 0; j < pieces; ++j) cudaEventDestroy(ready[j]);
  cudaStreamDestroy(copy_st);
  if (own_arena) cudaFree(d_all);
  if (debug_enabled())
    std::fprintf(stderr, "[wl_refine_host] host clock: cudaMalloc %.3f ms, uploads + rounds + download %.3f ms, cudaFree %.3f ms (%d pieces)\n",
                 t_malloc, t_done - t_malloc, host_ms() - t_done, pieces);
  return rc;
}

int wl_spmv_round(const wl_csr* g, const int32_t* colors, uint64_t key, uint64_t* y, uint32_t flags, void* workspace,
                  size_t workspace_bytes, void* cuda_stream) {
  int rc = basic_csr_check(g);
  if (rc) return rc;
  if (g->n == 0) return WL_OK;
  if (!colors || !y || !workspace) return WL_EINVAL;
  const Layout L = make_layout(g->n, g->m);
  if (workspace_bytes < L.bytes) return WL_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  int* tile_row = (int*)(ws + L.o_tile_row);
  u64* scal = (u64*)(ws + L.o_scal);
  const bool merge = (flags & WL_FLAG_MERGE_KERNEL) != 0;
  const bool narrow = !merge && (flags & WL_FLAG_NARROW_COLORS) != 0;
  SpmvArgs a{nullptr, g->n, colors, (unsigned short*)(ws + L.o_colour16), narrow, (int2*)(ws + L.o_hub), 0, nullptr, 0,
             false, 0, 0};
  if (merge) {
    launch_tile_search(L, *g, tile_row, st);
    cudaMemsetAsync(y, 0, sizeof(u64) * (size_t)g->n, st);
  } else {
    u64* hs = host_scal();
    if (!hs) return WL_ECUDA;
    cudaMemsetAsync(scal, 0, sizeof(u64) * kNumScal, st);
    launch_hub_collect(L, *g, (int2*)(ws + L.o_hub), scal + kScalHub, st);
    cudaMemcpyAsync(hs, scal, sizeof(u64) * kNumScal, cudaMemcpyDeviceToHost, st);
    rc = check_cuda(cudaStreamSynchronize(st));
    if (rc) return rc;
    a.num_hub_chunks = (int64_t)hs[kScalHub];
    if (narrow) { ++g_launches; narrow_kernel<<<blocks_for(g->n, 256), 256, 0, st>>>(g->n, colors, (unsigned short*)(ws + L.o_colour16)); }
    if ((flags & WL_FLAG_EDGE_BALANCED) && g->m > 0) {
      a.eb = true;
      a.chunk_row = (int*)(ws + L.o_chunk_row);
      a.n_targets = g->n;
    }
  }
  launch_spmv(L, *g, a, key, tile_row, (u64*)y, merge, st);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  return check_cuda(cudaGetLastError());
}

int wl_spmv_rows(const wl_csr* g, const int32_t* colors, uint64_t key, const int32_t* rows, int64_t num_rows, uint64_t* y,
                 uint32_t flags, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  int rc = basic_csr_check(g);
  if (rc) return rc;
  if (num_rows < 0 || num_rows > g->n) return WL_EINVAL;
  if (g->n == 0 || num_rows == 0) return WL_OK;
  if (!colors || !y || !workspace || !rows) return WL_EINVAL;
  const Layout L = make_layout(g->n, g->m);
  if (workspace_bytes < L.bytes) return WL_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  u64* scal = (u64*)(ws + L.o_scal);
  u64* hs = host_scal();
  if (!hs) return WL_ECUDA;
  const bool narrow = (flags & WL_FLAG_NARROW_COLORS) != 0;
  int2* chunks = (int2*)(ws + L.o_hub);
  cudaMemsetAsync(scal, 0, sizeof(u64) * kNumScal, st);
  ++g_launches; hub_collect_rows_kernel<<<blocks_for(num_rows, 256), 256, 0, st>>>(num_rows, rows, g->row_ptr, kHubThreshold, chunks, scal + kScalHub);
  cudaMemcpyAsync(hs, scal, sizeof(u64) * kNumScal, cudaMemcpyDeviceToHost, st);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  if (narrow) { ++g_launches; narrow_kernel<<<blocks_for(g->n, 256), 256, 0, st>>>(g->n, colors, (unsigned short*)(ws + L.o_colour16)); }
  SpmvArgs a{rows, num_rows, colors, (unsigned short*)(ws + L.o_colour16), narrow, chunks, (int64_t)hs[kScalHub], nullptr, 0,
             false, 0, 0};
  launch_spmv(L, *g, a, key, nullptr, (u64*)y, /*merge=*/false, st);
  rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  return check_cuda(cudaGetLastError());
}

int wl_relabel(int64_t n, const int32_t* colors, int64_t k, const uint64_t* y, int32_t* new_colors, int64_t* num_colors,
               void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (n < 0 || k < 0 || k > n) return WL_EINVAL;
  if (n > kMaxNodes) return WL_ERANGE;
  if (n == 0) {
    if (num_colors) *num_colors = 0;
    return WL_OK;
  }
  if (!colors || !y || !new_colors || !workspace) return WL_EINVAL;
  const Layout L = make_layout(n, 0);
  if (workspace_bytes < L.bytes) return WL_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  u64* scal = (u64*)(ws + L.o_scal);
  int* rep = (int*)(ws + L.o_rep);
  int* stamp = (int*)(ws + L.o_stamp);
  u32* slot_of = (u32*)(ws + L.o_tmp);
  Slot* table = (Slot*)(ws + L.o_table);
  u64* hs = host_scal();
  if (!hs) return WL_ECUDA;
  cudaMemsetAsync(scal, 0, sizeof(u64) * kNumScal, st);
  cudaMemsetAsync(table, 0xff, sizeof(Slot) * ((size_t)L.table_mask + 1), st);
  cudaMemsetAsync(stamp, 0xff, sizeof(int) * (size_t)n, st);
  if (new_colors != colors)
    cudaMemcpyAsync(new_colors, colors, sizeof(int) * (size_t)n, cudaMemcpyDeviceToDevice, st);
  ++g_launches; set_rep_kernel<<<blocks_for(n, 256), 256, 0, st>>>(n, new_colors, rep);
  const u64 k_u64 = (u64)k;
  cudaMemcpyAsync(scal + kScalK, &k_u64, sizeof(u64), cudaMemcpyHostToDevice, st);
  launch_relabel(L.table_mask, n, nullptr, new_colors, nullptr, (const u64*)y, rep, stamp, 1, table, slot_of, scal, nullptr, 0, /*clean=*/false, st,
                 nullptr, nullptr, /*ymask=*/~0ull);  // the step-level call keys on the exact pairs it is given
  cudaMemcpyAsync(hs, scal, sizeof(u64) * kNumScal, cudaMemcpyDeviceToHost, st);
  int rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  if (num_colors) *num_colors = (int64_t)hs[kScalK];
  return check_cuda(cudaGetLastError());
}

int wl_canonicalize(int64_t n, const int32_t* colors, int32_t* out, int64_t* num_colors, void* workspace,
                    size_t workspace_bytes, void* cuda_stream) {
  if (n < 0) return WL_EINVAL;
  if (n > kMaxNodes) return WL_ERANGE;
  if (n == 0) {
    if (num_colors) *num_colors = 0;
    return WL_OK;
  }
  if (!colors || !out || !workspace) return WL_EINVAL;
  const Layout L = make_layout(n, 0);
  if (workspace_bytes < L.bytes) return WL_ENOMEM;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  char* ws = (char*)workspace;
  u64* scal = (u64*)(ws + L.o_scal);
  u64* hs = host_scal();
  if (!hs) return WL_ECUDA;
  launch_canonical(L, n, colors, out, (int*)(ws + L.o_tmp), (int*)(ws + L.o_rep), (int*)(ws + L.o_bsum),
                   scal + kScalCanon, st);
  cudaMemcpyAsync(hs + kScalCanon, scal + kScalCanon, sizeof(u64), cudaMemcpyDeviceToHost, st);
  int rc = check_cuda(cudaStreamSynchronize(st));
  if (rc) return rc;
  if (num_colors) *num_colors = (int64_t)hs[kScalCanon];
  return check_cuda(cudaGetLastError());
}

const char* wl_strerror(int code) {
  switch (code) {
    case WL_OK: return "ok";
    case WL_EINVAL: return "invalid argument (null pointer, negative size, malformed CSR or negative label)";
    case WL_ERANGE: return "out of range (too many nodes for int32 ids, or a row sum above 2^32)";
    case WL_ENOMEM: return "workspace or device memory cap too small";
    case WL_ECUDA: return "CUDA error (see wl_last_cuda_error)";
    case WL_EMAXROUNDS: return "round / outer-iteration limit reached before the fixed point";
    default: return "unknown wl_status";
  }
}
int wl_last_cuda_error(void) { return g_last_cuda_error; }
int64_t wl_kernel_launches(void) { return g_launches; }
const char* wl_version(void) { return "wl_refine 0.2 (sm_100a)"; }

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// S6 without any allocation: wl_canonicalize_static (include/wl_refine.h).  The scratch of the S6 kernels (first node per
// colour, canonical id per colour, chunk sums + first-node bits, the colour count) lives in ONE file-scope device array of
// fixed size; every GPU that loads the library holds it until the process exits.  In host code `g_static_scratch` is only the
// host-side stand-in of the symbol: the address the kernels get is the one cudaGetSymbolAddress returns for the CURRENT
// device, looked up once per device below.
// ---------------------------------------------------------------------------------------------------------------------
#include <atomic>

namespace wl {

constexpr int64_t kStaticMaxNodes = WL_STATIC_MAX_NODES;
constexpr size_t kStaticFirstOff = 0;                                                        // int[kStaticMaxNodes]
constexpr size_t kStaticCidOff = kStaticFirstOff + sizeof(int) * (size_t)kStaticMaxNodes;    // int[kStaticMaxNodes]
constexpr size_t kStaticScanInts =
    (size_t)((kStaticMaxNodes + kCanonChunk - 1) / kCanonChunk) * (1 + kCanonChunk / 32) + 1;  // = canon_scratch_ints(max)
constexpr size_t kStaticBsumOff = kStaticCidOff + sizeof(int) * (size_t)kStaticMaxNodes;     // int[kStaticScanInts]
constexpr size_t kStaticTotalOff = (kStaticBsumOff + sizeof(int) * kStaticScanInts + 255) / 256 * 256;  // u64
constexpr size_t kStaticBytes = kStaticTotalOff + 256;
static_assert(kStaticCidOff % 256 == 0 && kStaticBsumOff % 256 == 0, "every part of the scratch stays 256-byte aligned");

static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

constexpr int kStaticMaxDevices = 64;
static std::atomic<unsigned char*> g_static_ptr[kStaticMaxDevices];  // device address of g_static_scratch, per device

// device address of the scratch on the current device (nullptr + WL_ECUDA on failure); no allocation, no synchronisation
static int static_scratch(unsigned char** out) {
  int dev = -1;
  int rc = check_cuda(cudaGetDevice(&dev));
  if (rc) return rc;
  if (dev < 0 || dev >= kStaticMaxDevices) return WL_ERANGE;
  unsigned char* p = g_static_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    void* sym = nullptr;
    rc = check_cuda(cudaGetSymbolAddress(&sym, g_static_scratch));
    if (rc) return rc;
    if (!sym) return WL_ECUDA;
    p = (unsigned char*)sym;
    g_static_ptr[dev].store(p, std::memory_order_release);  // two threads racing here store the same address
  }
  *out = p;
  return WL_OK;
}

}  // namespace wl

extern "C" {

int64_t wl_canonicalize_static_max_nodes(void) { return kStaticMaxNodes; }

int wl_canonicalize_static(int64_t n, const int32_t* colors, int32_t* out, int64_t* num_colors, void* cuda_stream) {
  if (n < 0) return WL_EINVAL;
  if (n > kStaticMaxNodes) return WL_ERANGE;  // beyond the fixed scratch: use wl_canonicalize with a workspace
  if (n == 0) return WL_OK;                   // nothing is written, num_colors included (it is device memory)
  if (!colors || !out) return WL_EINVAL;
  unsigned char* s = nullptr;
  int rc = static_scratch(&s);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Layout L{};
  L.nscan = (n + kCanonChunk - 1) / kCanonChunk;  // the only field launch_canonical reads
  u64* total = num_colors ? (u64*)num_colors : (u64*)(s + kStaticTotalOff);
  // every word of the scratch the kernels read is written earlier in this same call (first[] is filled with kNoNode, the
  // chunk sums and bits are stored for every chunk, cid[] is read only at colours whose first node wrote it): nothing
  // of the previous call's contents survives into the result
  launch_canonical(L, n, colors, out, (int*)(s + kStaticFirstOff), (int*)(s + kStaticCidOff), (int*)(s + kStaticBsumOff),
                   total, st);
  return check_cuda(cudaGetLastError());
}

}  // extern "C"
