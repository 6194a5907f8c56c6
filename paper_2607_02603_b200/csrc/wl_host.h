// Host-side declarations shared by the translation units of the CUDA path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/wl_refine.h"
#include "wl_device.cuh"

namespace wl {

constexpr int64_t kMaxNodes = (1ll << 31) - 2;
constexpr int kNoNode = 0x7fffffff;  // "no node yet" in the atomicMin arrays (first node per colour / block)
static_assert((int64_t)kNoNode > kMaxNodes - 1, "the sentinel must exceed every node index");
constexpr uint32_t kFlagLazyDeep = 1u << 30;  // internal (wl_refine_host): the engine may cudaMalloc the deep-round workspace

constexpr int kRunAhead = kNumScal - kScalLog;  // rounds queued per host synchronisation in the deep-round regime
constexpr int kCanonChunk = 2048;        // nodes per CTA of the canonicalisation scan (== kScanChunk)
constexpr int64_t kHubThreshold = 8192;  // rows longer than this are cut into chunks (spmv_hub_kernel)

struct Layout {
  int64_t n, m, ntiles, nscan;
  u32 table_mask;
  int64_t hub_cap;
  size_t o_scal, o_colour, o_rep, o_stamp, o_tmp, o_y, o_tile_row, o_bsum, o_table, o_colour16, o_act0, o_act1, o_hub,
      o_chunk_row, o_tag64, o_tag32, o_y2, bytes;
};
Layout make_layout(int64_t n, int64_t m);

// extra workspace of the deep-round regime (wl_deep.cuh), laid out after Layout::bytes
struct DeepLayout {
  size_t o_scal, o_tp_ptr, o_tp_src, o_size, o_lcount[2], o_inherit, o_mark, o_leavers[2], o_leaver_block[2], o_slots,
      o_changed[2], o_bsum, bytes;  // bytes = end of the whole workspace (base included)
};
DeepLayout make_deep_layout(const Layout& L);
void launch_scan32(const int* cnt, int64_t n, int64_t base_off, int64_t* out, u64* bsum, u64* total, cudaStream_t st);
constexpr int kScan32Chunk = 2048;  // elements per CTA of launch_scan32

struct CoreResult {
  int64_t k, edges_streamed, spmv_alg_bytes;
  int32_t rounds, spmv_launches, kernel_launches;
  double ms_spmv, ms_relabel, ms_spmv_kernel;
  double ms_spmv_top;                          // longest single S1+S2 launch and what it moved
  int64_t spmv_top_alg_bytes, spmv_top_edges, rows_top;
  double ms_rest_top;
  int* colour;  // dense ids, inside the workspace
};
// wl_refine_host: the column array arrives in pieces while the rounds already run.  row_ptr is complete once `rows_ready` has
// fired; piece j = the rows [node_end[j-1], node_end[j]) with all their entries, on the device once ready[j] has fired
// (node_end[pieces-1] = n).  refine_core makes its stream wait for exactly what the next launch reads.
struct ColumnFeed {
  int pieces;
  const int64_t* node_end;
  const cudaEvent_t* ready;
  cudaEvent_t rows_ready;
};
int refine_core(const wl_csr* g, const int32_t* init_colors, uint64_t seed, const wl_options* opt, bool ranged, int lo,
                int hi, int64_t n_targets, int64_t edge_first, void* workspace, size_t workspace_bytes, const Layout& L,
                cudaStream_t st, CoreResult* res, const ColumnFeed* feed = nullptr);
// ints of scan scratch the canonicalisation needs: chunk sums + one flag bit per node (kCanonChunk / 32 words per chunk)
static inline size_t canon_scratch_ints(int64_t n) {
  const size_t nscan = (size_t)((n + kCanonChunk - 1) / kCanonChunk);
  return nscan + 1 + nscan * (kCanonChunk / 32);
}
void launch_canonical(const Layout& L, int64_t n, const int* colour, int* out, int* first, int* cof, int* bsum, u64* total,
                      cudaStream_t st, int64_t k = -1);
u64* host_scal();
static inline unsigned blocks_for(int64_t count, int threads) { return (unsigned)((count + threads - 1) / threads); }
static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

struct EventPool {
  cudaEvent_t ev[8 + 2 * kRunAhead];
  int n = 0;
  ~EventPool() {
    for (int i = 0; i < n; ++i) cudaEventDestroy(ev[i]);
  }
  cudaEvent_t get(int i) {
    while (n <= i) cudaEventCreate(&ev[n++]);
    return ev[i];
  }
};

extern thread_local int g_last_cuda_error;
extern thread_local int64_t g_launches;
int check_cuda(cudaError_t e);
bool debug_enabled();
int basic_csr_check(const wl_csr* g);

}  // namespace wl
