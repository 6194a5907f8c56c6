// Host-side declarations shared by the translation units of the CUDA path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/wl_refine.h"
#include "wl_device.cuh"

namespace wl {

constexpr int64_t kMaxNodes = (1ll << 31) - 2;

// device scalar block (u64 each)
enum { kScalNew = 0, kScalErr = 1, kScalCanon = 2, kScalActive = 3, kScalActiveDeg = 4, kScalHub = 5, kNumScal = 16 };

constexpr int64_t kHubThreshold = 8192;  // rows longer than this are cut into chunks (spmv_hub_kernel)

struct Layout {
  int64_t n, m, ntiles, nscan;
  u32 table_mask;
  int64_t hub_cap;
  size_t o_scal, o_colour, o_rep, o_stamp, o_tmp, o_y, o_tile_row, o_bsum, o_table, o_colour16, o_act0, o_act1, o_hub,
      bytes;
};
Layout make_layout(int64_t n, int64_t m);

extern thread_local int g_last_cuda_error;
extern thread_local int64_t g_launches;
int check_cuda(cudaError_t e);
int basic_csr_check(const wl_csr* g);

}  // namespace wl
