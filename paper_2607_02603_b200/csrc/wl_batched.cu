// Batched path (Algorithm 2): placeholder translation unit, filled in by the batched engine.
#include "wl_host.h"

extern "C" {

int wl_refine_batched(int64_t, int32_t, const wl_edge_batch*, const wl_csr*, uint64_t, size_t, int64_t, int32_t*,
                      wl_stats*, const wl_options*, void*) {
  return WL_EINVAL;
}
int wl_inner_labels(int64_t, const int64_t*, const int32_t*, const int32_t*, int32_t*, void*) { return WL_EINVAL; }
int wl_quotient(const wl_csr*, const int32_t*, int64_t, int64_t*, int32_t*, uint32_t*, int64_t, int64_t*, void*, size_t,
                void*) {
  return WL_EINVAL;
}
size_t wl_quotient_workspace_bytes(int64_t, int64_t) { return 0; }
}
