"""paper_2607_02603_b200 — B200-native randomized 1-WL colour refinement (arxiv/paper_2607_02603).

The product is the C-ABI CUDA library `libwlrefine.so` (include/wl_refine.h); this package is its thin Python binding.
Importing the package does not load the library; the first call does, and raises if it is missing (no CPU fallback).
"""
from .binding import (  # noqa: F401
    EXPORTS, WL_EINVAL, WL_EMAXROUNDS, WL_ENOMEM, WL_ERANGE, WL_ECUDA, WL_FLAG_AGGRESSIVE_STOP, WL_FLAG_NARROW_COLORS, WL_FLAG_NO_CANONICAL,
    WL_FLAG_NO_PRUNE, WL_FLAG_NO_VALIDATE, WL_FLAG_SYNC_EVERY_ROUND, WL_FLAG_MERGE_KERNEL, WL_FLAG_EDGE_BALANCED, WL_FLAG_NO_DEEP, WL_FLAG_DEEP_EARLY, WL_FLAG_DEEP_CLUSTER, WL_FLAG_NO_FUSED_RECUT, WL_FLAG_NO_FINAL, WL_FLAG_INHERIT_BATCHES, WL_FLAG_CONSUME_INPUT, WL_FLAG_TAG_TABLE, WL_FLAG_TEST_SMALL_OVERFLOW, WL_OK, RefineResult, WlError, lib, wl_canonicalize, wl_canonicalize_static, wl_canonicalize_static_max_nodes,
    wl_inner_labels, wl_kernel_launches, wl_quotient, wl_quotient_workspace_bytes, wl_refine, wl_refine_batched, wl_refine_batched_host_bytes, wl_refine_batched_host_bytes_consume, wl_refine_batched_host_overflow_bytes,
    wl_refine_host, wl_refine_inner, wl_quotient_rows, wl_refine_workspace_bytes, wl_refine_deep_workspace_bytes, wl_refine_host_device_bytes, wl_relabel, wl_round_key, wl_spmv_round, wl_spmv_rows, wl_strerror,
    wl_version, wl_weight)
