"""Thin ctypes binding over libwlrefine.so (argument marshalling only: every step runs in the CUDA kernels).

Function names mirror include/wl_refine.h.  torch is used for device memory and streams only.  There is no CPU
fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import List, Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libwlrefine.so")

WL_OK, WL_EINVAL, WL_ERANGE, WL_ENOMEM, WL_ECUDA, WL_EMAXROUNDS = 0, -1, -2, -3, -4, -5
WL_FLAG_NO_VALIDATE, WL_FLAG_NO_PRUNE, WL_FLAG_MERGE_KERNEL, WL_FLAG_AGGRESSIVE_STOP, WL_FLAG_NO_CANONICAL = 1, 2, 4, 8, 16
WL_FLAG_NARROW_COLORS = 32
WL_FLAG_SYNC_EVERY_ROUND = 64
WL_FLAG_EDGE_BALANCED = 128
WL_FLAG_NO_DEEP = 256
WL_FLAG_DEEP_EARLY = 512
WL_FLAG_NO_FINAL = 1024
WL_FLAG_NO_FUSED_RECUT = 2048
WL_FLAG_DEEP_CLUSTER = 32768
WL_FLAG_INHERIT_BATCHES = 4096
WL_FLAG_CONSUME_INPUT = 8192
WL_FLAG_TAG_TABLE = 16384
WL_FLAG_TEST_SMALL_OVERFLOW = 1 << 29

EXPORTS = [
    "wl_refine_workspace_bytes", "wl_refine_deep_workspace_bytes", "wl_refine_host_device_bytes", "wl_refine", "wl_refine_host", "wl_round_key", "wl_weight", "wl_spmv_round",
    "wl_spmv_rows", "wl_relabel", "wl_canonicalize", "wl_canonicalize_static", "wl_canonicalize_static_max_nodes", "wl_refine_batched", "wl_refine_batched_host_bytes", "wl_refine_batched_host_bytes_consume", "wl_refine_batched_host_overflow_bytes", "wl_inner_labels", "wl_quotient",
    "wl_quotient_workspace_bytes", "wl_refine_inner", "wl_refine_inner_workspace_bytes", "wl_quotient_rows",
    "wl_quotient_rows_workspace_bytes", "wl_strerror", "wl_last_cuda_error", "wl_version", "wl_kernel_launches",
]


class WlError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = lib().wl_strerror(code).decode()
        if code == WL_ECUDA:
            msg += f" [cudaError {lib().wl_last_cuda_error()}]"
        super().__init__(f"{where}: {msg} ({code})")


class wl_csr(C.Structure):
    _fields_ = [("n", C.c_int64), ("m", C.c_int64), ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p),
                ("weights", C.c_void_p)]


class wl_options(C.Structure):
    _fields_ = [("flags", C.c_uint32), ("max_rounds", C.c_int32), ("stream_id", C.c_uint64),
                ("round_colors", C.c_void_p), ("round_colors_cap", C.c_int32), ("max_outer_iters", C.c_int32),
                ("host_workspace", C.c_void_p), ("host_workspace_bytes", C.c_size_t), ("ring_bits", C.c_int32),
                ("host_pieces", C.c_int32), ("device_workspace", C.c_void_p), ("device_workspace_bytes", C.c_size_t),
                ("batched_init_colors", C.c_void_p)]


class wl_stats(C.Structure):
    _fields_ = [("rounds", C.c_int32), ("outer_iters", C.c_int32), ("num_colors", C.c_int64),
                ("last_num_batches", C.c_int64), ("boundary_nodes", C.c_int64), ("edges_streamed", C.c_int64),
                ("bytes_h2d", C.c_int64), ("bytes_d2h", C.c_int64), ("ms_total", C.c_double), ("ms_spmv", C.c_double),
                ("ms_relabel", C.c_double), ("spmv_launches", C.c_int32), ("kernel_launches", C.c_int32),
                ("ms_spmv_kernel", C.c_double), ("spmv_alg_bytes", C.c_int64), ("ms_spmv_top", C.c_double),
                ("spmv_top_alg_bytes", C.c_int64), ("spmv_top_edges", C.c_int64), ("ms_rest_top", C.c_double),
                ("rows_top", C.c_int64)]


class wl_edge_batch(C.Structure):
    _fields_ = [("edge_begin", C.c_int64), ("num_edges", C.c_int64), ("row_ptr", C.c_void_p), ("col_idx", C.c_void_p),
                ("weights", C.c_void_p), ("src", C.c_void_p)]


_lib = None


def lib():
    """Load the CUDA library; raises if it has not been built (python paper_2607_02603_b200/build.py)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: build it with `python -m paper_2607_02603_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        vp, i64, i32, u64, u32, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_uint64, C.c_uint32, C.c_size_t
        L.wl_refine_workspace_bytes.restype = sz
        L.wl_refine_workspace_bytes.argtypes = [i64, i64]
        L.wl_refine_deep_workspace_bytes.restype = sz
        L.wl_refine_deep_workspace_bytes.argtypes = [i64, i64]
        L.wl_refine_host_device_bytes.restype = sz
        L.wl_refine_host_device_bytes.argtypes = [i64, i64, C.c_int, C.c_int]
        L.wl_refine.restype = C.c_int
        L.wl_refine.argtypes = [C.POINTER(wl_csr), vp, u64, vp, C.POINTER(wl_stats), C.POINTER(wl_options), vp, sz, vp]
        L.wl_refine_host.restype = C.c_int
        L.wl_refine_host.argtypes = [C.POINTER(wl_csr), vp, u64, vp, C.POINTER(wl_stats), C.POINTER(wl_options), vp]
        L.wl_round_key.restype = u64
        L.wl_round_key.argtypes = [u64, u64, u64]
        L.wl_weight.restype = u64
        L.wl_weight.argtypes = [u64, u64]
        L.wl_spmv_round.restype = C.c_int
        L.wl_spmv_round.argtypes = [C.POINTER(wl_csr), vp, u64, vp, u32, vp, sz, vp]
        L.wl_spmv_rows.restype = C.c_int
        L.wl_spmv_rows.argtypes = [C.POINTER(wl_csr), vp, u64, vp, i64, vp, u32, vp, sz, vp]
        L.wl_relabel.restype = C.c_int
        L.wl_relabel.argtypes = [i64, vp, i64, vp, vp, C.POINTER(i64), vp, sz, vp]
        L.wl_canonicalize.restype = C.c_int
        L.wl_canonicalize.argtypes = [i64, vp, vp, C.POINTER(i64), vp, sz, vp]
        L.wl_canonicalize_static.restype = C.c_int
        L.wl_canonicalize_static.argtypes = [i64, vp, vp, vp, vp]
        L.wl_canonicalize_static_max_nodes.restype = i64
        L.wl_canonicalize_static_max_nodes.argtypes = []
        L.wl_refine_batched.restype = C.c_int
        L.wl_refine_batched.argtypes = [i64, i32, C.POINTER(wl_edge_batch), C.POINTER(wl_csr), u64, sz, i64, vp,
                                        C.POINTER(wl_stats), C.POINTER(wl_options), vp]
        L.wl_refine_batched_host_bytes.restype = sz
        L.wl_refine_batched_host_bytes.argtypes = [i64, i64]
        L.wl_refine_batched_host_bytes_consume.restype = sz
        L.wl_refine_batched_host_bytes_consume.argtypes = [i64, i64, C.c_int]
        L.wl_refine_batched_host_overflow_bytes.restype = sz
        L.wl_refine_batched_host_overflow_bytes.argtypes = [i64]
        L.wl_inner_labels.restype = C.c_int
        L.wl_inner_labels.argtypes = [i64, vp, vp, vp, vp, vp]
        L.wl_quotient.restype = C.c_int
        L.wl_quotient.argtypes = [C.POINTER(wl_csr), vp, i64, vp, vp, vp, i64, C.POINTER(i64), vp, sz, vp]
        L.wl_quotient_workspace_bytes.restype = sz
        L.wl_quotient_workspace_bytes.argtypes = [i64, i64]
        L.wl_refine_inner_workspace_bytes.restype = sz
        L.wl_refine_inner_workspace_bytes.argtypes = [i64, i64]
        L.wl_refine_inner.restype = C.c_int
        L.wl_refine_inner.argtypes = [C.POINTER(wl_csr), i64, i64, u64, vp, vp, C.POINTER(i64), C.POINTER(wl_options), vp, sz, vp]
        L.wl_quotient_rows_workspace_bytes.restype = sz
        L.wl_quotient_rows_workspace_bytes.argtypes = [i64, i64, i64]
        L.wl_quotient_rows.restype = C.c_int
        L.wl_quotient_rows.argtypes = [C.POINTER(wl_csr), i64, vp, vp, i64, i64, vp, vp, vp, i64, C.POINTER(i64), vp, sz, vp]
        L.wl_strerror.restype = C.c_char_p
        L.wl_strerror.argtypes = [C.c_int]
        L.wl_last_cuda_error.restype = C.c_int
        L.wl_version.restype = C.c_char_p
        L.wl_kernel_launches.restype = C.c_int64
        _lib = L
    return _lib


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _check(t: Optional[torch.Tensor], dtype, device_type: str, name: str, numel: Optional[int] = None):
    if t is None:
        return
    if t.dtype != dtype or t.device.type != device_type or not t.is_contiguous():
        raise TypeError(f"{name}: expected contiguous {dtype} on {device_type}, got {t.dtype} on {t.device}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")


def _as_u32_weights(weights: Optional[torch.Tensor]) -> Optional[torch.Tensor]:
    """Edge weights travel as uint32; torch tensors hold them as int64 (values < 2^32) or int32 bit patterns."""
    if weights is None:
        return None
    if weights.dtype == torch.int64:
        return (weights & 0xFFFFFFFF).to(torch.uint32) if hasattr(torch, "uint32") else weights.to(torch.int32)
    return weights


@dataclass
class RefineResult:
    colors: torch.Tensor
    num_colors: int
    rounds: int
    round_colors: List[int]
    stats: dict
    status: int


def _stats_dict(s: wl_stats) -> dict:
    return {f: getattr(s, f) for f, _ in wl_stats._fields_}


def _make_csr(n, row_ptr, col_idx, weights, device_type):
    _check(row_ptr, torch.int64, device_type, "row_ptr", n + 1)
    _check(col_idx, torch.int32, device_type, "col_idx")
    w = _as_u32_weights(weights)
    if w is not None:
        if w.device.type != device_type or not w.is_contiguous() or w.numel() != col_idx.numel() or w.element_size() != 4:
            raise TypeError("weights: expected contiguous 4-byte integers, one per edge")
    g = wl_csr(n, col_idx.numel(), row_ptr.data_ptr() if n >= 0 else None, col_idx.data_ptr(),
               None if w is None else w.data_ptr())
    return g, w


def wl_refine_workspace_bytes(n: int, m: int) -> int:
    return int(lib().wl_refine_workspace_bytes(n, m))


def wl_refine_deep_workspace_bytes(n: int, m: int) -> int:
    return int(lib().wl_refine_deep_workspace_bytes(n, m))


def wl_refine_host_device_bytes(n: int, m: int, weighted: bool = False, with_init: bool = False) -> int:
    return int(lib().wl_refine_host_device_bytes(n, m, int(weighted), int(with_init)))


def wl_refine(n: int, row_ptr: torch.Tensor, col_idx: torch.Tensor, weights: Optional[torch.Tensor] = None,
              init_colors: Optional[torch.Tensor] = None, seed: int = 0, *, flags: int = 0, max_rounds: int = 0,
              stream_id: int = 0, workspace: Optional[torch.Tensor] = None, out: Optional[torch.Tensor] = None,
              round_cap: int = 4096, allow_max_rounds: bool = False, deep: bool = True, ring_bits: int = 0) -> RefineResult:
    """Algorithm 1 on device-resident CSR tensors.  Returns canonical colours (device int32[n]).  When no workspace is
    given, one large enough for the deep-round (worklist) regime is allocated unless deep=False."""
    L = lib()
    dev = row_ptr.device
    if dev.type != "cuda":
        raise RuntimeError("wl_refine needs CUDA tensors (no CPU fallback); use wl_refine_host for host buffers")
    g, w = _make_csr(n, row_ptr, col_idx, weights, "cuda")
    _check(init_colors, torch.int32, "cuda", "init_colors", n)
    if out is None:
        out = torch.empty(n, dtype=torch.int32, device=dev)
    _check(out, torch.int32, "cuda", "out", n)
    need = wl_refine_deep_workspace_bytes(n, col_idx.numel()) if deep else wl_refine_workspace_bytes(n, col_idx.numel())
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    rc_buf = (C.c_int64 * round_cap)()
    opt = wl_options(flags, max_rounds, stream_id, C.cast(rc_buf, C.c_void_p), round_cap, 0, None, 0, ring_bits)
    st = wl_stats()
    with torch.cuda.device(dev):
        rc = L.wl_refine(C.byref(g), _ptr(init_colors), seed, _ptr(out), C.byref(st), C.byref(opt), _ptr(workspace),
                         workspace.numel(), _stream_ptr(dev))
    if rc != WL_OK and not (allow_max_rounds and rc == WL_EMAXROUNDS):
        raise WlError(rc, "wl_refine")
    return RefineResult(out, st.num_colors, st.rounds, list(rc_buf[: min(st.rounds, round_cap)]), _stats_dict(st), rc)


def wl_refine_host(n: int, row_ptr: torch.Tensor, col_idx: torch.Tensor, weights: Optional[torch.Tensor] = None,
                   init_colors: Optional[torch.Tensor] = None, seed: int = 0, *, flags: int = 0, max_rounds: int = 0,
                   out: Optional[torch.Tensor] = None, round_cap: int = 4096, device=None, pieces: int = 0,
                   device_workspace: Optional[torch.Tensor] = None) -> RefineResult:
    """Same computation from HOST tensors (pinned recommended): H2D, refine, D2H all inside the call; the columns are uploaded
    in `pieces` pieces (0: chosen by the library) behind which the first rounds already run."""
    L = lib()
    if not torch.cuda.is_available():
        raise RuntimeError("wl_refine_host needs a CUDA device (no CPU fallback)")
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    g, w = _make_csr(n, row_ptr, col_idx, weights, "cpu")
    _check(init_colors, torch.int32, "cpu", "init_colors", n)
    if out is None:
        out = torch.empty(n, dtype=torch.int32, pin_memory=True)
    _check(out, torch.int32, "cpu", "out", n)
    rc_buf = (C.c_int64 * round_cap)()
    _check(device_workspace, torch.uint8, "cuda", "device_workspace")
    opt = wl_options(flags, max_rounds, 0, C.cast(rc_buf, C.c_void_p), round_cap, 0, None, 0, 0, pieces,
                     _ptr(device_workspace), 0 if device_workspace is None else device_workspace.numel())
    st = wl_stats()
    with torch.cuda.device(dev):
        rc = L.wl_refine_host(C.byref(g), _ptr(init_colors), seed, _ptr(out), C.byref(st), C.byref(opt),
                              _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_refine_host")
    return RefineResult(out, st.num_colors, st.rounds, list(rc_buf[: min(st.rounds, round_cap)]), _stats_dict(st), rc)


def wl_round_key(seed: int, stream_id: int, rnd: int) -> int:
    return int(lib().wl_round_key(seed, stream_id, rnd))


def wl_weight(key: int, color: int) -> int:
    return int(lib().wl_weight(key, color))


def wl_spmv_round(n, row_ptr, col_idx, weights, colors, key: int, *, flags: int = 0, workspace=None) -> torch.Tensor:
    """S1+S2: y = A w(colors) over Z/2^64.  Returns a device int64 tensor holding the u64 bit patterns."""
    L = lib()
    dev = row_ptr.device
    g, w = _make_csr(n, row_ptr, col_idx, weights, "cuda")
    _check(colors, torch.int32, "cuda", "colors", n)
    y = torch.empty(n, dtype=torch.int64, device=dev)
    need = wl_refine_workspace_bytes(n, col_idx.numel())
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    with torch.cuda.device(dev):
        rc = L.wl_spmv_round(C.byref(g), _ptr(colors), key, _ptr(y), flags, _ptr(workspace), workspace.numel(),
                             _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_spmv_round")
    return y


def wl_spmv_rows(n, row_ptr, col_idx, weights, colors, key: int, rows: torch.Tensor, y: torch.Tensor, *, flags: int = 0,
                 workspace=None) -> torch.Tensor:
    """S1+S2 over an active row list: y[rows] is written, every other entry of y keeps its value.  Returns y."""
    L = lib()
    dev = row_ptr.device
    g, w = _make_csr(n, row_ptr, col_idx, weights, "cuda")
    _check(colors, torch.int32, "cuda", "colors", n)
    _check(rows, torch.int32, "cuda", "rows")
    _check(y, torch.int64, "cuda", "y", n)
    need = wl_refine_workspace_bytes(n, col_idx.numel())
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    with torch.cuda.device(dev):
        rc = L.wl_spmv_rows(C.byref(g), _ptr(colors), key, _ptr(rows), rows.numel(), _ptr(y), flags, _ptr(workspace),
                            workspace.numel(), _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_spmv_rows")
    return y


def wl_relabel(colors: torch.Tensor, k: int, y: torch.Tensor, *, workspace=None):
    """S3+S4: dense ids of the exact pairs (colors[i], y[i]).  -> (new_colors, k')."""
    L = lib()
    n = colors.numel()
    dev = colors.device
    _check(colors, torch.int32, "cuda", "colors")
    _check(y, torch.int64, "cuda", "y", n)
    out = torch.empty_like(colors)
    need = wl_refine_workspace_bytes(n, 0)
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    kk = C.c_int64(0)
    with torch.cuda.device(dev):
        rc = L.wl_relabel(n, _ptr(colors), k, _ptr(y), _ptr(out), C.byref(kk), _ptr(workspace), workspace.numel(),
                          _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_relabel")
    return out, kk.value


def wl_canonicalize(colors: torch.Tensor, *, workspace=None):
    """S6: first-occurrence renumbering.  -> (canonical colours, k)."""
    L = lib()
    n = colors.numel()
    dev = colors.device
    _check(colors, torch.int32, "cuda", "colors")
    out = torch.empty_like(colors)
    need = wl_refine_workspace_bytes(n, 0)
    if workspace is None:
        workspace = torch.empty(max(need, 256), dtype=torch.uint8, device=dev)
    kk = C.c_int64(0)
    with torch.cuda.device(dev):
        rc = L.wl_canonicalize(n, _ptr(colors), _ptr(out), C.byref(kk), _ptr(workspace), workspace.numel(),
                               _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_canonicalize")
    return out, kk.value


def wl_canonicalize_static_max_nodes() -> int:
    """Largest n wl_canonicalize_static takes (the size its fixed device scratch was built for)."""
    return int(lib().wl_canonicalize_static_max_nodes())


def wl_canonicalize_static(colors: torch.Tensor, out: torch.Tensor, num_colors: torch.Tensor = None) -> None:
    """S6 with no allocation anywhere (library or binding): the caller owns `out` (int32[n], may be `colors`) and
    `num_colors` (int64[1] on the same device, or None).  Only enqueues on the current stream of the tensors' device and
    returns; results are valid once that stream gets there.  n above wl_canonicalize_static_max_nodes() raises
    WlError(WL_ERANGE).  Calls that overlap on one GPU race on the shared scratch (include/wl_refine.h)."""
    L = lib()
    n = colors.numel()
    dev = colors.device
    _check(colors, torch.int32, "cuda", "colors")
    _check(out, torch.int32, "cuda", "out")
    if out.numel() != n or out.device != dev:
        raise ValueError("out must have the shape and device of colors")
    if num_colors is not None:
        _check(num_colors, torch.int64, "cuda", "num_colors")
        if num_colors.numel() < 1 or num_colors.device != dev:
            raise ValueError("num_colors must be an int64 tensor on the device of colors")
    with torch.cuda.device(dev):
        rc = L.wl_canonicalize_static(n, _ptr(colors), _ptr(out), _ptr(num_colors) if num_colors is not None else None,
                                      _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_canonicalize_static")


def wl_inner_labels(n: int, row_ptr: torch.Tensor, edge_batch: torch.Tensor, sink_batch: torch.Tensor) -> torch.Tensor:
    """B2: inner-node labels of Def. 5 (-1 = boundary) for an arbitrary edge partition given per CSR edge slot."""
    L = lib()
    dev = row_ptr.device
    _check(row_ptr, torch.int64, "cuda", "row_ptr", n + 1)
    _check(edge_batch, torch.int32, "cuda", "edge_batch")
    _check(sink_batch, torch.int32, "cuda", "sink_batch", n)
    label = torch.empty(n, dtype=torch.int32, device=dev)
    with torch.cuda.device(dev):
        rc = L.wl_inner_labels(n, _ptr(row_ptr), _ptr(edge_batch), _ptr(sink_batch), _ptr(label), _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_inner_labels")
    return label


def wl_quotient_workspace_bytes(n: int, m: int) -> int:
    return int(lib().wl_quotient_workspace_bytes(n, m))


def wl_quotient(n, row_ptr, col_idx, weights, colors: torch.Tensor, k: int):
    """B6: quotient graph of Def. 4 for canonical colours.  -> (q_row_ptr int64[k+1], q_col int32[q_m], q_weights int64[q_m])
    with every (block, target block) pair stored once; order inside a row is unspecified."""
    L = lib()
    dev = row_ptr.device
    g, w = _make_csr(n, row_ptr, col_idx, weights, "cuda")
    _check(colors, torch.int32, "cuda", "colors", n)
    m = col_idx.numel()
    q_rp = torch.zeros(k + 1, dtype=torch.int64, device=dev)
    q_col = torch.empty(max(m, 1), dtype=torch.int32, device=dev)
    q_wt = torch.empty(max(m, 1), dtype=torch.int32, device=dev)
    ws = torch.empty(max(wl_quotient_workspace_bytes(n, m), 256), dtype=torch.uint8, device=dev)
    qm = C.c_int64(0)
    with torch.cuda.device(dev):
        rc = L.wl_quotient(C.byref(g), _ptr(colors), k, _ptr(q_rp), _ptr(q_col), _ptr(q_wt), m, C.byref(qm), _ptr(ws),
                           ws.numel(), _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_quotient")
    return q_rp, q_col[: qm.value], q_wt[: qm.value].to(torch.int64) & 0xFFFFFFFF


def wl_refine_inner(row_ptr: torch.Tensor, col_idx: torch.Tensor, weights: Optional[torch.Tensor], lo: int, n_targets: int,
                    seed: int = 0, *, stream_id: int = 0, flags: int = 0, ring_bits: int = 0):
    """B3 + B4 of one batch on device tensors: the rows of the inner nodes [lo, lo + n) (row_ptr[0] = 0, global targets), every
    other target an implicit singleton.  -> (local colours int32[n] in first-occurrence order, is_first uint8[n], k)."""
    L = lib()
    dev = row_ptr.device
    nr = row_ptr.numel() - 1
    g, w = _make_csr(nr, row_ptr, col_idx, weights, "cuda")
    colors = torch.empty(nr, dtype=torch.int32, device=dev)
    first = torch.empty(nr, dtype=torch.uint8, device=dev)
    ws = torch.empty(max(int(L.wl_refine_inner_workspace_bytes(nr, col_idx.numel())), 256), dtype=torch.uint8, device=dev)
    opt = wl_options(flags, 0, stream_id, None, 0, 0, None, 0, ring_bits)
    k = C.c_int64(0)
    with torch.cuda.device(dev):
        rc = L.wl_refine_inner(C.byref(g), lo, n_targets, seed, _ptr(colors), _ptr(first), C.byref(k), C.byref(opt), _ptr(ws),
                               ws.numel(), _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_refine_inner")
    return colors, first, k.value


def wl_quotient_rows(row_ptr: torch.Tensor, col_idx: torch.Tensor, weights: Optional[torch.Tensor], lo: int, block_of: torch.Tensor,
                     is_first: torch.Tensor, first_block: int, num_blocks: int, raw: bool = False):
    """B6 for whole rows on device tensors: quotient rows of the blocks whose first node lies in [lo, lo + n).
    -> (q_row_ptr int64[num_blocks + 1], q_col int32[q_m], q_weights int64[q_m]); raw: the buffers as the library wrote them
    (q_row_ptr, q_col int32[capacity], q_weights int32[capacity] = uint32 bit patterns, q_m)."""
    L = lib()
    dev = row_ptr.device
    nr = row_ptr.numel() - 1
    g, w = _make_csr(nr, row_ptr, col_idx, weights, "cuda")
    _check(block_of, torch.int32, "cuda", "block_of")
    _check(is_first, torch.uint8, "cuda", "is_first", nr)
    m = col_idx.numel()
    q_rp = torch.zeros(num_blocks + 1, dtype=torch.int64, device=dev)
    q_col = torch.empty(max(m, 1), dtype=torch.int32, device=dev)
    q_wt = torch.empty(max(m, 1), dtype=torch.int32, device=dev)
    ws = torch.empty(max(int(L.wl_quotient_rows_workspace_bytes(nr, m, num_blocks)), 256), dtype=torch.uint8, device=dev)
    qm = C.c_int64(0)
    with torch.cuda.device(dev):
        rc = L.wl_quotient_rows(C.byref(g), lo, _ptr(block_of), _ptr(is_first), first_block, num_blocks, _ptr(q_rp), _ptr(q_col),
                                _ptr(q_wt), m, C.byref(qm), _ptr(ws), ws.numel(), _stream_ptr(dev))
    if rc != WL_OK:
        raise WlError(rc, "wl_quotient_rows")
    if raw:
        return q_rp, q_col, q_wt, qm.value
    return q_rp, q_col[: qm.value], q_wt[: qm.value].to(torch.int64) & 0xFFFFFFFF


def wl_refine_batched(n: int, row_ptr: torch.Tensor, col_idx: torch.Tensor, weights: Optional[torch.Tensor] = None, *,
                      max_batch_edges: int = 0, cuts=None, seed: int = 0, device_cap_bytes: int = 0, flags: int = 0,
                      max_outer_iters: int = 0, out: Optional[torch.Tensor] = None, device=None,
                      allow_limit: bool = False, host_workspace: Optional[torch.Tensor] = None,
                      coo_batches=None, init_colors: Optional[torch.Tensor] = None,
                      device_workspace: Optional[torch.Tensor] = None) -> RefineResult:
    """Algorithm 2 over a HOST-resident CSR (pinned recommended).  cuts (optional, increasing edge positions from 0 to m)
    gives the edge partition of the first outer iteration as consecutive CSR slices; otherwise the library cuts by
    max_batch_edges; max_batch_edges <= 0 (with device_cap_bytes > 0): the library derives M_b from the cap.
    coo_batches (optional): an ARBITRARY edge partition as a list of (src int32[e], col int32[e],
    weights or None) host tensors, one triple per batch; row_ptr / col_idx / weights are then ignored (pass None).
    init_colors (optional): HOST int32[n] initial classes (wl_options.batched_init_colors, reading Q18).
    device_workspace (optional): a device uint8 arena the call cuts all its device buffers from (no cudaMalloc / cudaFree).
    Returns canonical colours on the original nodes (host int32[n])."""
    L = lib()
    if not torch.cuda.is_available():
        raise RuntimeError("wl_refine_batched needs a CUDA device (no CPU fallback)")
    dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    keep = []
    if coo_batches is not None:
        g, w = None, None
    else:
        g, w = _make_csr(n, row_ptr, col_idx, weights, "cpu")
    if out is None:
        out = torch.empty(n, dtype=torch.int32)
    _check(out, torch.int32, "cpu", "out", n)
    if host_workspace is not None:
        if host_workspace.device.type != "cpu" or host_workspace.dtype != torch.uint8 or not host_workspace.is_contiguous():
            raise ValueError("host_workspace must be a contiguous host uint8 tensor (pinned: the transfers then overlap)")
    opt = wl_options(flags, 0, 0, None, 0, max_outer_iters, _ptr(host_workspace),
                     0 if host_workspace is None else host_workspace.numel())
    if init_colors is not None:
        _check(init_colors, torch.int32, "cpu", "init_colors", n)
        opt.batched_init_colors = init_colors.data_ptr()
    if device_workspace is not None:
        _check(device_workspace, torch.uint8, "cuda", "device_workspace")
        opt.device_workspace = device_workspace.data_ptr()
        opt.device_workspace_bytes = device_workspace.numel()
    st = wl_stats()
    nb = 0
    batches = None
    if coo_batches is not None:
        nb = len(coo_batches)
        arr = (wl_edge_batch * max(nb, 1))()
        for k, (bs, bc, bw) in enumerate(coo_batches):
            _check(bs, torch.int32, "cpu", "coo src")
            _check(bc, torch.int32, "cpu", "coo col", bs.numel())
            bw = _as_u32_weights(bw)
            if bw is not None and (bw.device.type != "cpu" or bw.numel() != bs.numel() or bw.element_size() != 4):
                raise TypeError("coo weights: expected contiguous 4-byte integers, one per edge")
            keep.append((bs, bc, bw))
            arr[k].edge_begin = 0
            arr[k].num_edges = bs.numel()
            arr[k].row_ptr = None
            arr[k].col_idx = bc.data_ptr()
            arr[k].weights = None if bw is None else bw.data_ptr()
            arr[k].src = bs.data_ptr()
        batches = arr
    elif cuts is not None:
        cuts = [int(c) for c in cuts]
        nb = len(cuts) - 1
        arr = (wl_edge_batch * nb)()
        for k in range(nb):
            arr[k].edge_begin = cuts[k]
            arr[k].num_edges = cuts[k + 1] - cuts[k]
            arr[k].row_ptr = row_ptr.data_ptr()
            arr[k].col_idx = col_idx.data_ptr() + 4 * cuts[k]
            arr[k].weights = None if w is None else w.data_ptr() + 4 * cuts[k]
            arr[k].src = None
        batches = arr
    with torch.cuda.device(dev):
        rc = L.wl_refine_batched(n, nb, batches, C.byref(g) if batches is None else None, seed, device_cap_bytes,
                                 max_batch_edges, _ptr(out), C.byref(st), C.byref(opt), _stream_ptr(dev))
    if rc != WL_OK and not (allow_limit and rc == WL_EMAXROUNDS):
        raise WlError(rc, "wl_refine_batched")
    return RefineResult(out, st.num_colors, st.rounds, [], _stats_dict(st), rc)


def wl_refine_batched_host_bytes(n: int, m: int) -> int:
    return int(lib().wl_refine_batched_host_bytes(n, m))


def wl_refine_batched_host_bytes_consume(n: int, m: int, weighted: bool = False) -> int:
    return int(lib().wl_refine_batched_host_bytes_consume(n, m, 1 if weighted else 0))


def wl_refine_batched_host_overflow_bytes(m: int) -> int:
    return int(lib().wl_refine_batched_host_overflow_bytes(m))


def wl_strerror(code: int) -> str:
    return lib().wl_strerror(code).decode()


def wl_kernel_launches() -> int:
    return int(lib().wl_kernel_launches())


def wl_version() -> str:
    return lib().wl_version().decode()
