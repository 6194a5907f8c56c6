"""ORACLE — test infrastructure only (see the header of wl_oracle.cpp).

ctypes wrapper over oracle/liboracle.so.  Takes and returns numpy arrays.  Imports nothing from the
CUDA package; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from .build import build as _build

_lib = None


def _p(a, ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        i64, i32, u64 = C.c_int64, C.c_int32, C.c_uint64
        pi64, pi32, pu32, pu64 = (C.POINTER(t) for t in (C.c_int64, C.c_int32, C.c_uint32, C.c_uint64))
        L.oracle_canonical.restype = i64
        L.oracle_canonical.argtypes = [i64, pi32, pi32]
        L.oracle_is_stable.restype = C.c_int
        L.oracle_is_stable.argtypes = [i64, pi64, pi32, pu32, pi32]
        L.oracle_refine.restype = i64
        L.oracle_refine.argtypes = [i64, pi64, pi32, pu32, pi32, pi32, i32, pi64, pi32]
        L.oracle_inner_labels.restype = None
        L.oracle_inner_labels.argtypes = [i64, pi64, pi32, pi32, pi32]
        L.oracle_quotient.restype = i64
        L.oracle_quotient.argtypes = [i64, pi64, pi32, pu32, pi32, i64, pi64, pi32, pu32]
        L.oracle_rbsc.restype = i64
        L.oracle_rbsc.argtypes = [i64, pi64, pi32, pu32, i64, i32, pi64, pi32, i32, i32, i32, pi32, pi64]
        L.oracle_rbsc_init.restype = i64
        L.oracle_rbsc_init.argtypes = [i64, pi64, pi32, pu32, pi32, i64, i32, pi64, pi32, i32, i32, i32, pi32, pi64]
        L.oracle_round_key.restype = u64
        L.oracle_round_key.argtypes = [u64, u64, u64]
        L.oracle_weight.restype = u64
        L.oracle_weight.argtypes = [u64, u64]
        L.oracle_spmv_u64.restype = None
        L.oracle_spmv_u64.argtypes = [i64, pi64, pi32, pu32, pu64, i32, pu64]
        L.oracle_rsc.restype = i64
        L.oracle_rsc.argtypes = [i64, pi64, pi32, pu32, pi32, u64, u64, i32, pi32, i32, pi64, pi32, i32, pu64]
        _lib = L
    return _lib


def _csr(n, row_ptr, col, wt):
    rp = np.ascontiguousarray(row_ptr, dtype=np.int64)
    ci = np.ascontiguousarray(col, dtype=np.int32)
    w = None if wt is None else np.ascontiguousarray(wt, dtype=np.uint32)
    assert rp.shape == (n + 1,) and ci.shape == (rp[-1],)
    return rp, ci, w


def canonical(colors) -> np.ndarray:
    c = np.ascontiguousarray(colors, dtype=np.int32)
    out = np.empty_like(c)
    lib().oracle_canonical(c.size, _p(c, C.c_int32), _p(out, C.c_int32))
    return out


def is_stable(n, row_ptr, col, wt, colors) -> bool:
    rp, ci, w = _csr(n, row_ptr, col, wt)
    c = np.ascontiguousarray(colors, dtype=np.int32)
    return bool(lib().oracle_is_stable(n, _p(rp, C.c_int64), _p(ci, C.c_int32), _p(w, C.c_uint32), _p(c, C.c_int32)))


def refine(n, row_ptr, col, wt=None, init=None, max_rounds: Optional[int] = None, allow_unconverged: bool = False):
    """-> (colors int32[n] canonical, counts per round list, rounds).  allow_unconverged: return the partition reached after
    max_rounds rounds instead of raising (used to walk the trajectory round by round)."""
    rp, ci, w = _csr(n, row_ptr, col, wt)
    ini = None if init is None else np.ascontiguousarray(init, dtype=np.int32)
    max_rounds = n + 2 if max_rounds is None else max_rounds
    out = np.empty(n, dtype=np.int32)
    counts = np.zeros(max(max_rounds, 1), dtype=np.int64)
    rounds = C.c_int32(0)
    k = lib().oracle_refine(n, _p(rp, C.c_int64), _p(ci, C.c_int32), _p(w, C.c_uint32), _p(ini, C.c_int32),
                            _p(out, C.c_int32), max_rounds, _p(counts, C.c_int64), C.byref(rounds))
    if k < 0 and not allow_unconverged:
        raise RuntimeError("oracle_refine: max_rounds reached")
    return out, counts[: rounds.value].tolist(), rounds.value


def inner_labels(n, row_ptr, edge_batch, sink_batch) -> np.ndarray:
    rp = np.ascontiguousarray(row_ptr, dtype=np.int64)
    eb = np.ascontiguousarray(edge_batch, dtype=np.int32)
    sb = np.ascontiguousarray(sink_batch, dtype=np.int32)
    out = np.empty(n, dtype=np.int32)
    lib().oracle_inner_labels(n, _p(rp, C.c_int64), _p(eb, C.c_int32), _p(sb, C.c_int32), _p(out, C.c_int32))
    return out


def quotient(n, row_ptr, col, wt, colors):
    """colors must be canonical.  -> (k, q_row_ptr, q_col, q_wt)."""
    rp, ci, w = _csr(n, row_ptr, col, wt)
    c = np.ascontiguousarray(colors, dtype=np.int32)
    k = int(c.max()) + 1 if n else 0
    qrp = np.zeros(k + 1, dtype=np.int64)
    qc = np.zeros(max(ci.size, 1), dtype=np.int32)
    qw = np.zeros(max(ci.size, 1), dtype=np.uint32)
    qm = lib().oracle_quotient(n, _p(rp, C.c_int64), _p(ci, C.c_int32), _p(w, C.c_uint32), _p(c, C.c_int32), k,
                               _p(qrp, C.c_int64), _p(qc, C.c_int32), _p(qw, C.c_uint32))
    return k, qrp, qc[:qm].copy(), qw[:qm].copy()


def rbsc(n, row_ptr, col, wt, max_batch_edges, first_cuts=None, first_edge_batch=None, num_first_batches=0,
         max_outer=1 << 30, inherit=False, aggressive=False, init=None):
    """Algorithm 2 with the deterministic oracle as RSC.  -> (colors, k, outer_iters, last_num_batches).
    inherit: the quotient keeps the batches of its graph instead of being re-cut by max_batch_edges (reading Q14b).
    aggressive: stop as soon as the next iteration would not run with fewer batches.
    init: initial classes (reading Q18): Eq. 3's local start intersected with them."""
    rp, ci, w = _csr(n, row_ptr, col, wt)
    fc = None if first_cuts is None else np.ascontiguousarray(first_cuts, dtype=np.int64)
    fb = None if first_edge_batch is None else np.ascontiguousarray(first_edge_batch, dtype=np.int32)
    nb0 = num_first_batches if fb is not None else (0 if fc is None else fc.size - 1)
    out = np.empty(n, dtype=np.int32)
    stats = np.zeros(2, dtype=np.int64)
    ini = None if init is None else np.ascontiguousarray(init, dtype=np.int32)
    k = lib().oracle_rbsc_init(n, _p(rp, C.c_int64), _p(ci, C.c_int32), _p(w, C.c_uint32), _p(ini, C.c_int32), max_batch_edges,
                               nb0, _p(fc, C.c_int64), _p(fb, C.c_int32), max_outer, 1 if inherit else 0,
                               1 if aggressive else 0, _p(out, C.c_int32), _p(stats, C.c_int64))
    return out, int(k), int(stats[0]), int(stats[1])


def round_key(seed, stream, rnd) -> int:
    return int(lib().oracle_round_key(seed, stream, rnd))


def weight(key, c) -> int:
    return int(lib().oracle_weight(key, c))


def spmv_u64(n, row_ptr, col, wt, w, qbits=64) -> np.ndarray:
    rp, ci, ww = _csr(n, row_ptr, col, wt)
    wv = np.ascontiguousarray(w, dtype=np.uint64)
    z = np.empty(n, dtype=np.uint64)
    lib().oracle_spmv_u64(n, _p(rp, C.c_int64), _p(ci, C.c_int32), _p(ww, C.c_uint32), _p(wv, C.c_uint64), qbits,
                          _p(z, C.c_uint64))
    return z


def rsc(n, row_ptr, col, wt=None, init=None, seed=0, stream=0, qbits=64, max_rounds=None, z_round=0):
    """Algorithm 1 in Z/2^q on the CPU.  -> (colors, counts, rounds, z of round z_round or None)."""
    rp, ci, w = _csr(n, row_ptr, col, wt)
    ini = None if init is None else np.ascontiguousarray(init, dtype=np.int32)
    max_rounds = n + 2 if max_rounds is None else max_rounds
    out = np.empty(n, dtype=np.int32)
    counts = np.zeros(max(max_rounds, 1), dtype=np.int64)
    rounds = C.c_int32(0)
    z = np.zeros(n, dtype=np.uint64) if z_round > 0 else None
    k = lib().oracle_rsc(n, _p(rp, C.c_int64), _p(ci, C.c_int32), _p(w, C.c_uint32), _p(ini, C.c_int32), seed, stream,
                         qbits, _p(out, C.c_int32), max_rounds, _p(counts, C.c_int64), C.byref(rounds), z_round,
                         _p(z, C.c_uint64))
    if k < 0:
        raise RuntimeError("oracle_rsc: max_rounds reached")
    return out, counts[: rounds.value].tolist(), rounds.value, z
