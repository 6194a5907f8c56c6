"""wl_canonicalize_static: S6 (canonical first-occurrence ids) with its scratch in a fixed device
array of the library, for callers that cannot allocate.  Collected last on purpose (the suite runs with pytest -x).

Bar: integer work, so bit-exact -- against the existing wl_canonicalize path and against the oracle -- on two calls in a row
(the second reuses the scratch the first one left behind), and no device allocation across the calls."""
import ctypes

import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu

wl = pytest.importorskip("paper_2607_02603_b200")


def dev():
    return torch.device("cuda:0")


def _colours(n, k, seed):
    rng = np.random.default_rng(seed)
    return rng.integers(0, max(1, k), n).astype(np.int32)


def test_static_matches_the_workspace_path_on_two_calls_in_a_row():
    nmax = wl.wl_canonicalize_static_max_nodes()
    assert nmax == 1 << 20
    # first call: many colours over several scan chunks and a ragged tail; second call: a SHORTER input with other colours,
    # so stale first-node / id / bit entries of the first call sit right behind what the second one writes
    cases = [_colours(300_007, 150_000, 1), _colours(70_001, 999, 2)]
    d_in = [torch.from_numpy(c).to(dev()) for c in cases]
    d_out = [torch.full_like(t, -7) for t in d_in]
    d_k = [torch.full((1,), -1, dtype=torch.int64, device=dev()) for _ in cases]
    want = [wl.wl_canonicalize(t) for t in d_in]  # existing path (allocates its workspace)
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for t, o, k in zip(d_in, d_out, d_k):  # back to back on one stream, no synchronisation in between
        wl.wl_canonicalize_static(t, o, k)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == before  # nothing was allocated on the device (driver's own count)
    for c, o, k, (w_out, w_k) in zip(cases, d_out, d_k, want):
        assert torch.equal(o, w_out)
        assert int(k.item()) == w_k == np.unique(c).size
        assert o.cpu().numpy().tolist() == oracle.canonical(c).tolist()


def test_static_at_the_maximum_in_place_and_without_a_count():
    nmax = wl.wl_canonicalize_static_max_nodes()
    c = _colours(nmax, nmax, 3)
    t = torch.from_numpy(c).to(dev())
    want, _ = wl.wl_canonicalize(t)
    wl.wl_canonicalize_static(t, t)  # out aliases colors, num_colors NULL
    wl.wl_canonicalize_static(t, t)  # canonical ids are a fixed point of S6
    torch.cuda.synchronize()
    assert torch.equal(t, want)
    assert t.cpu().numpy().tolist() == oracle.canonical(c).tolist()
    # n = 1 and n = 0 (nothing written)
    one = torch.tensor([0], dtype=torch.int32, device=dev())
    out = torch.tensor([5], dtype=torch.int32, device=dev())
    k = torch.tensor([-1], dtype=torch.int64, device=dev())
    wl.wl_canonicalize_static(one, out, k)
    torch.cuda.synchronize()
    assert out.item() == 0 and k.item() == 1
    empty = torch.empty(0, dtype=torch.int32, device=dev())
    k.fill_(-1)
    wl.wl_canonicalize_static(empty, torch.empty_like(empty), k)
    torch.cuda.synchronize()
    assert k.item() == -1


def test_static_on_a_side_stream_two_calls_in_a_row():
    """The call only enqueues on the stream it is given: two calls back to back on a non-default stream, the second one over the
    first one's output (canonical ids are a fixed point of S6), read after synchronising that stream only."""
    c = _colours(200_003, 50_000, 7)
    t = torch.from_numpy(c).to(dev())
    want, want_k = wl.wl_canonicalize(t)
    torch.cuda.synchronize()
    side = torch.cuda.Stream(dev())
    a, b = torch.empty_like(t), torch.empty_like(t)
    ka = torch.zeros(1, dtype=torch.int64, device=dev())
    kb = torch.zeros(1, dtype=torch.int64, device=dev())
    with torch.cuda.stream(side):
        wl.wl_canonicalize_static(t, a, ka)
        wl.wl_canonicalize_static(a, b, kb)
    side.synchronize()
    assert torch.equal(a, want) and torch.equal(b, want)
    assert ka.item() == kb.item() == want_k


def test_static_rejects_what_it_cannot_hold():
    nmax = wl.wl_canonicalize_static_max_nodes()
    t = torch.zeros(nmax + 1, dtype=torch.int32, device=dev())
    out = torch.full_like(t, -7)
    with pytest.raises(wl.WlError) as e:
        wl.wl_canonicalize_static(t, out)
    assert e.value.code == wl.WL_ERANGE
    torch.cuda.synchronize()
    assert bool((out == -7).all())  # nothing was enqueued
    L = wl.lib()
    assert L.wl_canonicalize_static(-1, None, None, None, None) == wl.WL_EINVAL
    assert L.wl_canonicalize_static(8, None, ctypes.c_void_p(out.data_ptr()), None, None) == wl.WL_EINVAL
    assert L.wl_canonicalize_static(8, ctypes.c_void_p(t.data_ptr()), None, None, None) == wl.WL_EINVAL
    assert b"out of range" in L.wl_strerror(wl.WL_ERANGE)
