"""rfoe_bounds_static: the Gershgorin bounds (row A1) through the entry point that allocates nothing -- scratch in a
file-scope device array, no handle (include/rfoe.h) -- against the existing path, rfoe_bounds, and the CPU oracle.

Collected last on purpose (the suite runs with `pytest -x`).  The test holds when run alone in a fresh process (the
first call resolves the array's address) and after every other GPU test (the array then carries whatever an earlier
call left in it: each call here uses a different size and different matrices, so stale entries would show)."""
import gc
import math

import numpy as np
import pytest

import oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

import paper_2301_04642_b200 as rfoe  # noqa: E402

EPS = np.finfo(np.float64).eps


def _sym(k, seed):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((k, k))
    return np.ascontiguousarray(0.5 * (A + A.T))


def _check(handle, H, out):
    """one call of the new entry point against rfoe_bounds (bit for bit: same kernels, same row order) and the oracle
    (the tolerance of test_bounds_parity)."""
    k = H.shape[0]
    Hd = torch.from_numpy(H).cuda()
    out.fill_(float("nan"))
    gc.collect()                                           # tensors of earlier tests must not be freed in mid-measurement
    torch.cuda.synchronize()
    before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    got = rfoe.bounds_static(Hd, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() <= before         # torch's allocator: nothing new
    if _check.warm:                                        # the first call of a process may load the module
        assert torch.cuda.mem_get_info()[0] >= free_before   # cudaMemGetInfo: no device allocation by anybody
    _check.warm = True
    lo, hi = (float(v) for v in got.cpu())
    ref_lo, ref_hi = handle.bounds(Hd)
    assert (lo, hi) == (ref_lo, ref_hi)
    olo, ohi = oracle.bounds(H)
    tol = 4 * k * EPS * max(abs(olo), abs(ohi), 1.0)
    assert abs(lo - olo) <= tol and abs(hi - ohi) <= tol
    return lo, hi


_check.warm = False


def test_bounds_static_two_calls_in_a_row_match_rfoe_bounds():
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    with rfoe.Rfoe(2048) as h:
        # two calls in a row, the second SMALLER and shifted: entries [k2, k1) of the shared array still hold the first
        # call's discs, which reach far below / above the second matrix's spectrum -- a reduction that read them would fail
        a = _check(h, 50.0 * _sym(1537, 1), out)
        b = _check(h, _sym(777, 2) + 3.0 * np.eye(777), out)
        assert a[0] < b[0] and a[1] > b[1]
        # and again larger, odd size (the scalar path of the rows kernel), then the smallest
        _check(h, _sym(2047, 3), out)
        _check(h, np.array([[2.5]]), out)
        # back-to-back on one stream WITHOUT a host sync in between: the second call's kernels follow the first's
        H1, H2 = torch.from_numpy(_sym(1024, 4)).cuda(), torch.from_numpy(_sym(640, 5) - 7.0 * np.eye(640)).cuda()
        o1, o2 = torch.empty(2, dtype=torch.float64, device="cuda"), torch.empty(2, dtype=torch.float64, device="cuda")
        rfoe.bounds_static(H1, o1)
        rfoe.bounds_static(H2, o2)
        torch.cuda.synchronize()
        assert tuple(o1.tolist()) == h.bounds(H1) and tuple(o2.tolist()) == h.bounds(H2)


def test_bounds_static_on_a_side_stream_and_non_finite_input():
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    H = torch.from_numpy(_sym(900, 6)).cuda()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        rfoe.bounds_static(H, out, stream=s)
    s.synchronize()
    with rfoe.Rfoe(900) as h:
        assert tuple(out.tolist()) == h.bounds(H)
        # a non-finite H^p never yields finite bounds, exactly as in rfoe_bounds: NaN -> (NaN, NaN), inf -> (-inf, inf)
        H[5, 5] = float("nan")
        rfoe.bounds_static(H, out)
        assert torch.isnan(out).all() and all(math.isnan(v) for v in h.bounds(H))
        H[5, 5] = 0.25
        H[17, 300] = float("inf")
        H[300, 17] = float("inf")
        rfoe.bounds_static(H, out)
        assert tuple(out.tolist()) == (-math.inf, math.inf) == h.bounds(H)


def test_bounds_static_rejects_sizes_beyond_its_array():
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    L = rfoe.load_library()
    import ctypes as C

    H = torch.zeros(16, 16, dtype=torch.float64, device="cuda")
    err = C.c_int(-1)
    # the size is checked before anything is read or launched, so a small buffer may stand for the too-large matrix
    rc = L.rfoe_bounds_static(C.c_void_p(H.data_ptr()), rfoe.STATIC_MAX_K + 1, C.c_void_p(out.data_ptr()), None, C.byref(err))
    assert rc == rfoe.ERR_STATIC_LIMIT and err.value == 0
    assert b"RFOE_STATIC_MAX_K" in L.rfoe_strerror(rc)
    assert L.rfoe_bounds_static(C.c_void_p(H.data_ptr()), 0, C.c_void_p(out.data_ptr()), None, None) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_bounds_static(None, 16, C.c_void_p(out.data_ptr()), None, None) == rfoe.ERR_INVALID_ARG
    assert L.rfoe_bounds_static(C.c_void_p(H.data_ptr()), 16, None, None, None) == rfoe.ERR_INVALID_ARG
    with pytest.raises(ValueError):
        rfoe.bounds_static(H, torch.empty(1, dtype=torch.float64, device="cuda"))


def test_bounds_static_largest_size():
    """k = RFOE_STATIC_MAX_K fills the array to its last entry (8.6 GB matrix, generated on the device)."""
    k = rfoe.STATIC_MAX_K
    g = torch.Generator(device="cuda").manual_seed(7)
    H = torch.randn(k, k, dtype=torch.float64, device="cuda", generator=g)
    H = torch.triu(H) + torch.triu(H, 1).T
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    rfoe.bounds_static(H, out)
    d = torch.diagonal(H)
    r = H.abs().sum(dim=1) - d.abs()
    lo, hi = (d - r).min().item(), (d + r).max().item()
    got = out.tolist()
    assert abs(got[0] - lo) <= 1e-12 * abs(lo) and abs(got[1] - hi) <= 1e-12 * abs(hi)
