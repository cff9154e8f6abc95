"""tcw_select_above_static -- the threshold selection for callers that must not allocate device memory.

Some users of this library cannot let it allocate on the GPU: a search job that has sized its own
spectrograms and result arrays to fill the device, a host program whose caching allocator owns the
memory (a cudaMalloc from a library can then fail although memory looks free), or a follow-up loop
that runs beside searches on other streams and cannot afford the device-wide synchronisation of
cudaMalloc / cudaFree.  For them the library has one entry point whose scratch is a fixed array
inside libtcw.so (include/tcw.h: tcw_select_above_static).  It needs no handle and takes every
input and output from the caller.

What is checked here: its output equals the existing path's (Handle.select_above, which takes its
scratch from the handle) index for index -- selection is integer work, so the bar is equality, the
one tests/test_gpu_select.py uses -- on TWO calls in a row, the second on a shorter array with
fewer hits, so that anything the first call left in the shared array and the second failed to
clear would show.  Also: sizes beyond the fixed maximum are refused with a clear message.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It passes alone in a fresh process and after the other tests.
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tcw():
    import torch
    assert torch.cuda.is_available()
    import paper_2507_07816_b200 as pkg
    pkg.load_library()
    return pkg


def _static(tcw, d, thr, cap):
    import torch
    out_idx = torch.full((cap,), -7, dtype=torch.int64, device=d.device)
    out_cnt = torch.full((1,), -7, dtype=torch.int64, device=d.device)
    tcw.select_above_static(d, thr, out_idx, out_cnt)
    return out_idx, out_cnt


def test_static_selection_equals_the_handle_path_on_two_calls_in_a_row(tcw):
    import torch
    import tcw_inputs
    rng = np.random.default_rng(20260711)
    # call 1: 3 000 017 values (many CTAs, a ragged tail), about 2 % selected, plus a NaN and both zeros;
    # call 2: a shorter array over the same scratch rows with ~0.1 % selected, then an int32 array
    a = rng.standard_normal(3_000_017).astype(np.float32)
    a[[5, 77, 1_000_000]] = [np.nan, -0.0, 0.0]
    b = rng.standard_normal(1_000_003).astype(np.float32)
    c = rng.integers(0, 100, size=700_001).astype(np.int32)
    da, db, dc = (torch.from_numpy(x).cuda() for x in (a, b, c))
    cases = ((da, 2.05, 100_000), (db, 3.1, 4096), (dc, 97.5, 30_000), (db, -10.0, 64), (da, 10.0, 0))
    # the new entry point first, back to back on one stream, before the handle exists
    got = [_static(tcw, d, thr, cap) for d, thr, cap in cases]
    torch.cuda.synchronize()
    with tcw.Handle.from_workload(tcw_inputs.make_workload("cfg1")) as h:
        for (d, thr, cap), (idx, cnt) in zip(cases, got):
            ref_idx, ref_cnt = h.select_above(d, thr, cap)
            torch.cuda.synchronize()
            n_hits = int(ref_cnt.item())
            assert int(cnt.item()) == n_hits
            m = min(cap, n_hits)
            assert torch.equal(idx[:m], ref_idx[:m])
            assert bool((idx[m:] == -7).all())          # nothing written past the hits
            # and the hits are what the definition says (plain torch on the same device array)
            want = torch.nonzero(d.view(-1) > thr).view(-1)
            assert want.numel() == n_hits and torch.equal(idx[:m], want[:m])
        # once more after the handle's own selections ran: the two paths do not disturb each other
        idx, cnt = _static(tcw, da, 2.05, 100_000)
        ref_idx, ref_cnt = h.select_above(da, 2.05, 100_000)
        torch.cuda.synchronize()
        assert int(cnt.item()) == int(ref_cnt.item()) and torch.equal(idx[:int(cnt.item())], ref_idx[:int(cnt.item())])


def test_static_selection_refuses_sizes_beyond_its_scratch(tcw):
    import torch
    L = tcw.load_library()
    d = torch.zeros(1024, dtype=torch.float32, device="cuda")
    cnt = torch.full((1,), -7, dtype=torch.int64, device="cuda")
    # the size check comes before any CUDA work, so a short array can stand in for the oversized one
    rc = L.tcw_select_above_static(d.data_ptr(), 0, tcw.SELECT_STATIC_MAX_N + 1, 0.0, 0, None, cnt.data_ptr(), None)
    assert rc == tcw.TCW_EUNSUPPORTED
    msg = L.tcw_last_error().decode()
    assert "TCW_SELECT_STATIC_MAX_N" in msg and str(tcw.SELECT_STATIC_MAX_N) in msg
    torch.cuda.synchronize()
    assert int(cnt.item()) == -7                       # nothing was touched
    assert L.tcw_select_above_static(None, 0, 10, 0.0, 0, None, cnt.data_ptr(), None) == tcw.TCW_EINVAL
    assert L.tcw_select_above_static(d.data_ptr(), 0, 10, 0.0, 4, None, cnt.data_ptr(), None) == tcw.TCW_EINVAL
    # the largest size it accepts: the whole scratch in use (1 GiB of float32; skipped if the box is short of memory)
    free, _ = torch.cuda.mem_get_info()
    if free < 6 << 30:
        pytest.skip("not enough free device memory for the maximum-size case")
    n = tcw.SELECT_STATIC_MAX_N
    big = torch.zeros(n, dtype=torch.float32, device="cuda")
    hits = torch.tensor([0, 127, 128, n // 2 + 1, n - 129, n - 1], dtype=torch.int64, device="cuda")
    big[hits] = 1.0
    idx, c = _static(tcw, big, 0.5, 16)
    torch.cuda.synchronize()
    assert int(c.item()) == hits.numel() and torch.equal(idx[:hits.numel()], hits)
    # and a small call right after the maximum-size one sees none of its leftovers
    idx, c = _static(tcw, d, -1.0, 2048)
    torch.cuda.synchronize()
    assert int(c.item()) == 1024 and torch.equal(idx[:1024], torch.arange(1024, device="cuda"))
