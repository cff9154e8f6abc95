"""GPU parity of tcw_topk / tcw_select_above (NEXT-4) against oracle/select.py:
exact (values bit-identical, indices identical), ties by lowest index."""
import numpy as np
import pytest

import oracle
import tcw_inputs
from oracle import select

from test_gpu_parity import tcw  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def handle(tcw):
    w = tcw_inputs.make_workload("cfg1")
    with tcw.Handle.from_workload(w) as h:
        yield h


def _topk(handle, arr, K):
    import torch
    val, idx, cnt = handle.topk(torch.from_numpy(arr).cuda(), K)
    torch.cuda.synchronize()
    c = int(cnt.item())
    return val.cpu().numpy()[:c], idx.cpu().numpy()[:c]


def _check_topk(handle, arr, K):
    val, idx = _topk(handle, arr, K)
    rv, ri = select.topk(arr, K)
    assert np.array_equal(idx, ri), (idx[:8], ri[:8])
    assert np.array_equal(val.view(np.uint32) if val.dtype == np.float32 else val,
                          rv.view(np.uint32) if rv.dtype == np.float32 else rv)


@pytest.mark.parametrize("n,K", [(1, 1), (5, 8), (257, 16), (4096, 2048), (100_003, 100), (3_000_017, 2048)])
def test_topk_float_random_and_tied(handle, n, K):
    rng = np.random.default_rng(n)
    _check_topk(handle, rng.standard_normal(n).astype(np.float32), K)
    _check_topk(handle, rng.integers(-3, 4, size=n).astype(np.float32), K)      # heavy ties: lowest index first


@pytest.mark.parametrize("K", [1, 1000, 2048])
def test_topk_two_read_route_large_arrays(handle, K):
    """Arrays of 2^22 values or more take the two-read route (zoomed histogram, ordered compaction of the
    candidates, exact selection on them) or, when the candidates do not fit, the full-array route; every
    case must equal oracle/select.py exactly: values, indices, ties by lowest index."""
    n = 5_000_011
    rng = np.random.default_rng(K)
    a = rng.standard_normal(n).astype(np.float32)                       # the shape of a Psi array
    _check_topk(handle, a, K)
    a[[11, 4_999_999, 2_500_000]] = [np.nan, np.inf, -np.inf]
    a[123_456] = a[4_000_000] = a.max()                                  # a tie at the very top
    _check_topk(handle, a, K)
    _check_topk(handle, (10800.0 + 104.0 * rng.standard_normal(n)).astype(np.float32), K)   # power sums: all positive
    p = (10800.0 + 104.0 * rng.standard_normal(n)).astype(np.float32)
    p[rng.integers(0, n, size=n // 3)] = 0.0                             # many out-of-band templates with stat 0
    _check_topk(handle, p, K)
    _check_topk(handle, rng.integers(-3, 4, size=n).astype(np.float32), K)      # 7 distinct values: ties everywhere
    _check_topk(handle, np.full(n, 2.5, dtype=np.float32), K)                   # one value: candidates cannot fit
    c = rng.binomial(10800, 0.2019, size=n).astype(np.int32)                   # number counts (cfg5's out_stat)
    _check_topk(handle, c, K)
    c[[5, n - 1]] = [np.iinfo(np.int32).max, np.iinfo(np.int32).min]
    _check_topk(handle, c, K)
    _check_topk(handle, np.arange(n, dtype=np.int32)[::-1].copy(), K)           # all distinct, descending


def test_topk_special_values(handle):
    v = np.array([0.5, np.nan, -0.0, 0.0, np.inf, -np.inf, 0.5, -np.nan, 1e-45, -1e-45, 3.4e38], dtype=np.float32)
    _check_topk(handle, v, 11)
    _check_topk(handle, v, 3)
    _check_topk(handle, np.full(1000, np.nan, dtype=np.float32), 5)            # nothing selectable: count 0
    _check_topk(handle, np.full(5000, 2.5, dtype=np.float32), 7)               # all equal: indices 0..6


def test_unaligned_array_start(handle):
    """An array that starts 4 bytes into a 16-byte line takes the scalar-load path."""
    import torch
    rng = np.random.default_rng(9)
    v = rng.standard_normal(50_001).astype(np.float32)
    d = torch.from_numpy(v).cuda()[1:]
    assert d.data_ptr() % 16 == 4
    val, idx, cnt = handle.topk(d, 33)
    sidx, scnt = handle.select_above(d, 1.0, 50_000)
    torch.cuda.synchronize()
    rv, ri = select.topk(v[1:], 33)
    assert np.array_equal(idx.cpu().numpy(), ri) and np.array_equal(val.cpu().numpy(), rv)
    ref = select.select_above(v[1:], 1.0)
    assert int(scnt.item()) == ref.size and np.array_equal(sidx.cpu().numpy()[:ref.size], ref)


def test_topk_int32(handle):
    rng = np.random.default_rng(3)
    v = rng.integers(-50, 50, size=200_001).astype(np.int32)
    v[[7, 199_999]] = [np.iinfo(np.int32).max, np.iinfo(np.int32).min]
    _check_topk(handle, v, 300)
    _check_topk(handle, np.full(100, np.iinfo(np.int32).min, dtype=np.int32), 100)


@pytest.mark.parametrize("n", [1, 1000, 1_000_003])
def test_select_above(handle, n):
    import torch
    rng = np.random.default_rng(n + 1)
    v = rng.standard_normal(n).astype(np.float32)
    if n > 10:
        v[3] = np.nan
    d = torch.from_numpy(v).cuda()
    for thr, cap in ((2.5, 100_000), (-10.0, 64), (10.0, 10), (0.0, 0)):
        idx, cnt = handle.select_above(d, thr, cap)
        torch.cuda.synchronize()
        ref = select.select_above(v, thr)
        assert int(cnt.item()) == ref.size
        m = min(cap, ref.size)
        assert np.array_equal(idx.cpu().numpy()[:m], ref[:m])
    vi = rng.integers(0, 100, size=n).astype(np.int32)
    idx, cnt = handle.select_above(torch.from_numpy(vi).cuda(), 97.5, n)
    torch.cuda.synchronize()
    ref = select.select_above(vi, 97.5)
    assert int(cnt.item()) == ref.size and np.array_equal(idx.cpu().numpy()[:ref.size], ref)


def test_detection_rule_on_a_weighted_search(tcw):
    """PAPER.md:79 end to end on cfg1: Psi_noise max from a noise-only spectrogram with the same
    templates, then the templates of the injected data above it; all against the oracle's Psi."""
    import dataclasses
    import torch
    w = tcw_inputs.make_workload("cfg1")
    noise = dataclasses.replace(w, spectrogram=np.random.default_rng(5).standard_exponential(
        w.spectrogram.shape).astype(np.float32))
    wt = tcw_inputs.synthetic_weights(w.sky, w.timestamps, 1)
    grid = tcw.Grid.of(w)
    with tcw.Handle.from_workload(noise) as hn, tcw.Handle.from_workload(w) as hs:
        psi_n, _, _ = hn.search_weighted(grid, wt, 1.0, 1.0)
        thr_v, thr_i, _ = hn.topk(psi_n, 1)
        psi_s, _, _ = hs.search_weighted(grid, wt, 1.0, 1.0)
        torch.cuda.synchronize()
        thr = float(thr_v.item())
        idx, cnt = hs.select_above(psi_s, thr, 768)
        top_v, top_i, _ = hs.topk(psi_s, 10)
        torch.cuda.synchronize()
    pn, ps = psi_n.cpu().numpy().reshape(-1), psi_s.cpu().numpy().reshape(-1)
    assert thr == select.noise_max(pn) and int(thr_i.item()) == int(np.argmax(pn))
    ref = select.select_above(ps, thr)
    assert int(cnt.item()) == ref.size and np.array_equal(idx.cpu().numpy()[:ref.size], ref)
    rv, ri = select.topk(ps, 10)
    assert np.array_equal(top_i.cpu().numpy(), ri) and np.array_equal(top_v.cpu().numpy(), rv)
    # the oracle's Psi agrees on who is detected wherever its value is clear of the threshold
    ro = oracle.evaluate_weighted(w, wt, 1.0, 1.0)
    clear = np.abs(ro.psi - thr) > 1e-3
    assert np.array_equal((ps > thr)[clear], (ro.psi > thr)[clear])
