"""GPU parity of tcw_prepare (NEXT-3) against oracle/prep.py.

Bars: the GPU computes in float32 (cuFFT), the oracle in float64, so
  * rho: |gpu - oracle| <= 2e-4 * max(1, oracle)   (float32 transform of N <= 32768 points: the
         power of a bin carries a few 1e-6 of the mean power; the median of 101 such values likewise)
  * nu:  identical wherever the oracle's rho is not within that tolerance of the threshold
         (the decision is taken in float32 on the GPU, the precision of the path)
  * u8 and bit-packed outputs carry the same nu.
"""
import math

import numpy as np
import pytest

import tcw_inputs
from oracle import prep

from test_gpu_parity import tcw  # noqa: F401

pytestmark = pytest.mark.gpu

TOL = 2e-4


def _unpack(words, n_bins):
    w = np.ascontiguousarray(words).view(np.uint32)
    bits = (w[:, :, None] >> np.arange(32, dtype=np.uint32)[None, None, :]) & 1
    return bits.reshape(w.shape[0], -1)[:, :n_bins].astype(np.uint8)


def _check(tcw, x, fs, T, f_min, n_bins, W, thr, device_input=False):
    import torch
    rho_o, nu_o = prep.prepare(x, fs, T, f_min, n_bins, W, thr)
    src = torch.from_numpy(x).cuda() if device_input else x
    rho = tcw.prepare(src, fs, T, f_min, n_bins, W, thr, "f32").cpu().numpy()
    nu8 = tcw.prepare(src, fs, T, f_min, n_bins, W, thr, "u8").cpu().numpy()
    nub = _unpack(tcw.prepare(src, fs, T, f_min, n_bins, W, thr, "bits").cpu().numpy(), n_bins)
    assert rho.shape == rho_o.shape
    tol = TOL * np.maximum(1.0, rho_o)
    err = np.abs(rho.astype(np.float64) - rho_o)
    assert np.all(err <= tol), (float((err / tol).max()), np.unravel_index(np.argmax(err / tol), err.shape))
    clear = np.abs(rho_o - thr) > tol
    assert clear.mean() > 0.999
    assert np.array_equal(nu8[clear], nu_o[clear])
    assert np.array_equal(nu8, nub)
    assert np.array_equal(nu8, (rho > np.float32(thr)).astype(np.uint8))     # the GPU's own decision, in float32
    return rho, nu8


def test_small_segments_ragged_band(tcw):
    """N = 512, W = 9, a band that is not a multiple of 32 or of the CTA size, trailing partial segment."""
    rng = np.random.default_rng(0)
    x = rng.standard_normal(11 * 512 + 77).astype(np.float32)
    rho, _ = _check(tcw, x, 64.0, 8.0, 8.0, 173, 9, 1.6)
    assert rho.shape == (11, 173)
    _check(tcw, x, 64.0, 8.0, 0.5, 251, 1, 0.5)          # W = 1: rho = ln 2 everywhere -> nothing above 0.7
    _check(tcw, x, 64.0, 8.0, 2.0, 200, 33, 1.6, device_input=True)


def test_paper_shapes_8s_sfts_with_lines(tcw):
    """8-s SFTs at 4096 Hz (N = 32768), band 500-1000 Hz (4000 bins), W = 101, a strong line at
    600 Hz and a weak one at 812.3 Hz on a non-stationary floor."""
    x = tcw_inputs.synthetic_strain(24, 4096.0, 8.0, 3, lines=[(600.0, 0.5), (812.3, 0.02)])
    rho, nu = _check(tcw, x, 4096.0, 8.0, 500.0, 4000, 101, 1.6)
    assert rho.shape == (24, 4000)
    k = int(round((600.0 - 500.0) * 8.0))
    assert (rho[:, k] > 300.0).all() and nu[:, k].all()                    # the line stands far above the floor
    off = np.ones(4000, dtype=bool)
    off[[k - 1, k, k + 1, int(round(312.3 * 8.0))]] = False
    assert abs(rho[:, off].mean() - 1.0) < 0.02                             # normalised: mean 1 off the lines
    assert abs(nu[:, off].mean() - math.exp(-1.6)) < 0.01                   # P(rho > 1.6) = e^-1.6


def test_prepared_spectrogram_feeds_the_search(tcw):
    """tcw_prepare -> tcw_create -> tcw_search on the device, against the oracle's search over the
    oracle's nu: identical counts for the templates whose lookups avoid threshold-ambiguous bins."""
    import dataclasses
    import torch
    import oracle
    fs, T, f_min, n_bins, W, thr = 2048.0, 8.0, 500.0, 1024, 51, 1.6
    n_sft = 64
    x = tcw_inputs.synthetic_strain(n_sft, fs, T, 5)
    rho_o, nu_o = prep.prepare(x, fs, T, f_min, n_bins, W, thr)
    nu = tcw.prepare(x, fs, T, f_min, n_bins, W, thr, "u8")
    ts = 8.0 * np.arange(n_sft) + 4.0
    w = dataclasses.replace(tcw_inputs.make_workload("cfg1"), fmt="u8", spectrogram=nu_o, n_sft=n_sft,
                            timestamps=ts, velocities=tcw_inputs.detector_velocity(ts))
    with tcw.Handle(nu, "u8", n_bins, f_min, T, ts, w.velocities) as h:
        stat, _ = h.search(tcw.Grid.of(w))
        torch.cuda.synchronize()
    ref = oracle.evaluate(w, want_k=True)
    amb = np.abs(rho_o - thr) <= TOL * np.maximum(1.0, rho_o)              # [n_sft][n_bins]
    kk = np.clip(ref.k, 0, n_bins - 1)
    touched = (amb[np.arange(n_sft)[None, :], kk] & (ref.k >= 0) & (ref.k < n_bins)).any(axis=1)
    got = stat.cpu().numpy().reshape(-1)
    assert (~touched).mean() > 0.9
    assert np.array_equal(got[~touched].astype(np.int64), ref.stat[~touched])


def test_prepare_argument_errors(tcw):
    x = np.zeros(4096, dtype=np.float32)
    bad = [dict(fs=63.9), dict(n_bins=0), dict(median_bins=4), dict(median_bins=2001), dict(f_min=0.05),
           dict(f_min=31.0, n_bins=40), dict(f_min=0.0, median_bins=9)]
    for kw in bad:
        args = dict(fs=64.0, T_sft=8.0, f_min=8.0, n_bins=64, median_bins=9, threshold=1.6)
        args.update(kw)
        with pytest.raises(tcw.TcwError) as e:
            tcw.prepare(x, args["fs"], args["T_sft"], args["f_min"], args["n_bins"], args["median_bins"], args["threshold"])
        assert e.value.code == tcw.TCW_EINVAL, kw
    with pytest.raises(tcw.TcwError) as e:
        tcw.prepare(np.zeros(100, dtype=np.float32), 64.0, 8.0, 8.0, 64, 9, 1.6)
    assert e.value.code == tcw.TCW_EINVAL
