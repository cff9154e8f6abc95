"""Pins for the weighted statistic and the critical ratio of oracle/ (NEXT-1; no GPU).

PAPER.md:57 ("weighed taking into account the antenna patterns and changing noise floors")
and eq. (4): Psi = (s - <s>)/sigma_s.  Reading Q21: weights are an
input w[sky][SFT]; <s> = mean1 * sum w and sigma_s^2 = var1 * sum w^2 over the template's
in-band SFTs.  A dropped weight, W1 and W2 swapped, a missing square root, sums taken over all
SFTs instead of the in-band ones, or weights indexed by the wrong axis each fail a test here.
"""
import dataclasses
import math
import os

import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
P_NU = math.exp(-1.6)          # P(rho > 1.6) for rho ~ Exp(1): BASELINE.json:configs[2] threshold


def _mk(spec, ts, vel, f0, tau, brk, sky, fmt="f32", f_min=500.0, T0=0.0, T_sft=8.0):
    spec = np.ascontiguousarray(spec)
    n_bins = spec.shape[1] if fmt != "bits" else None
    return Workload("custom", fmt, spec, len(ts), n_bins, f_min, T_sft,
                    np.asarray(ts, dtype=np.float64), np.asarray(vel, dtype=np.float64), T0,
                    np.asarray(f0, dtype=np.float64), np.asarray(tau, dtype=np.float64),
                    np.asarray(brk, dtype=np.float64), np.asarray(sky, dtype=np.float64).reshape(-1, 3))


def test_eq4_hand_example_golden():
    """tests/golden/eq4_hand_example.txt: two in-band SFTs, one out of band, by hand."""
    rho = np.full((3, 4001), 100.0, dtype=np.float32)
    rho[0, 4000] = 3.5
    rho[1, 0] = 0.25
    w = _mk(rho, [0.0, 75000.0, 400000.0], np.zeros((3, 3)), [1000.0], [5000.0], [5.0], [1.0, 0.0, 0.0])
    wt = np.array([[0.5, 2.0, 4.0]], dtype=np.float32)
    n = 0
    with open(os.path.join(GOLDEN, "eq4_hand_example.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if not line:
                continue
            mean1, var1, s, w1, w2, psi = map(float, line)
            for literal in (False, True):
                r = oracle.evaluate_weighted(w, wt, mean1, var1, literal=literal)
                assert r.s[0] == s and r.w1[0] == w1 and r.w2[0] == w2
                assert r.psi[0] == pytest.approx(psi, rel=1e-15)
            n += 1
    assert n == 2


def test_unit_weights_reduce_to_the_unweighted_sum(cfg1):
    """w = 1: s is the (pinned) unweighted track sum, W1 = W2 = N_inband, Psi = (s - N)/sqrt(N)."""
    ref = oracle.evaluate(cfg1)
    for wt in (None, np.ones((1, cfg1.n_sft), dtype=np.float32)):
        r = oracle.evaluate_weighted(cfg1, wt, 1.0, 1.0)
        assert np.array_equal(r.s, ref.stat)
        assert np.array_equal(r.w1, ref.n_inband) and np.array_equal(r.w2, ref.n_inband)
        n = ref.n_inband.astype(np.float64)
        assert np.allclose(r.psi, (ref.stat - n) / np.sqrt(n), rtol=1e-14, atol=0)


def test_constant_spectrogram_gives_closed_form_psi(cfg1):
    """rho = c everywhere: s = c*W1 so Psi = (c - mean1)*W1/sqrt(var1*W2); c = mean1 gives 0 exactly."""
    wt = tcw_inputs.synthetic_weights(cfg1.sky, cfg1.timestamps, 3)
    for c in (1.0, 2.5):
        w = dataclasses.replace(cfg1, spectrogram=np.full_like(cfg1.spectrogram, c))
        r = oracle.evaluate_weighted(w, wt, 1.0, 4.0)
        assert np.allclose(r.s, c * r.w1, rtol=1e-14)
        assert np.allclose(r.psi, (c - 1.0) * r.w1 / np.sqrt(4.0 * r.w2), rtol=1e-12, atol=1e-12)
    # in-band sums only: W1 is the weight of the in-band SFTs, which for these tracks (k_j is
    # non-increasing, test_zero_velocity...) are the first N_inband SFTs of the list
    n_in = oracle.evaluate(cfg1).n_inband
    csum = np.concatenate([[0.0], np.cumsum(wt[0].astype(np.float64))])
    assert np.allclose(r.w1, csum[n_in], rtol=1e-13)
    assert n_in.min() < cfg1.n_sft                      # the restriction is exercised


def test_weight_scaling_and_linearity(cfg1):
    """Psi is invariant under w -> 4w (exactly: a power of two); s is linear in w."""
    rng = np.random.default_rng(11)
    w1 = rng.uniform(0.2, 2.0, size=(1, cfg1.n_sft)).astype(np.float32)
    w2 = rng.uniform(0.2, 2.0, size=(1, cfg1.n_sft)).astype(np.float32)
    a = oracle.evaluate_weighted(cfg1, w1, 1.0, 1.0)
    b = oracle.evaluate_weighted(cfg1, 4.0 * w1, 1.0, 1.0)
    assert np.array_equal(b.s, 4.0 * a.s) and np.array_equal(b.w2, 16.0 * a.w2)
    assert np.array_equal(a.psi, b.psi)
    c = oracle.evaluate_weighted(cfg1, w2, 1.0, 1.0)
    wsum = (w1.astype(np.float64) + w2.astype(np.float64)).astype(np.float32)
    if np.array_equal(wsum.astype(np.float64), w1.astype(np.float64) + w2.astype(np.float64)):
        d = oracle.evaluate_weighted(cfg1, wsum, 1.0, 1.0)
        assert np.allclose(d.s, a.s + c.s, rtol=1e-13)
    else:                                              # float32 sum not exact: use exactly representable halves
        h1, h2 = np.round(w1 * 64) / 64, np.round(w2 * 64) / 64
        a, c = (oracle.evaluate_weighted(cfg1, h.astype(np.float32), 1.0, 1.0) for h in (h1, h2))
        d = oracle.evaluate_weighted(cfg1, (h1 + h2).astype(np.float32), 1.0, 1.0)
        assert np.allclose(d.s, a.s + c.s, rtol=1e-13)
        assert np.allclose(d.w1, a.w1 + c.w1, rtol=1e-13)


def test_zero_weight_equals_missing_sft(cfg1):
    """An SFT of weight 0 contributes nothing to s, W1, W2: same as dropping it from the list (Q16)."""
    keep = np.ones(cfg1.n_sft, dtype=bool)
    keep[[3, 17, 18, 100, 255]] = False
    wt = tcw_inputs.synthetic_weights(cfg1.sky, cfg1.timestamps, 5)
    wz = wt.copy()
    wz[:, ~keep] = 0.0
    a = oracle.evaluate_weighted(cfg1, wz, 1.0, 1.0)
    sub = dataclasses.replace(cfg1, spectrogram=np.ascontiguousarray(cfg1.spectrogram[keep]), n_sft=int(keep.sum()),
                              timestamps=cfg1.timestamps[keep], velocities=np.ascontiguousarray(cfg1.velocities[keep]))
    b = oracle.evaluate_weighted(sub, np.ascontiguousarray(wt[:, keep]), 1.0, 1.0)
    assert np.allclose(a.s, b.s, rtol=1e-14) and np.allclose(a.w1, b.w1, rtol=1e-14)
    assert np.allclose(a.psi, b.psi, rtol=1e-12, atol=1e-12)


def test_weights_are_indexed_sky_major():
    """w[s][j]: sky point s uses row s.  Two sky points with zero velocity have identical tracks, so
    their statistics differ only through their weight rows."""
    rng = np.random.default_rng(2)
    n_sft = 40
    ts = 8.0 * np.arange(n_sft) + 4.0
    rho = rng.standard_exponential((n_sft, 64)).astype(np.float32)
    w = _mk(rho, ts, np.zeros((n_sft, 3)), 500.0 + 0.125 * np.arange(8, 40), [1e6], [5.0],
            [[1.0, 0.0, 0.0], [0.0, 1.0, 0.0]])
    wt = np.stack([np.ones(n_sft), np.arange(n_sft) % 2]).astype(np.float32)
    r = oracle.evaluate_weighted(w, wt, 1.0, 1.0)
    n_f0 = len(w.f0)
    even = dataclasses.replace(w, sky=w.sky[:1])
    r_odd = oracle.evaluate_weighted(even, wt[1:], 1.0, 1.0)
    assert np.array_equal(r.s[n_f0:], r_odd.s) and np.array_equal(r.w1[n_f0:], r_odd.w1)
    assert np.array_equal(r.s[:n_f0], oracle.evaluate(even).stat)
    assert not np.array_equal(r.s[:n_f0], r.s[n_f0:])


def test_numpy_twin_on_cfg1(cfg1):
    """Independent numpy write of steps 1-16 (np.power instead of powq: the bins agree on cfg1,
    see test_tiny_brute_force_numpy_twin) against the C oracle, power and count formats."""
    wt = tcw_inputs.synthetic_weights(cfg1.sky, cfg1.timestamps, cfg1.seed)
    t, f0 = cfg1.timestamps, cfg1.f0
    k_min = 4000
    for fmt, mean1, var1 in (("f32", 1.0, 1.0), ("u8", P_NU, P_NU * (1 - P_NU))):
        w = cfg1.with_format(fmt)
        r = oracle.evaluate_weighted(w, wt, mean1, var1)
        data = w.spectrogram.astype(np.float64)
        D = 1.0 + (cfg1.velocities @ cfg1.sky[0]) / tcw_inputs.C_LIGHT
        q = 0
        for tau in cfg1.tau:
            for n in cfg1.brk:
                g = np.power(t / tau + 1.0, 1.0 / (1.0 - n))
                k = np.rint(f0[:, None] * g[None, :] * D[None, :] * 8.0).astype(np.int64) - k_min
                ok = (k >= 0) & (k < cfg1.n_bins)
                val = data[np.arange(cfg1.n_sft)[None, :], np.clip(k, 0, cfg1.n_bins - 1)]
                wd = wt[0].astype(np.float64)[None, :]
                s = np.where(ok, wd * val, 0.0).sum(axis=1)
                W1 = np.where(ok, wd, 0.0).sum(axis=1)
                W2 = np.where(ok, wd * wd, 0.0).sum(axis=1)
                sl = slice(q, q + len(f0))
                assert np.allclose(r.s[sl], s, rtol=1e-12)
                assert np.allclose(r.w1[sl], W1, rtol=1e-12) and np.allclose(r.w2[sl], W2, rtol=1e-12)
                assert np.allclose(r.psi[sl], (s - mean1 * W1) / np.sqrt(var1 * W2), rtol=1e-10, atol=1e-10)
                q += len(f0)


def test_psi_noise_moments():
    """Pure noise: Psi has mean 0 and variance 1 over templates for both statistics (textbook moments
    of a weighted sum of independent Exp(1) / Bernoulli(p) variables)."""
    rng = np.random.default_rng(5)
    n_sft, n_bins = 512, 4096
    ts = 8.0 * np.arange(n_sft) + 4.0
    rho = rng.standard_exponential((n_sft, n_bins)).astype(np.float32)
    f0 = 520.0 + 0.125 * np.arange(0, 3600, 9)       # well separated templates: near-independent sums
    w = _mk(rho, ts, tcw_inputs.detector_velocity(ts), f0, [20000.0], [5.0], tcw_inputs.sky_vector(1.0, 0.3))
    wt = tcw_inputs.synthetic_weights(w.sky, ts, 9)
    r = oracle.evaluate_weighted(w, wt, 1.0, 1.0)
    n = len(f0)
    assert abs(r.psi.mean()) < 4.0 / math.sqrt(n)
    assert abs(r.psi.var() - 1.0) < 0.35
    nu = dataclasses.replace(w, fmt="u8", spectrogram=(rho > np.float32(1.6)).astype(np.uint8))
    r = oracle.evaluate_weighted(nu, wt, P_NU, P_NU * (1 - P_NU))
    assert abs(r.psi.mean()) < 4.0 / math.sqrt(n)
    assert abs(r.psi.var() - 1.0) < 0.35
    # the wrong moments are visibly off: mean1 = 1 on counts shifts Psi by -(1-p) W1/sigma
    r_bad = oracle.evaluate_weighted(nu, wt, 1.0, 1.0)
    assert r_bad.psi.mean() < -5.0


def test_no_inband_sft_gives_zero_psi():
    """W2 = 0 (template never in band): Psi = 0, s = 0."""
    rho = np.ones((4, 16), dtype=np.float32)
    w = _mk(rho, [4.0, 12.0, 20.0, 28.0], np.zeros((4, 3)), [400.0], [5000.0], [5.0], [1.0, 0.0, 0.0])
    r = oracle.evaluate_weighted(w, None, 1.0, 1.0)
    assert r.s[0] == 0.0 and r.w1[0] == 0.0 and r.psi[0] == 0.0


def test_bits_equals_u8_weighted(cfg1):
    wt = tcw_inputs.synthetic_weights(cfg1.sky, cfg1.timestamps, 1)
    a = oracle.evaluate_weighted(cfg1.with_format("u8"), wt, P_NU, P_NU * (1 - P_NU))
    b = oracle.evaluate_weighted(cfg1.with_format("bits"), wt, P_NU, P_NU * (1 - P_NU))
    assert np.array_equal(a.s, b.s) and np.array_equal(a.psi, b.psi)
