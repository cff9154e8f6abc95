"""Pins for the random-template-bank entry of oracle/ (NEXT-2, PAPER.md:63 (ii); no GPU).

The bank statistic is the same ten steps as the grid statistic with per-template parameters,
so it is pinned to the (separately pinned) grid oracle on banks built from a grid, to the
hand-worked values of eq. (1), and to an independent numpy write on a random bank.
"""
import os

import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload, sky_vector

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _grid_as_bank(w):
    """(f0, tau, brk, sky) per template, in the grid's linear order (sky, tau, n, f0 fastest)."""
    s, a, b, i = np.meshgrid(np.arange(len(w.sky)), np.arange(len(w.tau)), np.arange(len(w.brk)),
                             np.arange(len(w.f0)), indexing="ij")
    return w.f0[i.ravel()], w.tau[a.ravel()], w.brk[b.ravel()], w.sky[s.ravel()]


@pytest.mark.parametrize("fmt", ["f32", "bits"])
def test_bank_built_from_a_grid_equals_the_grid_oracle(cfg1, fmt):
    w = cfg1.with_format(fmt)
    f0, tau, brk, sky = _grid_as_bank(w)
    ref = oracle.evaluate(w, want_k=True, literal=True)
    for sk in (sky, w.sky[0]):                       # per-template vectors and the shared vector
        r = oracle.evaluate_bank(w, f0, tau, brk, sk, want_k=True)
        assert np.array_equal(r.k, ref.k)
        assert np.array_equal(r.stat, ref.stat) and np.array_equal(r.n_inband, ref.n_inband)


def test_bank_per_template_sky_is_used(cfg1):
    """Two sky points whose Doppler shifts differ by about a bin move some indices; template q
    must use row q of the sky array."""
    w = cfg1
    n = 64
    f0 = np.full(n, 600.0)
    tau = np.full(n, 9000.0)
    brk = np.full(n, 4.0)
    sky = np.tile(sky_vector(1.0, 0.3), (n, 1))
    sky[1::2] = sky_vector(4.0, -0.3)
    r = oracle.evaluate_bank(w, f0, tau, brk, sky, want_k=True)
    a = oracle.evaluate_bank(w, f0[:1], tau[:1], brk[:1], sky[0], want_k=True)
    b = oracle.evaluate_bank(w, f0[:1], tau[:1], brk[:1], sky[1], want_k=True)
    assert not np.array_equal(a.k, b.k)
    assert np.array_equal(r.k[0::2], np.tile(a.k, (n // 2, 1))) and np.array_equal(r.k[1::2], np.tile(b.k, (n // 2, 1)))


def test_bank_eq1_closed_forms():
    """tests/golden/eq1_closed_forms.txt through the bank entry: one template per row, zero velocity."""
    rows = []
    with open(os.path.join(GOLDEN, "eq1_closed_forms.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if line:
                rows.append(line)
    for f0, tau, n, t, base, g, fgw, x in rows:
        f0, tau, n, t, x = map(float, (f0, tau, n, t, x))
        k = int(x) - 4000
        n_bins = k + 3
        rho = np.zeros((1, n_bins), dtype=np.float32)
        rho[0, k] = 7.0
        w = Workload("one", "f32", rho, 1, n_bins, 500.0, 8.0, np.array([t]), np.zeros((1, 3)), 0.0,
                     np.array([f0]), np.array([tau]), np.array([n]), np.array([[1.0, 0.0, 0.0]]))
        r = oracle.evaluate_bank(w, [f0], [tau], [n], [1.0, 0.0, 0.0], want_k=True)
        assert r.k[0, 0] == k and r.stat[0] == 7.0 and r.n_inband[0] == 1


def test_bank_numpy_twin_and_permutation(cfg1):
    """Independent numpy write on a random bank (np.power for the spin-down factor: bins compared
    where x is not within 1e-6 of a half-integer), and order independence of the templates."""
    w = cfg1
    f0, tau, brk, sky = tcw_inputs.random_bank(600, 500.0, 628.0, 3)
    r = oracle.evaluate_bank(w, f0, tau, brk, sky, want_k=True)
    t = w.timestamps
    g = np.power(t[None, :] / tau[:, None] + 1.0, 1.0 / (1.0 - brk[:, None]))
    D = 1.0 + (sky @ w.velocities.T) / tcw_inputs.C_LIGHT
    x = f0[:, None] * g * D * 8.0
    k = np.rint(x).astype(np.int64) - 4000
    safe = np.abs((x - np.floor(x)) - 0.5) > 1e-6
    assert safe.mean() > 0.999 and np.array_equal(k[safe], r.k[safe])
    ok = (k >= 0) & (k < w.n_bins)
    val = w.spectrogram.astype(np.float64)[np.arange(w.n_sft)[None, :], np.clip(k, 0, w.n_bins - 1)]
    want = np.where(ok, val, 0.0).sum(axis=1)
    clean = safe.all(axis=1)
    assert np.allclose(r.stat[clean], want[clean], rtol=1e-12)
    assert np.array_equal(r.n_inband[clean], ok.sum(axis=1)[clean])
    perm = np.random.default_rng(0).permutation(len(f0))
    rp = oracle.evaluate_bank(w, f0[perm], tau[perm], brk[perm], sky[perm])
    assert np.array_equal(rp.stat, r.stat[perm])


def test_random_bank_generator_ranges():
    f0, tau, brk, sky = tcw_inputs.random_bank(5000, 1000.0, 1200.0, 9)
    assert f0.min() >= 1000 and f0.max() <= 1200 and tau.min() >= 3500 and tau.max() <= 35000
    assert brk.min() >= 3 and brk.max() <= 7 and np.allclose(np.linalg.norm(sky, axis=1), 1.0, atol=1e-12)
    assert abs(sky.mean(axis=0)).max() < 0.05           # isotropic
    f0b, _, _, skyb = tcw_inputs.random_bank(10, 1000.0, 1200.0, 9, sky=sky_vector(1.0, 0.3))
    assert skyb.shape == (1, 3)
