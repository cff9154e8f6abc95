"""Pins for oracle/prep.py (NEXT-3: strain -> Hann SFTs -> normalised power -> number count; no GPU)."""
import math

import numpy as np

from oracle import prep


def test_hann_sinusoid_closed_form():
    """A real sinusoid A cos(2 pi k0 t / N) on a bin centre through the Hann window: |X[k0]| = A N / 4,
    |X[k0 +- 1]| = A N / 8, everything else zero (textbook three-line spectrum of the Hann window)."""
    fs, T, A, k0 = 256.0, 8.0, 3.0, 400
    N = int(fs * T)
    t = np.arange(2 * N)
    x = A * np.cos(2 * np.pi * k0 * t / N)
    P = prep.sft_power(x, fs, T)
    assert P.shape == (2, N // 2 + 1)
    for row in P:
        assert math.isclose(row[k0], (A * N / 4) ** 2, rel_tol=1e-10)
        assert math.isclose(row[k0 - 1], (A * N / 8) ** 2, rel_tol=1e-9)
        assert math.isclose(row[k0 + 1], (A * N / 8) ** 2, rel_tol=1e-9)
        rest = np.delete(row, [k0 - 1, k0, k0 + 1])
        assert rest.max() < 1e-12 * row[k0]


def test_dft_against_direct_sum_and_segmenting():
    """rfft against the defining sum on a tiny segment; a trailing partial segment is dropped; segment j
    uses samples [jN, (j+1)N)."""
    rng = np.random.default_rng(0)
    fs, T = 4.0, 8.0                       # N = 32
    N = 32
    x = rng.standard_normal(3 * N + 5)
    P = prep.sft_power(x, fs, T)
    assert P.shape == (3, N // 2 + 1)
    w = [0.5 - 0.5 * math.cos(2 * math.pi * t / N) for t in range(N)]
    for j in (0, 2):
        for k in (0, 1, 7, 16):
            re = sum(w[t] * x[j * N + t] * math.cos(2 * math.pi * k * t / N) for t in range(N))
            im = -sum(w[t] * x[j * N + t] * math.sin(2 * math.pi * k * t / N) for t in range(N))
            assert math.isclose(P[j, k], re * re + im * im, rel_tol=1e-10, abs_tol=1e-12)


def test_running_median_brute_force():
    rng = np.random.default_rng(1)
    P = rng.standard_exponential((3, 40))
    for W in (1, 3, 9):
        m = prep.running_median(P, W)
        assert m.shape == (3, 40 - W + 1)
        for r in range(3):
            for q in range(40 - W + 1):
                assert m[r, q] == sorted(P[r, q:q + W])[W // 2]


def test_normalisation_scale_invariance_and_band_alignment():
    """rho is invariant under scaling of the strain; rho[k] uses the window centred on bin k_min + k."""
    rng = np.random.default_rng(2)
    fs, T, W = 64.0, 8.0, 5
    x = rng.standard_normal(4 * 512)
    rho, nu = prep.prepare(x, fs, T, 8.0, 100, W, 1.6)          # k_min = 64
    rho2, _ = prep.prepare(1000.0 * x, fs, T, 8.0, 100, W, 1.6)
    assert np.allclose(rho, rho2, rtol=1e-12)
    P = prep.sft_power(x, fs, T)
    for k in (0, 57, 99):
        med = sorted(P[1, 64 + k - 2: 64 + k + 3])[2]
        assert math.isclose(rho[1, k], P[1, 64 + k] * math.log(2.0) / med, rel_tol=1e-13)
    assert np.array_equal(nu, (rho > 1.6).astype(np.uint8))


def test_white_noise_gives_exp1_statistics():
    """Gaussian white noise: rho ~ Exp(1): mean 1 and P(rho > 1.6) = exp(-1.6), within sampling error
    (the finite-window median adds a small positive bias to the mean, well inside the bound used)."""
    rng = np.random.default_rng(3)
    fs, T = 512.0, 8.0
    x = rng.standard_normal(40 * 4096)
    rho, nu = prep.prepare(x, fs, T, 50.0, 1200, 101, 1.6)
    assert rho.shape == (40, 1200)
    assert abs(rho.mean() - 1.0) < 0.03
    assert abs(nu.mean() - math.exp(-1.6)) < 0.01
    assert abs(np.median(rho) - math.log(2.0)) < 0.02
