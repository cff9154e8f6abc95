"""oracle.prep -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain float64 definition of the data preparation upstream of the track sum (SURVEY.md section
8(f) NEXT-3), after PAPER.md:51: "The data used in this study are 8-second Han-windowed Short
Fourier Transforms (SFTs), which are processed into either normalized power rho_j or number count
nu_j as described by Oliver et al. [14]."  Ref. [14] is not available; the normalisation below is
reading Q24 of DESIGN.md (the standard running-median noise-floor estimate):

  1  segment j = samples [j*N, (j+1)*N), N = fs * T_sft (no overlap; a trailing partial segment is dropped)
  2  w[t]  = 0.5 - 0.5 cos(2 pi t / N), t = 0..N-1                      (Hann window, DFT-even form)
  3  X_j[k] = sum_t w[t] x[j*N + t] exp(-2 pi i k t / N)                 (numpy.fft.rfft, float64)
  4  P_j[k] = |X_j[k]|^2
  5  m_j[k] = median of P_j[k-h .. k+h], h = (W-1)/2, W odd             (running median along frequency)
  6  rho_j[k] = P_j[k] * ln 2 / m_j[k]        (the median of an exponential variable is ln 2 times its
                                               mean, so rho has mean 1 in Gaussian noise: rho ~ Exp(1))
  7  nu_j[k] = 1 if rho_j[k] > threshold else 0
for the band bins k = k_min .. k_min + n_bins - 1, k_min = rint(f_min * T_sft); the band must leave
h bins on both sides inside 0..N/2.  Pinned in tests/test_oracle_prep_pins.py.
Imports nothing from the CUDA package.
"""
from __future__ import annotations

import math

import numpy as np


def hann(N: int) -> np.ndarray:
    t = np.arange(N, dtype=np.float64)
    return 0.5 - 0.5 * np.cos(2.0 * np.pi * t / N)


def sft_power(strain, fs: float, T_sft: float) -> np.ndarray:
    """Steps 1-4: float64 [n_seg][N/2 + 1]."""
    N = int(round(fs * T_sft))
    x = np.asarray(strain, dtype=np.float64)
    n_seg = len(x) // N
    seg = x[: n_seg * N].reshape(n_seg, N) * hann(N)[None, :]
    X = np.fft.rfft(seg, axis=1)
    return X.real ** 2 + X.imag ** 2


def running_median(P: np.ndarray, W: int) -> np.ndarray:
    """Step 5 along the last axis: output[..., q] = median(P[..., q : q + W]) (valid positions only)."""
    win = np.lib.stride_tricks.sliding_window_view(P, W, axis=-1)
    return np.median(win, axis=-1)


def prepare(strain, fs: float, T_sft: float, f_min: float, n_bins: int, W: int, threshold: float):
    """Steps 1-7.  Returns (rho float64 [n_seg][n_bins], nu uint8 [n_seg][n_bins])."""
    if W % 2 != 1:
        raise ValueError("W must be odd")
    h = (W - 1) // 2
    k_min = int(round(f_min * T_sft))
    P = sft_power(strain, fs, T_sft)
    if k_min - h < 0 or k_min + n_bins + h > P.shape[1]:
        raise ValueError("band plus median half-window does not fit 0..N/2")
    band = P[:, k_min - h: k_min + n_bins + h]
    m = running_median(band, W)
    rho = P[:, k_min: k_min + n_bins] * math.log(2.0) / m
    return rho, (rho > threshold).astype(np.uint8)
