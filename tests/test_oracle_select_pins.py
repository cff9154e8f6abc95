"""Pins for oracle/select.py (NEXT-4 selection; no GPU): brute force and closed forms."""
import math

import numpy as np

from oracle import select


def _brute_topk(vals, K):
    """Pure-Python selection by repeated maximum (first maximum wins = lowest index on ties)."""
    left = [(float(v), i) for i, v in enumerate(vals) if not math.isnan(float(v))]
    out = []
    while left and len(out) < K:
        best = 0
        for q in range(1, len(left)):
            if left[q][0] > left[best][0]:
                best = q
        out.append(left.pop(best))
    return [v for v, _ in out], [i for _, i in out]


def test_topk_matches_brute_force_with_ties_nan_inf_and_zeros():
    rng = np.random.default_rng(0)
    for n, K in ((1, 1), (7, 3), (50, 50), (50, 80), (300, 17)):
        v = rng.integers(-4, 5, size=n).astype(np.float32)        # many ties
        if n >= 50:
            v[[3, 11]] = np.nan
            v[5], v[9] = np.inf, -np.inf
            v[20], v[21] = -0.0, 0.0
        val, idx = select.topk(v, K)
        bv, bi = _brute_topk(v, K)
        assert list(idx) == bi and [float(x) for x in val] == bv
        assert len(idx) == min(K, int(np.sum(~np.isnan(v))))


def test_topk_closed_form_permutation():
    """values = a permutation of 0..n-1: the K largest are n-1, n-2, ... at the positions the
    permutation put them."""
    n, K = 1000, 25
    perm = np.random.default_rng(1).permutation(n)
    v = perm.astype(np.float32)
    val, idx = select.topk(v, K)
    assert list(val) == [float(n - 1 - q) for q in range(K)]
    inv = np.argsort(perm)
    assert list(idx) == [int(inv[n - 1 - q]) for q in range(K)]


def test_topk_integer_values():
    v = np.array([3, 9, 9, -2, 9, 0], dtype=np.int32)
    val, idx = select.topk(v, 4)
    assert list(val) == [9, 9, 9, 3] and list(idx) == [1, 2, 4, 0]


def test_select_above_and_noise_max():
    v = np.array([0.5, np.nan, 2.0, -1.0, 2.0, 3.5, -0.0], dtype=np.float32)
    assert list(select.select_above(v, 2.0)) == [5]
    assert list(select.select_above(v, 1.9999)) == [2, 4, 5]
    assert list(select.select_above(v, -0.0)) == [0, 2, 4, 5]      # -0.0 is not > 0.0
    assert select.noise_max(v) == np.float32(3.5)
    # the detection rule of PAPER.md:79: candidates are exactly those above the noise-only maximum
    noise = np.random.default_rng(2).standard_normal(5000).astype(np.float32)
    sig = noise.copy()
    sig[[7, 4000]] += 9.0
    thr = select.noise_max(noise)
    assert list(select.select_above(sig, thr)) == [7, 4000]
    assert select.select_above(noise, thr).size == 0
