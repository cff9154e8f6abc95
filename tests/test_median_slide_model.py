"""CPU model of the running-median slide rule of prep_normalise_kernel (csrc/tcw_prep.cuh), checked against
brute force on data with heavy ties.

The kernel keeps the median mu of a sliding window of W = 2h + 1 keys (float bits of non-negative numbers, so
unsigned order = value order, all below 2^31) and per slide scans the window ONCE for three things:
the largest key below mu (as the unsigned maximum of x - mu), the smallest key above mu (as the unsigned minimum
of x - mu - 1) and ONE count C = #(x < mu + s) (from the sign bit of x - mu - s).  The other count K is carried
incrementally, and is re-seeded exactly whenever the median moves: down to pred => LE(pred) = L, so K := L, s := 0;
up to succ => L(succ) = LE, so K := LE, s := 1.  This file restates that rule in Python integers (mod 2^32 where
the kernel wraps) and compares every median with numpy's sort.  It pins the RULE (ties are what a wrong
re-seeding would get wrong); tests/test_gpu_prep.py compares the kernel itself with oracle/prep.py on the GPU.
(reading Q24: rho = P ln 2 / running median.)
"""
import numpy as np
import pytest

M32 = 0xFFFFFFFF


def slide_medians(keys, W):
    """medians of every window of W consecutive keys, by the kernel's rule"""
    h = (W - 1) // 2
    n = len(keys) - W + 1
    out = []
    mu = sorted(keys[:W])[h]                        # the kernel's bitwise binary search finds exactly this
    K = sum(1 for x in keys[:W] if x <= mu)         # LE of the first window
    s = 0
    out.append(mu)
    for k in range(1, n):
        win = keys[k:k + W]
        x_out, x_in = keys[k - 1], keys[k + W - 1]
        mk = mu + 1 - s                             # K = #(x < mk)
        K += int(x_in < mk) - int(x_out < mk)
        maxd, mine, C = 0, M32, 0
        for x in win:
            maxd = max(maxd, (x - mu) & M32)
            mine = min(mine, (x - mu - 1) & M32)
            C += ((x - mu - s) & M32) >> 31
        L, LE = (K, C) if s else (C, K)
        assert L == sum(1 for x in win if x < mu) and LE == sum(1 for x in win if x <= mu)
        if L > h:
            mu = (mu + maxd) & M32
            K, s = L, 0
        elif LE <= h:
            mu = (mu + 1 + mine) & M32
            K, s = LE, 1
        out.append(mu)
    return out


def brute(keys, W):
    h = (W - 1) // 2
    return [int(np.sort(keys[k:k + W])[h]) for k in range(len(keys) - W + 1)]


@pytest.mark.parametrize("W", [1, 3, 5, 11, 101])
@pytest.mark.parametrize("levels", [2, 3, 7, 1000, 2 ** 31 - 1])
def test_slide_rule_matches_brute_force_with_ties(W, levels):
    rng = np.random.default_rng(1000 * W + levels % 997)
    n = 400 + W
    keys = [int(v) for v in rng.integers(0, levels, size=n)]
    assert slide_medians(keys, W) == brute(np.array(keys, dtype=np.int64), W)


def test_slide_rule_on_float_bits():
    rng = np.random.default_rng(7)
    p = rng.exponential(1.0, size=700).astype(np.float32)
    p[::5] = p[1::5][: len(p[::5])]                 # exact duplicates of neighbours
    p[100:140] = 0.0                                # a run of zeros (key 0)
    keys = [int(v) for v in p.view(np.uint32)]
    got = slide_medians(keys, 101)
    want = brute(np.array(keys, dtype=np.int64), 101)
    assert got == want
    # and the keys order like the values
    assert np.array_equal(np.array(got, dtype=np.uint32).view(np.float32),
                          np.array([np.sort(p[k:k + 101])[50] for k in range(len(p) - 100)], dtype=np.float32))


def test_monotone_and_constant_inputs():
    for keys in ([5] * 300, list(range(300)), list(range(300, 0, -1)), [0, 2 ** 31 - 1] * 150):
        assert slide_medians(keys, 21) == brute(np.array(keys, dtype=np.int64), 21)
