"""CPU model of the staged kernel's one-FMA bin index, checked against the
defining chain with exact rational arithmetic.  No GPU: this pins the *derivation* -- the fixed-point
layout of the fused multiply-add's result, the error budget |x~ - x| <= 3*x*2^-52 + 2^-32 and the guard
band -- independently of the CUDA code, which tests/test_gpu_round2.py then compares bit for bit with
the defining chain on the device.

The model restates the kernel's arithmetic operation by operation (each a correctly rounded binary64
operation, the FMA with a single rounding, emulated with fractions.Fraction):
    c  = RN(g*Dp)                                     Dp = D*T_sft (T_sft a power of two: exact)
    Q  = RN(RN(RN(RN(f_first*c) - rint(x_first)) + (1/2 + thr + W)) + 1.5*2^20)
    y  = fma(f0 - f_first, c, Q)                      in [2^20, 2^21): one unit in the last place = 2^-32
    high word(y) - 0x41380000 - W + (rint(x_first))   = the bin, unless low word(y) <= 2*thr*2^32
and the oracle's chain x = RN(RN(f0*g)*Dp), k = rint(x) (round half to even)."""
import math
import struct
from fractions import Fraction

import numpy as np

FIX_BASE = 1572864.0          # 1.5 * 2^20
FIX_HC = 0x41380000


def rn(x: Fraction) -> float:
    return float(x)            # Fraction -> float is correctly rounded (nearest, ties to even)


def fma(a: float, b: float, c: float) -> float:
    return rn(Fraction(a) * Fraction(b) + Fraction(c))


def words(y: float):
    bits = struct.unpack("<Q", struct.pack("<d", y))[0]
    return bits >> 32, bits & 0xFFFFFFFF


def chain_bin(f0, g, Dp):
    """the defining chain (bin_lo in csrc/tcw_sum.cuh; lines 4, 7, 8, 9 of the oracle's definition)"""
    x = rn(Fraction(rn(Fraction(f0) * Fraction(g))) * Fraction(Dp))
    return x, int(np.rint(x))


def thr_units_for(x_max: float) -> int:
    """the host's choice (base_params in csrc/tcw_api.cu)"""
    return max(64, math.ceil((4.0 * x_max * 2.0 ** -52 + 2.0 ** -31) * 2.0 ** 32))


def fast_bin(f0, f_first, g, Dp, W, thr_units):
    c = rn(Fraction(g) * Fraction(Dp))
    _, lo_f = chain_bin(f_first, g, Dp)
    fix_add = 0.5 + thr_units * 2.0 ** -32
    q = rn(Fraction(rn(Fraction(f_first) * Fraction(c))) - lo_f)
    q = rn(Fraction(q) + Fraction(fix_add + float(W)))
    q = rn(Fraction(q) + Fraction(FIX_BASE))
    y = fma(rn(Fraction(f0) - Fraction(f_first)), c, q)
    assert 2.0 ** 20 <= y < 2.0 ** 21
    hi, lo = words(y)
    x_fast = Fraction(f0 - f_first) * Fraction(c) + Fraction(f_first) * Fraction(c)     # exact fast value of x
    return hi - FIX_HC - W + lo_f, lo, x_fast


def _cases(rng, n):
    for _ in range(n):
        f_first = float(rng.uniform(20.0, 3000.0))
        f0 = f_first + float(rng.integers(0, 512)) * float(rng.choice([0.0625, 0.125, 0.25, 0.1]))
        g = float(rng.uniform(0.15, 1.0))
        Dp = 8.0 * (1.0 + float(rng.uniform(-1.1e-4, 1.1e-4)))
        yield f0, f_first, g, Dp, int(rng.integers(1200, 58000))


def test_fast_index_equals_the_chain_outside_the_guard_band_and_within_the_error_budget():
    rng = np.random.default_rng(250707816)
    n_guard = 0
    for f0, f_first, g, Dp, W in _cases(rng, 6000):
        x, k = chain_bin(f0, g, Dp)
        thr_units = thr_units_for(3000.0 * 8.0008 * 1.0001)
        kf, lo, x_fast = fast_bin(f0, f_first, g, Dp, W, thr_units)
        # error budget: |x~ - x| <= 3*x*2^-52 (+ the 2^-32 of the fixed-point roundings, which act on y, not on x~)
        assert abs(x_fast - Fraction(x)) <= Fraction(3 * x) * Fraction(1, 2 ** 52)
        if lo <= 2 * thr_units:
            n_guard += 1                    # the kernel hands this lookup to the defining chain
            continue
        assert kf == k, (f0, f_first, g, Dp, W, kf, k, lo)
    assert n_guard <= 2                     # a guard band of 3e-8 bin is hit about once in 3e7 lookups


def test_near_half_integers_are_either_right_or_flagged():
    """Tracks pushed to within 1e-13 .. 1e-7 bin of a rounding boundary, and exactly onto it: the fast
    index is never silently wrong -- it agrees with the chain (which rounds half to even) or sits inside
    the guard band."""
    rng = np.random.default_rng(7)
    thr_units = thr_units_for(3000.0 * 8.0008 * 1.0001)
    flagged = wrong = 0
    for _ in range(3000):
        f_first = float(rng.uniform(500.0, 2900.0))
        g = float(rng.uniform(0.2, 1.0))
        Dp = 8.0 * (1.0 + float(rng.uniform(-1e-4, 1e-4)))
        # choose f0 so that x = f0*g*Dp lands at (integer + 1/2 + eps)
        k = int(f_first * g * Dp) + int(rng.integers(1, 400))
        eps = float(rng.choice([0.0, 1e-13, -1e-13, 1e-11, -1e-11, 1e-9, -1e-9, 2e-8, -2e-8, 1e-7, -1e-7]))
        f0 = (k + 0.5 + eps) / (g * Dp)
        x, kc = chain_bin(f0, g, Dp)
        kf, lo, _ = fast_bin(f0, f_first, g, Dp, 2000, thr_units)
        if lo <= 2 * thr_units:
            flagged += 1
        elif kf != kc:
            wrong += 1
    assert wrong == 0
    assert flagged > 1500                   # everything within 1.5e-8 bin of the boundary is flagged


def test_exact_ties_are_always_flagged():
    """x exactly on a half-integer (g = 1, Dp = 8, f0 = (k + 1/2)/8): the low word is the guard offset itself."""
    thr_units = thr_units_for(24000.0)
    for k in (4001, 4002, 12345, 23999):
        f0 = (k + 0.5) / 8.0
        kf, lo, _ = fast_bin(f0, 500.0, 1.0, 8.0, 1500, thr_units)
        assert lo <= 2 * thr_units
        assert chain_bin(f0, 1.0, 8.0)[1] == (k if k % 2 == 0 else k + 1)      # half to even
