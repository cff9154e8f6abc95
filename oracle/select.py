"""oracle.select -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain definitions of the downstream selection step, after
PAPER.md:79: "a threshold was set on Psi based on the distribution of critical ratios on only
noise using the same amount of templates (Psi_noise max).  That is, an injection was considered
detected if a template close to the injection had Psi > Psi_noise max."

  topk(values, K)            the K largest values, in descending order; equal values in ascending
                             index order (reading Q23: the paper does not order candidates; this is
                             the order that extends "lowest f0 index on ties" of the per-group best)
  select_above(values, thr)  indices i with values[i] > thr, ascending
  noise_max(values)          Psi_noise max = the largest value of a noise-only search (= topk(., 1))

NaN never compares greater than anything and is never selected; -0.0 and +0.0 are equal.
Written with numpy sorting primitives; pinned in tests/test_oracle_select_pins.py against
pure-Python brute force and closed forms.  Imports nothing from the CUDA package.
"""
from __future__ import annotations

import numpy as np


def topk(values, K: int):
    v = np.asarray(values).reshape(-1)
    idx = np.arange(v.size, dtype=np.int64)
    if v.dtype.kind == "f":
        ok = ~np.isnan(v)
        v, idx = v[ok], idx[ok]
    # stable sort of the negated values: descending values, ascending index among equals
    order = np.argsort(-v.astype(np.float64), kind="stable")[:max(0, int(K))]
    return v[order], idx[order]


def select_above(values, threshold):
    v = np.asarray(values).reshape(-1)
    with np.errstate(invalid="ignore"):
        return np.nonzero(v > threshold)[0].astype(np.int64)


def noise_max(values):
    val, _ = topk(values, 1)
    if val.size == 0:
        raise ValueError("no finite value")
    return val[0]
