"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper around oracle/tcw_oracle.c, the plain float64 CPU definition of the tCW track
sum written from the paper.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline
/ --impl reference legs may import this package.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tcw_oracle.c")
_LIB = os.path.join(_HERE, "libtcw_oracle.so")

FORMATS = {"f32": 0, "u8": 1, "bits": 2}
GCC_FLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-Wall"]


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp oracle/tcw_oracle.c -> oracle/libtcw_oracle.so"""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", *GCC_FLAGS, _SRC, "-o", _LIB, "-lquadmath", "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        L.tcwo_spindown.restype = ctypes.c_double
        L.tcwo_spindown.argtypes = [ctypes.c_double] * 4
        L.tcwo_doppler.restype = ctypes.c_double
        L.tcwo_doppler.argtypes = [dp, dp]
        L.tcwo_track_x.restype = ctypes.c_double
        L.tcwo_track_x.argtypes = [ctypes.c_double] * 4
        L.tcwo_bin.restype = ctypes.c_long
        L.tcwo_bin.argtypes = [ctypes.c_double, ctypes.c_long]
        L.tcwo_kmin.restype = ctypes.c_long
        L.tcwo_kmin.argtypes = [ctypes.c_double, ctypes.c_double]
        L.tcwo_num_threads.restype = ctypes.c_int
        L.tcwo_set_num_threads.restype = None
        L.tcwo_set_num_threads.argtypes = [ctypes.c_int]
        L.tcwo_spindown_table.restype = None
        L.tcwo_spindown_table.argtypes = [ctypes.c_int, dp, ctypes.c_double, ctypes.c_int, dp,
                                          ctypes.c_int, dp, dp, ctypes.c_void_p]
        L.tcwo_doppler_table.restype = None
        L.tcwo_doppler_table.argtypes = [ctypes.c_int, dp, ctypes.c_int, dp, dp]
        L.tcwo_eval.restype = ctypes.c_int
        L.tcwo_eval.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_long, ctypes.c_int, ctypes.c_int,
                                ctypes.c_double, ctypes.c_double, dp, dp, ctypes.c_double,
                                ctypes.c_int, dp, ctypes.c_int, dp, ctypes.c_int, dp, ctypes.c_int, dp,
                                ctypes.c_long, ctypes.c_void_p,
                                ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                ctypes.c_void_p, ctypes.c_int]
        L.tcwo_eval_weighted.restype = ctypes.c_int
        L.tcwo_eval_weighted.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_long, ctypes.c_int, ctypes.c_int,
                                         ctypes.c_double, ctypes.c_double, dp, dp, ctypes.c_double,
                                         ctypes.c_int, dp, ctypes.c_int, dp, ctypes.c_int, dp, ctypes.c_int, dp,
                                         ctypes.c_void_p, ctypes.c_double, ctypes.c_double,
                                         ctypes.c_long, ctypes.c_void_p,
                                         ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                         ctypes.c_int]
        L.tcwo_eval_bank.restype = ctypes.c_int
        L.tcwo_eval_bank.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_long, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_double, ctypes.c_double, dp, dp, ctypes.c_double,
                                     ctypes.c_long, dp, dp, dp, dp, ctypes.c_int,
                                     ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.tcwo_best_f64.restype = None
        L.tcwo_best_f64.argtypes = [dp, ctypes.c_long, ctypes.c_int, dp, ctypes.c_void_p]
        L.tcwo_best_i64.restype = None
        L.tcwo_best_i64.argtypes = [ctypes.c_void_p, ctypes.c_long, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().tcwo_num_threads())


def set_num_threads(n: int) -> None:
    lib().tcwo_set_num_threads(int(n))


def spindown(t: float, T0: float, tau: float, n: float) -> float:
    """g = RN(((t - T0)/tau + 1)^(1/(1-n))), eq. (1) PAPER.md:25."""
    return float(lib().tcwo_spindown(t, T0, tau, n))


def doppler(v, nhat) -> float:
    """D = 1 + (v . n-hat)/c, eq. (2) PAPER.md:32."""
    v, nhat = _f64(v), _f64(nhat)
    return float(lib().tcwo_doppler(_dp(v), _dp(nhat)))


def track_x(f0: float, g: float, D: float, T_sft: float) -> float:
    return float(lib().tcwo_track_x(f0, g, D, T_sft))


def bin_index(x: float, k_min: int) -> int:
    return int(lib().tcwo_bin(x, k_min))


def kmin(f_min: float, T_sft: float) -> int:
    return int(lib().tcwo_kmin(f_min, T_sft))


def spindown_table(ts, T0, tau, brk, want_hard: bool = False):
    ts, tau, brk = _f64(ts), _f64(tau), _f64(brk)
    out = np.empty((len(tau), len(brk), len(ts)), dtype=np.float64)
    hard = np.zeros(out.shape, dtype=np.uint8) if want_hard else None
    lib().tcwo_spindown_table(len(ts), _dp(ts), float(T0), len(tau), _dp(tau), len(brk), _dp(brk),
                              _dp(out), hard.ctypes.data if want_hard else None)
    return (out, hard) if want_hard else out


def doppler_table(vel, sky):
    vel, sky = _f64(vel), _f64(sky)
    out = np.empty((len(sky), len(vel)), dtype=np.float64)
    lib().tcwo_doppler_table(len(vel), _dp(vel), len(sky), _dp(sky), _dp(out))
    return out


@dataclass
class OracleResult:
    stat: np.ndarray               # float64 [n_sel] (power) or int64 [n_sel] (counts)
    n_inband: np.ndarray           # int32 [n_sel]
    n_ambig: np.ndarray            # int32 [n_sel]  lookups within 1e-9 bin of a half-integer
    k: np.ndarray | None = None    # int32 [n_sel][n_sft] (INT32_MIN where t_j < T0)


def evaluate(w, sel=None, want_k: bool = False, literal: bool = False) -> OracleResult:
    """Track sums of workload `w` (a tcw_inputs.Workload-like object: attributes spectrogram,
    fmt, n_sft, n_bins, f_min, T_sft, timestamps, velocities, T0, f0, tau, brk, sky) for the
    template linear indices `sel` (None = all), index = ((s*n_tau + a)*n_brk + b)*n_f0 + i."""
    spec = np.ascontiguousarray(w.spectrogram)
    fmt = FORMATS[w.fmt]
    pitch = spec.strides[0]
    ts, vel = _f64(w.timestamps), _f64(w.velocities)
    f0, tau, brk, sky = _f64(w.f0), _f64(w.tau), _f64(w.brk), _f64(w.sky)
    n_templates = len(sky) * len(tau) * len(brk) * len(f0)
    if sel is None:
        n_sel, sel_arr, sel_ptr = n_templates, None, None
    else:
        sel_arr = np.ascontiguousarray(sel, dtype=np.int64)
        n_sel, sel_ptr = len(sel_arr), sel_arr.ctypes.data
    stat_f = np.empty(n_sel, dtype=np.float64)
    stat_i = np.empty(n_sel, dtype=np.int64) if fmt != 0 else None
    n_in = np.empty(n_sel, dtype=np.int32)
    n_amb = np.empty(n_sel, dtype=np.int32)
    k = np.empty((n_sel, w.n_sft), dtype=np.int32) if want_k else None
    rc = lib().tcwo_eval(spec.ctypes.data, fmt, pitch, int(w.n_sft), int(w.n_bins),
                         float(w.f_min), float(w.T_sft), _dp(ts), _dp(vel), float(w.T0),
                         len(f0), _dp(f0), len(tau), _dp(tau), len(brk), _dp(brk), len(sky), _dp(sky),
                         n_sel, sel_ptr, stat_f.ctypes.data,
                         stat_i.ctypes.data if stat_i is not None else None,
                         k.ctypes.data if k is not None else None,
                         n_in.ctypes.data, n_amb.ctypes.data, int(bool(literal)))
    if rc != 0:
        raise ValueError("tcwo_eval: bad arguments")
    return OracleResult(stat_i if stat_i is not None else stat_f, n_in, n_amb, k)


@dataclass
class WeightedResult:
    s: np.ndarray      # float64 [n_sel]  weighted statistic  sum_j w_j * spectrogram[j][k_j]
    w1: np.ndarray     # float64 [n_sel]  sum of the weights of the in-band SFTs
    w2: np.ndarray     # float64 [n_sel]  sum of their squares
    psi: np.ndarray    # float64 [n_sel]  critical ratio, eq. (4)


def evaluate_weighted(w, weights, mean1: float, var1: float, sel=None, literal: bool = False) -> WeightedResult:
    """Weighted statistic and critical ratio (eq. (4)) of workload `w` with
    float32 weights [n_sky][n_sft] (None = all ones) and per-bin noise moments (mean1, var1)."""
    spec = np.ascontiguousarray(w.spectrogram)
    fmt = FORMATS[w.fmt]
    pitch = spec.strides[0]
    ts, vel = _f64(w.timestamps), _f64(w.velocities)
    f0, tau, brk, sky = _f64(w.f0), _f64(w.tau), _f64(w.brk), _f64(w.sky)
    n_templates = len(sky) * len(tau) * len(brk) * len(f0)
    if weights is not None:
        weights = np.ascontiguousarray(weights, dtype=np.float32)
        assert weights.shape == (len(sky), w.n_sft), weights.shape
    if sel is None:
        n_sel, sel_arr, sel_ptr = n_templates, None, None
    else:
        sel_arr = np.ascontiguousarray(sel, dtype=np.int64)
        n_sel, sel_ptr = len(sel_arr), sel_arr.ctypes.data
    out = [np.empty(n_sel, dtype=np.float64) for _ in range(4)]
    rc = lib().tcwo_eval_weighted(spec.ctypes.data, fmt, pitch, int(w.n_sft), int(w.n_bins),
                                  float(w.f_min), float(w.T_sft), _dp(ts), _dp(vel), float(w.T0),
                                  len(f0), _dp(f0), len(tau), _dp(tau), len(brk), _dp(brk), len(sky), _dp(sky),
                                  weights.ctypes.data if weights is not None else None,
                                  float(mean1), float(var1), n_sel, sel_ptr,
                                  *[o.ctypes.data for o in out], int(bool(literal)))
    if rc != 0:
        raise ValueError("tcwo_eval_weighted: bad arguments")
    return WeightedResult(*out)


def evaluate_bank(w, f0, tau, brk, sky, want_k: bool = False) -> OracleResult:
    """Track sums of a template bank (PAPER.md:63 (ii)): per-template f0, tau, brk [n] and sky
    [n][3], or one shared sky vector [3] / [1][3].  Data (spectrogram, timestamps, velocities,
    band, T0) come from the workload-like object `w`."""
    spec = np.ascontiguousarray(w.spectrogram)
    fmt = FORMATS[w.fmt]
    ts, vel = _f64(w.timestamps), _f64(w.velocities)
    f0, tau, brk = _f64(f0), _f64(tau), _f64(brk)
    sky = _f64(sky).reshape(-1, 3)
    n = len(f0)
    assert len(tau) == n and len(brk) == n and len(sky) in (1, n)
    shared = len(sky) == 1
    stat_f = np.empty(n, dtype=np.float64)
    stat_i = np.empty(n, dtype=np.int64) if fmt != 0 else None
    n_in = np.empty(n, dtype=np.int32)
    n_amb = np.empty(n, dtype=np.int32)
    k = np.empty((n, w.n_sft), dtype=np.int32) if want_k else None
    rc = lib().tcwo_eval_bank(spec.ctypes.data, fmt, spec.strides[0], int(w.n_sft), int(w.n_bins),
                              float(w.f_min), float(w.T_sft), _dp(ts), _dp(vel), float(w.T0),
                              n, _dp(f0), _dp(tau), _dp(brk), _dp(sky), int(shared),
                              stat_f.ctypes.data, stat_i.ctypes.data if stat_i is not None else None,
                              k.ctypes.data if k is not None else None, n_in.ctypes.data, n_amb.ctypes.data)
    if rc != 0:
        raise ValueError("tcwo_eval_bank: bad arguments")
    return OracleResult(stat_i if stat_i is not None else stat_f, n_in, n_amb, k)


def best(stat: np.ndarray, n_f0: int):
    """Per group of n_f0 consecutive templates: (max, lowest f0 index attaining it)."""
    stat = np.ascontiguousarray(stat)
    assert stat.size % n_f0 == 0
    n_groups = stat.size // n_f0
    idx = np.empty(n_groups, dtype=np.int32)
    if stat.dtype == np.int64:
        val = np.empty(n_groups, dtype=np.int64)
        lib().tcwo_best_i64(stat.ctypes.data, n_groups, n_f0, val.ctypes.data, idx.ctypes.data)
    else:
        stat = stat.astype(np.float64, copy=False)
        val = np.empty(n_groups, dtype=np.float64)
        lib().tcwo_best_f64(_dp(stat), n_groups, n_f0, _dp(val), idx.ctypes.data)
    return val, idx


def group_templates(w, groups) -> np.ndarray:
    """Linear template indices of whole (sky, tau, n) groups (all f0), for sampled parity."""
    groups = np.asarray(groups, dtype=np.int64)
    n_f0 = len(w.f0)
    return (groups[:, None] * n_f0 + np.arange(n_f0, dtype=np.int64)[None, :]).reshape(-1)
