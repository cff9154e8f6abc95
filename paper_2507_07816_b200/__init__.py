"""paper_2507_07816_b200 -- thin Python binding of libtcw.so (include/tcw.h).

Argument marshalling only: every step of the tCW track sum (eqs. (1)-(2),
PAPER.md:57) runs in the CUDA kernels under csrc/.  PyTorch appears here for device memory and
streams.  There is no CPU fallback: if the library cannot be loaded, or no CUDA device is
usable, the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

__all__ = [
    "TcwError", "Handle", "Grid", "load_library", "library_path", "shard_groups", "split_groups", "measure_peaks",
    "TCW_F32_POWER", "TCW_U8_COUNT", "TCW_BIT_COUNT", "FORMATS",
]

TCW_OK, TCW_EINVAL, TCW_ENOMEM, TCW_ECUDA, TCW_EUNSUPPORTED, TCW_EINTERNAL = 0, -1, -2, -3, -4, -5
TCW_F32_POWER, TCW_U8_COUNT, TCW_BIT_COUNT = 0, 1, 2
TCW_OPT_KERNEL, TCW_OPT_TIMING, TCW_OPT_F0_PER_LANE, TCW_OPT_STAGES, TCW_OPT_SKY_BLOCK = 0, 1, 2, 3, 4
TCW_OPT_CHUNK_ROWS = 5
TCW_OPT_EXACT_INDEX = 6
TCW_OPT_GENERAL_F0 = 7
TCW_OPT_ROW_COPIES = 8
TCW_OPT_DEBUG_SHRINK_SLOT = 100
TCW_OPT_DEBUG_FAIL_WAIT = 101
TCW_OPT_DEBUG_CHUNK_SCRATCH = 102
KERNELS = {"auto": 0, "gather": 1, "staged": 2, "skyblock": 3}
FORMATS = {"f32": TCW_F32_POWER, "u8": TCW_U8_COUNT, "bits": TCW_BIT_COUNT}

EXPORTS = (
    "tcw_create", "tcw_create_async", "tcw_upload_wait", "tcw_search", "tcw_search_groups", "tcw_split_groups", "tcw_check", "tcw_measure_peaks", "tcw_search_host", "tcw_search_weighted", "tcw_search_bank", "tcw_get_counter", "tcw_topk", "tcw_select_above", "tcw_select_above_static", "tcw_prepare", "tcw_destroy", "tcw_last_error",
    "tcw_track_indices", "tcw_tables", "tcw_set_option", "tcw_get_timing", "tcw_get_info",
)


class TcwError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"tcw error {code}: {message}")
        self.code = code


class _CGrid(ctypes.Structure):
    _fields_ = [
        ("T0", ctypes.c_double),
        ("n_f0", ctypes.c_int), ("f0", ctypes.POINTER(ctypes.c_double)),
        ("n_tau", ctypes.c_int), ("tau", ctypes.POINTER(ctypes.c_double)),
        ("n_brk", ctypes.c_int), ("brk", ctypes.POINTER(ctypes.c_double)),
        ("n_sky", ctypes.c_int), ("sky", ctypes.POINTER(ctypes.c_double)),
    ]


class _CBank(ctypes.Structure):
    _fields_ = [("T0", ctypes.c_double), ("n", ctypes.c_long),
                ("f0", ctypes.POINTER(ctypes.c_double)), ("tau", ctypes.POINTER(ctypes.c_double)),
                ("brk", ctypes.POINTER(ctypes.c_double)), ("sky", ctypes.POINTER(ctypes.c_double)),
                ("sky_shared", ctypes.c_int)]


class _CPrep(ctypes.Structure):
    _fields_ = [("fs", ctypes.c_double), ("T_sft", ctypes.c_double), ("f_min", ctypes.c_double),
                ("n_bins", ctypes.c_int), ("median_bins", ctypes.c_int), ("threshold", ctypes.c_double)]


class _CWeighting(ctypes.Structure):
    _fields_ = [("weights", ctypes.c_void_p), ("mean1", ctypes.c_double), ("var1", ctypes.c_double)]


_lib = None


def library_path() -> str:
    return _build.LIB


def load_library(rebuild: bool = False) -> ctypes.CDLL:
    """dlopen libtcw.so (building it with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is not None and not rebuild:
        return _lib
    path = _build.build(force=rebuild)
    L = ctypes.CDLL(path)
    vp, dp, ci, cl = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_long
    L.tcw_create.restype = ci
    L.tcw_create.argtypes = [ctypes.POINTER(vp), vp, ci, cl, ci, ci, ctypes.c_double, ctypes.c_double, dp, dp, vp]
    L.tcw_create_async.restype = ci
    L.tcw_create_async.argtypes = L.tcw_create.argtypes
    L.tcw_upload_wait.restype = ci
    L.tcw_upload_wait.argtypes = [vp]
    L.tcw_search.restype = ci
    L.tcw_search.argtypes = [vp, ctypes.POINTER(_CGrid), vp, vp, vp]
    L.tcw_search_groups.restype = ci
    L.tcw_search_groups.argtypes = [vp, ctypes.POINTER(_CGrid), cl, cl, vp, vp, vp]
    L.tcw_split_groups.restype = ci
    L.tcw_split_groups.argtypes = [ci, ci, cl, cl, vp, ctypes.POINTER(ci)]
    L.tcw_measure_peaks.restype = ci
    L.tcw_measure_peaks.argtypes = [dp, ci, vp]
    L.tcw_check.restype = ci
    L.tcw_check.argtypes = [vp]
    L.tcw_search_host.restype = ci
    L.tcw_search_host.argtypes = [vp, ctypes.POINTER(_CGrid), vp, vp, vp]
    L.tcw_search_weighted.restype = ci
    L.tcw_search_weighted.argtypes = [vp, ctypes.POINTER(_CGrid), ctypes.POINTER(_CWeighting), vp, vp, vp, vp]
    L.tcw_search_bank.restype = ci
    L.tcw_search_bank.argtypes = [vp, ctypes.POINTER(_CBank), vp, vp, vp, vp]
    L.tcw_get_counter.restype = ci
    L.tcw_get_counter.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_longlong)]
    L.tcw_topk.restype = ci
    L.tcw_topk.argtypes = [vp, vp, ci, cl, ci, vp, vp, vp, vp]
    L.tcw_select_above.restype = ci
    L.tcw_select_above.argtypes = [vp, vp, ci, cl, ctypes.c_double, cl, vp, vp, vp]
    L.tcw_select_above_static.restype = ci
    L.tcw_select_above_static.argtypes = [vp, ci, cl, ctypes.c_double, cl, vp, vp, vp]
    L.tcw_prepare.restype = ci
    L.tcw_prepare.argtypes = [vp, cl, ctypes.POINTER(_CPrep), ci, vp, cl, ctypes.POINTER(ci), vp]
    L.tcw_destroy.restype = ci
    L.tcw_destroy.argtypes = [vp]
    L.tcw_last_error.restype = ctypes.c_char_p
    L.tcw_last_error.argtypes = []
    L.tcw_track_indices.restype = ci
    L.tcw_track_indices.argtypes = [vp, ctypes.POINTER(_CGrid), cl, ctypes.POINTER(cl), vp, vp]
    L.tcw_tables.restype = ci
    L.tcw_tables.argtypes = [vp, dp, dp, vp]
    L.tcw_set_option.restype = ci
    L.tcw_set_option.argtypes = [vp, ci, cl]
    L.tcw_get_timing.restype = ci
    L.tcw_get_timing.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ci)]
    L.tcw_get_info.restype = ci
    L.tcw_get_info.argtypes = [vp, ctypes.POINTER(cl)]
    _lib = L
    return L


def _check(rc: int):
    if rc != TCW_OK:
        raise TcwError(rc, load_library().tcw_last_error().decode("utf-8", "replace"))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


@dataclass
class Grid:
    """The cubic-lattice template bank as explicit axes; mirrors tcw_grid."""
    f0: np.ndarray
    tau: np.ndarray
    brk: np.ndarray
    sky: np.ndarray            # [n_sky][3]
    T0: float = 0.0

    def __post_init__(self):
        self.f0, self.tau, self.brk = _f64(self.f0), _f64(self.tau), _f64(self.brk)
        self.sky = _f64(self.sky).reshape(-1, 3)

    @classmethod
    def of(cls, w) -> "Grid":
        """From any object with attributes f0, tau, brk, sky, T0 (e.g. tcw_inputs.Workload)."""
        return cls(w.f0, w.tau, w.brk, w.sky, float(w.T0))

    @property
    def n_groups(self) -> int:
        return len(self.sky) * len(self.tau) * len(self.brk)

    @property
    def n_templates(self) -> int:
        return self.n_groups * len(self.f0)

    def _c(self) -> _CGrid:
        return _CGrid(float(self.T0), len(self.f0), _dp(self.f0), len(self.tau), _dp(self.tau),
                      len(self.brk), _dp(self.brk), len(self.sky), _dp(self.sky))


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class Handle:
    """tcw_create / tcw_search / tcw_destroy with the same argument meaning as include/tcw.h."""

    def __init__(self, spectrogram, fmt, n_bins: int, f_min: float, T_sft: float, timestamps, velocities,
                 stream=None, async_upload: bool = False):
        """`spectrogram`: a CUDA torch tensor, or a host numpy array / CPU torch tensor, 2-D,
        SFT-major, dtype float32 (fmt "f32"), uint8 ("u8") or int32/uint32 words ("bits")."""
        import torch
        L = load_library()
        self._h = ctypes.c_void_p()
        self.fmt = FORMATS[fmt] if isinstance(fmt, str) else int(fmt)
        if isinstance(spectrogram, np.ndarray):
            spec = np.ascontiguousarray(spectrogram)
            ptr, pitch, n_sft = spec.ctypes.data, spec.strides[0], spec.shape[0]
        else:
            spec = spectrogram if spectrogram.stride(-1) == 1 else spectrogram.contiguous()
            ptr, pitch, n_sft = spec.data_ptr(), spec.stride(0) * spec.element_size(), spec.shape[0]
            if spec.is_cuda:
                torch.cuda.set_device(spec.device)
        ts, vel = _f64(timestamps), _f64(velocities)
        if ts.shape != (n_sft,) or vel.shape != (n_sft, 3):
            raise ValueError("timestamps must be [n_sft] and velocities [n_sft][3]")
        self.n_sft, self.n_bins = int(n_sft), int(n_bins)
        self._keep = spec if async_upload else None     # tcw_create_async reads the host rows after returning
        create = L.tcw_create_async if async_upload else L.tcw_create
        _check(create(ctypes.byref(self._h), ptr, self.fmt, pitch, self.n_sft, self.n_bins,
                            float(f_min), float(T_sft), _dp(ts), _dp(vel), _stream_ptr(stream)))

    @classmethod
    def from_workload(cls, w, device="cuda", host: bool = False, stream=None) -> "Handle":
        """Bind a tcw_inputs.Workload-like object.  host=False first moves the spectrogram to
        `device` with torch; host=True hands the host array to tcw_create, which copies it."""
        import torch
        spec = w.spectrogram
        if not host:
            arr = np.ascontiguousarray(spec)
            if arr.dtype == np.uint32:
                arr = arr.view(np.int32)
            spec = torch.from_numpy(arr).to(device)
        return cls(spec, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities, stream=stream)

    # ------------------------------------------------------------------ the path
    @property
    def stat_dtype(self):
        import torch
        return torch.float32 if self.fmt == TCW_F32_POWER else torch.int32

    def search(self, grid: Grid, out_stat=None, out_best=None, want_stat: bool = True, want_best: bool = True,
               stream=None):
        """tcw_search.  Returns (stat, best): stat a CUDA tensor [n_sky][n_tau][n_brk][n_f0]
        (float32 or int32), best a CUDA int32 tensor [n_groups][2] whose column 0 holds the
        statistic's bits (view as float32 for the power format) and column 1 the f0 index.
        Asynchronous: synchronise the stream before reading."""
        import torch
        L = load_library()
        dev = torch.device("cuda", torch.cuda.current_device())
        if out_stat is None and want_stat:
            out_stat = torch.empty((len(grid.sky), len(grid.tau), len(grid.brk), len(grid.f0)),
                                   dtype=self.stat_dtype, device=dev)
        if out_best is None and want_best:
            out_best = torch.empty((grid.n_groups, 2), dtype=torch.int32, device=dev)
        cg = grid._c()
        _check(L.tcw_search(self._h, ctypes.byref(cg),
                            out_stat.data_ptr() if out_stat is not None else None,
                            out_best.data_ptr() if out_best is not None else None, _stream_ptr(stream)))
        return out_stat, out_best

    def search_groups(self, grid: Grid, group_begin: int, group_end: int, out_stat=None, out_best=None,
                      want_stat: bool = True, want_best: bool = True, stream=None):
        """tcw_search_groups: the groups [group_begin, group_end) of the grid's flattened
        (sky, tau, n) index.  Returns (stat [n][n_f0], best [n][2]) for those groups.  Asynchronous."""
        import torch
        L = load_library()
        dev = torch.device("cuda", torch.cuda.current_device())
        n = int(group_end) - int(group_begin)
        if out_stat is None and want_stat:
            out_stat = torch.empty((max(n, 0), len(grid.f0)), dtype=self.stat_dtype, device=dev)
        if out_best is None and want_best:
            out_best = torch.empty((max(n, 0), 2), dtype=torch.int32, device=dev)
        if n == 0 and 0 <= int(group_begin) <= grid.n_groups:
            return out_stat, out_best       # a rank with no groups (world_size > n_groups) has nothing to launch
        cg = grid._c()
        _check(L.tcw_search_groups(self._h, ctypes.byref(cg), int(group_begin), int(group_end),
                                   out_stat.data_ptr() if out_stat is not None else None,
                                   out_best.data_ptr() if out_best is not None else None, _stream_ptr(stream)))
        return out_stat, out_best

    def check(self):
        """tcw_check: synchronise and raise TcwError(TCW_EINTERNAL) if the last search was invalid."""
        _check(load_library().tcw_check(self._h))

    def search_weighted(self, grid: Grid, weights, mean1: float, var1: float, out_psi=None, out_stat=None,
                        out_best=None, want_psi: bool = True, want_stat: bool = True, want_best: bool = True,
                        stream=None):
        """tcw_search_weighted.  `weights`: None (all ones), a host numpy float32 array or a CUDA
        float32 tensor, [n_sky][n_sft].  Returns (psi, stat, best): float32 CUDA tensors
        [n_sky][n_tau][n_brk][n_f0] and an int32 tensor [n_groups][2] (column 0: bits of the float32
        maximum of Psi, column 1: f0 index).  Asynchronous."""
        import torch
        L = load_library()
        dev = torch.device("cuda", torch.cuda.current_device())
        shape = (len(grid.sky), len(grid.tau), len(grid.brk), len(grid.f0))
        if out_psi is None and want_psi:
            out_psi = torch.empty(shape, dtype=torch.float32, device=dev)
        if out_stat is None and want_stat:
            out_stat = torch.empty(shape, dtype=torch.float32, device=dev)
        if out_best is None and want_best:
            out_best = torch.empty((grid.n_groups, 2), dtype=torch.int32, device=dev)
        if weights is None:
            wptr = None
        elif isinstance(weights, np.ndarray):
            weights = np.ascontiguousarray(weights, dtype=np.float32)
            wptr = weights.ctypes.data
        else:
            weights = weights.contiguous()
            if weights.dtype != torch.float32:
                raise ValueError("weights must be float32")
            wptr = weights.data_ptr()
        if weights is not None and tuple(weights.shape) != (len(grid.sky), self.n_sft):
            raise ValueError("weights must be [n_sky][n_sft]")
        cg = grid._c()
        cw = _CWeighting(wptr, float(mean1), float(var1))
        _check(L.tcw_search_weighted(self._h, ctypes.byref(cg), ctypes.byref(cw),
                                     out_psi.data_ptr() if out_psi is not None else None,
                                     out_stat.data_ptr() if out_stat is not None else None,
                                     out_best.data_ptr() if out_best is not None else None, _stream_ptr(stream)))
        return out_psi, out_stat, out_best

    def search_bank(self, f0, tau, brk, sky, T0: float = 0.0, out_stat=None, want_inband: bool = True,
                    want_k: bool = False, stream=None):
        """tcw_search_bank: per-template f0, tau, brk [n] and sky [n][3], or one shared vector
        ([3] / [1][3]).  Returns (stat [n], n_inband [n] or None, k [n][n_sft] or None) as CUDA
        tensors.  Asynchronous."""
        import torch
        L = load_library()
        f0, tau, brk = _f64(f0), _f64(tau), _f64(brk)
        sky = _f64(sky).reshape(-1, 3)
        n = len(f0)
        if len(tau) != n or len(brk) != n or len(sky) not in (1, n):
            raise ValueError("bank arrays must have equal lengths (sky: [n][3] or one vector)")
        shared = len(sky) == 1
        dev = torch.device("cuda", torch.cuda.current_device())
        if out_stat is None:
            out_stat = torch.empty(n, dtype=self.stat_dtype, device=dev)
        inband = torch.empty(n, dtype=torch.int32, device=dev) if want_inband else None
        k = torch.empty((n, self.n_sft), dtype=torch.int32, device=dev) if want_k else None
        cb = _CBank(float(T0), n, _dp(f0), _dp(tau), _dp(brk), _dp(sky), int(shared))
        _check(L.tcw_search_bank(self._h, ctypes.byref(cb), out_stat.data_ptr(),
                                 inband.data_ptr() if inband is not None else None,
                                 k.data_ptr() if k is not None else None, _stream_ptr(stream)))
        return out_stat, inband, k

    @staticmethod
    def _sel_dtype(values) -> int:
        import torch
        if values.dtype == torch.float32:
            return 0
        if values.dtype == torch.int32:
            return 1
        raise ValueError("values must be a float32 or int32 CUDA tensor")

    def topk(self, values, K: int, stream=None):
        """tcw_topk over a CUDA tensor of statistics (flattened).  Returns (val [K], idx [K] int64,
        count int32 scalar tensor); only the first `count` entries are meaningful.  Asynchronous."""
        import torch
        v = values.contiguous().view(-1)
        out_val = torch.empty(K, dtype=v.dtype, device=v.device)
        out_idx = torch.empty(K, dtype=torch.int64, device=v.device)
        out_cnt = torch.zeros((), dtype=torch.int32, device=v.device)
        _check(load_library().tcw_topk(self._h, v.data_ptr(), self._sel_dtype(v), v.numel(), int(K),
                                       out_val.data_ptr(), out_idx.data_ptr(), out_cnt.data_ptr(), _stream_ptr(stream)))
        return out_val, out_idx, out_cnt

    def select_above(self, values, threshold: float, capacity: int, stream=None):
        """tcw_select_above: (idx [capacity] int64, count int64 scalar tensor).  Asynchronous."""
        import torch
        v = values.contiguous().view(-1)
        out_idx = torch.empty(max(capacity, 1), dtype=torch.int64, device=v.device)
        out_cnt = torch.zeros((), dtype=torch.int64, device=v.device)
        _check(load_library().tcw_select_above(self._h, v.data_ptr(), self._sel_dtype(v), v.numel(), float(threshold),
                                               int(capacity), out_idx.data_ptr() if capacity > 0 else None,
                                               out_cnt.data_ptr(), _stream_ptr(stream)))
        return out_idx[:capacity], out_cnt

    def counter(self, which: int = 0) -> int:
        """tcw_get_counter (0: bank lookups decided by the defining chain in the last bank search)."""
        v = ctypes.c_longlong(0)
        _check(load_library().tcw_get_counter(self._h, int(which), ctypes.byref(v)))
        return int(v.value)

    def search_host(self, grid: Grid, out_stat: np.ndarray | None = None, out_best: np.ndarray | None = None,
                    want_stat: bool = True, stream=None):
        """tcw_search_host: results land in host numpy arrays; synchronous."""
        L = load_library()
        if out_stat is None and want_stat:
            out_stat = np.empty((len(grid.sky), len(grid.tau), len(grid.brk), len(grid.f0)),
                                dtype=np.float32 if self.fmt == TCW_F32_POWER else np.int32)
        if out_best is None:
            out_best = np.empty((grid.n_groups, 2), dtype=np.int32)
        cg = grid._c()
        _check(L.tcw_search_host(self._h, ctypes.byref(cg),
                                 out_stat.ctypes.data if out_stat is not None else None,
                                 out_best.ctypes.data, _stream_ptr(stream)))
        return out_stat, out_best

    def best_fields(self, best):
        """Split a best array ([n_groups][2] int32, torch or numpy) into (stat, f0_index)."""
        if isinstance(best, np.ndarray):
            stat = best[:, 0].copy().view(np.float32) if self.fmt == TCW_F32_POWER else best[:, 0].copy()
            return stat, best[:, 1].copy()
        b = best.cpu().numpy()
        return self.best_fields(b)

    # ------------------------------------------------------------------ inspection
    def track_indices(self, grid: Grid, sel, stream=None):
        """tcw_track_indices: int32 CUDA tensor [n_sel][n_sft] of bin indices k_j."""
        import torch
        L = load_library()
        sel = np.ascontiguousarray(sel, dtype=np.int64)
        out = torch.empty((len(sel), self.n_sft), dtype=torch.int32, device="cuda")
        cg = grid._c()
        _check(L.tcw_track_indices(self._h, ctypes.byref(cg), len(sel),
                                   sel.ctypes.data_as(ctypes.POINTER(ctypes.c_long)), out.data_ptr(),
                                   _stream_ptr(stream)))
        return out

    def tables(self, grid: Grid, stream=None):
        """(g [n_tau][n_brk][n_sft], D [n_sky][n_sft]) of the last search, as host float64 arrays."""
        L = load_library()
        g = np.empty((len(grid.tau), len(grid.brk), self.n_sft), dtype=np.float64)
        d = np.empty((len(grid.sky), self.n_sft), dtype=np.float64)
        _check(L.tcw_tables(self._h, _dp(g), _dp(d), _stream_ptr(stream)))
        return g, d

    def upload_wait(self):
        """tcw_upload_wait: block until an asynchronous upload (async_upload=True) has arrived."""
        _check(load_library().tcw_upload_wait(self._h))

    def set_option(self, key: int, value: int):
        _check(load_library().tcw_set_option(self._h, int(key), int(value)))

    def timing(self):
        """Average device milliseconds per search since timing was enabled or last read:
        ((tables, sum kernel, best kernel, whole call), searches averaged)."""
        ms = (ctypes.c_float * 4)()
        n = ctypes.c_int(0)
        _check(load_library().tcw_get_timing(self._h, ms, ctypes.byref(n)))
        return tuple(float(x) for x in ms), int(n.value)

    def info(self, check: bool = True) -> dict:
        """tcw_get_info.  Raises TcwError(TCW_EINTERNAL) if the device status word is set, unless
        check=False (the dict's "status" then carries the word)."""
        v = (ctypes.c_long * 12)()
        rc = load_library().tcw_get_info(self._h, v)
        if rc != TCW_OK and (check or rc != TCW_EINTERNAL):
            _check(rc)
        return dict(kernel={1: "gather", 2: "staged", 3: "skyblock", 4: "bank"}.get(v[0], "?"), tile=int(v[1]), ctas=int(v[2]),
                    smem_bytes=int(v[3]), status=int(v[4]), launches=int(v[5]), stages=int(v[6]),
                    sky_block=int(v[7]), chunks=int(v[8]), chunk_rows=int(v[9]), readback_parts=int(v[10]),
                    box_copies=int(v[11]))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().tcw_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


def prepare(strain, fs: float, T_sft: float, f_min: float, n_bins: int, median_bins: int = 101,
            threshold: float = 1.6, fmt: str = "f32", stream=None):
    """tcw_prepare: strain (host numpy float32 or CUDA float32 tensor) -> spectrogram CUDA tensor
    [n_sft][n_bins] float32 (fmt "f32"), uint8 ("u8") or int32 words [n_sft][ceil(n_bins/32)] ("bits")."""
    import torch
    L = load_library()
    if isinstance(strain, np.ndarray):
        x = np.ascontiguousarray(strain, dtype=np.float32)
        ptr, n = x.ctypes.data, x.size
    else:
        x = strain.contiguous()
        if x.dtype != torch.float32:
            raise ValueError("strain must be float32")
        ptr, n = x.data_ptr(), x.numel()
    N = int(round(fs * T_sft))
    n_seg = max(n // max(N, 1), 1)
    dev = torch.device("cuda", torch.cuda.current_device())
    if fmt == "f32":
        out = torch.empty((n_seg, n_bins), dtype=torch.float32, device=dev)
    elif fmt == "u8":
        out = torch.empty((n_seg, n_bins), dtype=torch.uint8, device=dev)
    else:
        out = torch.empty((n_seg, (n_bins + 31) // 32), dtype=torch.int32, device=dev)
    cp = _CPrep(float(fs), float(T_sft), float(f_min), int(n_bins), int(median_bins), float(threshold))
    got = ctypes.c_int(0)
    _check(L.tcw_prepare(ptr, n, ctypes.byref(cp), FORMATS[fmt], out.data_ptr(), out.stride(0) * out.element_size(),
                         ctypes.byref(got), _stream_ptr(stream)))
    return out[: got.value]


SELECT_STATIC_MAX_N = 1 << 28   # TCW_SELECT_STATIC_MAX_N of include/tcw.h


def select_above_static(values, threshold: float, out_idx, out_count, stream=None) -> None:
    """tcw_select_above_static: Handle.select_above for callers that may not allocate on the GPU
    (the job already filled the device with its own arrays, the host program's allocator owns the
    memory, or a cudaMalloc would stall searches running on other streams).  No handle, and nothing
    is allocated here either: the caller passes the outputs, `out_idx` an int64 CUDA tensor whose
    length is the capacity (may be empty) and `out_count` an int64 CUDA tensor with one element.
    The scratch is a fixed array inside libtcw.so, so `values` holds at most SELECT_STATIC_MAX_N
    entries (TcwError beyond that) and calls that overlap on one GPU race; on one stream they are
    safe back to back.  Runs on the current device; make the first call before any stream capture.
    Asynchronous."""
    import torch
    if not values.is_contiguous():
        raise ValueError("values must be contiguous (this call makes no copy)")
    if out_idx.dtype != torch.int64 or out_count.dtype != torch.int64 or out_count.numel() < 1 or not out_idx.is_contiguous():
        raise ValueError("out_idx and out_count must be contiguous int64 CUDA tensors, out_count with one element")
    cap = out_idx.numel()
    _check(load_library().tcw_select_above_static(values.data_ptr(), Handle._sel_dtype(values), values.numel(), float(threshold),
                                                  cap, out_idx.data_ptr() if cap > 0 else None, out_count.data_ptr(),
                                                  _stream_ptr(stream)))


def measure_peaks(stream=None) -> dict:
    """tcw_measure_peaks: measured whole-GPU rates of the limits that bind the kernels (per second)."""
    out = (ctypes.c_double * 12)()
    _check(load_library().tcw_measure_peaks(out, 12, _stream_ptr(stream)))
    keys = ("fp64_dfma_winst_per_s", "fp64_dmul_winst_per_s", "fp64_dadd_winst_per_s", "issue_winst_per_s",
            "lds32_winst_per_s", "chain_lookups_per_s", "n_sm", "sm_clock_max_hz",
            "count_chain_u8_lookups_per_s", "count_chain_bitpacked_lookups_per_s",
            "stage_row_copies_bytes_per_s", "stage_box_copies_bytes_per_s")
    return dict(zip(keys, (float(x) for x in out)))


def split_groups(n_tau: int, n_brk: int, group_begin: int, group_end: int) -> list[tuple[slice, slice, slice]]:
    """tcw_split_groups: the sub-grids (sky, tau, brk index slices) that tile a contiguous range
    of the flattened group index, in ascending order (host-only; what tcw_search_groups runs)."""
    rects = ((ctypes.c_int * 6) * 7)()
    n = ctypes.c_int(0)
    _check(load_library().tcw_split_groups(int(n_tau), int(n_brk), int(group_begin), int(group_end), rects, ctypes.byref(n)))
    return [(slice(r[0], r[1]), slice(r[2], r[3]), slice(r[4], r[5])) for r in list(rects)[: n.value]]


def shard_groups(n_groups: int, rank: int, world_size: int, weights=None) -> tuple[int, int]:
    """Multi-GPU partition: the flattened (sky, tau, n)
    group index 0..n_groups-1 is cut into world_size contiguous ranges and rank r searches
    [begin, end) with Handle.search_groups.  Whole groups per rank, so each per-group argmax stays on
    one rank; the spectrogram is replicated; no collective on the data path.
    weights = None: nearly equal group COUNTS.  weights = [n_groups] non-negative work per group
    (group_work): cut r is placed where the running sum of the weights is nearest r/world_size of the
    total, so ranks get nearly equal WORK (groups with small tau or small n leave the band early and
    cost less).  Every rank computes the same cuts from the same weights; no communication.
    A rank may get an empty range (begin == end) when world_size > n_groups."""
    if not (0 <= rank < world_size):
        raise ValueError("rank out of range")
    n_groups = int(n_groups)
    if weights is None:
        base, rem = divmod(n_groups, world_size)
        lo = rank * base + min(rank, rem)
        return lo, lo + base + (1 if rank < rem else 0)
    wt = np.asarray(weights, dtype=np.float64).reshape(-1)
    if wt.size != n_groups or not np.all(np.isfinite(wt)) or np.any(wt < 0):
        raise ValueError("weights must be n_groups finite non-negative numbers")
    cum = np.concatenate(([0.0], np.cumsum(wt)))           # cum[i] = work of groups 0..i-1
    if not cum[-1] > 0:
        return shard_groups(n_groups, rank, world_size)
    cuts = [0]
    for r in range(1, world_size):
        target = cum[-1] * r / world_size
        i = int(np.searchsorted(cum, target))               # first i with cum[i] >= target
        if i > 0 and target - cum[i - 1] <= cum[min(i, n_groups)] - target:
            i -= 1                                          # the cut below is at least as near
        cuts.append(min(max(i, cuts[-1]), n_groups))
    cuts.append(n_groups)
    return cuts[rank], cuts[rank + 1]


def group_work(grid: Grid, timestamps, T_sft: float, f_min: float, n_bins: int) -> np.ndarray:
    """Scheduling estimate for shard_groups(weights=): per group of the flattened (sky, tau, n) index,
    how many (f0, SFT) lookups fall inside the band.  From eq. (1) alone -- the
    track f0 (1 + t/tau)^(-1/(n-1)) crosses a band edge f_e at t = tau ((f0/f_e)^(n-1) - 1) -- with the
    1e-4 Doppler factor left out, so it is the same for every sky point.  It only decides where the
    group axis is cut between GPUs; no search result depends on it."""
    ts = np.sort(_f64(timestamps)) - float(grid.T0)
    k_min = float(np.rint(f_min * T_sft))
    f_lo, f_hi = (k_min - 0.5) / T_sft, (k_min + n_bins - 0.5) / T_sft
    per = np.zeros((len(grid.tau), len(grid.brk)))
    for a, tau in enumerate(grid.tau):
        for b, n in enumerate(grid.brk):
            t_exit = tau * (np.maximum(grid.f0 / f_lo, 0.0) ** (n - 1.0) - 1.0)     # below f_lo from here on
            t_enter = tau * (np.maximum(grid.f0 / f_hi, 0.0) ** (n - 1.0) - 1.0)    # above f_hi before
            hi = np.searchsorted(ts, t_exit, side="left")
            lo = np.searchsorted(ts, np.maximum(t_enter, 0.0), side="left")
            per[a, b] = float(np.maximum(hi - lo, 0).sum())
    return np.tile(per.reshape(-1), len(grid.sky))
