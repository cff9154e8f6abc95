"""CPU-side checks of the boundary: libtcw.so builds, loads without a GPU, exports every symbol
include/tcw.h declares, and rejects bad arguments before touching CUDA.  No compute call is made."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2507_07816_b200 as tcw

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "tcw.h")


@pytest.fixture(scope="module")
def lib():
    return tcw.load_library()


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tcw_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_functions()
    assert set(names) == set(tcw.EXPORTS)
    for n in names:
        assert getattr(lib, n) is not None


def test_header_constants_match_binding():
    text = open(HEADER).read()
    for name in ("TCW_OK", "TCW_EINVAL", "TCW_ENOMEM", "TCW_ECUDA", "TCW_EUNSUPPORTED",
                 "TCW_F32_POWER", "TCW_U8_COUNT", "TCW_BIT_COUNT",
                 "TCW_OPT_KERNEL", "TCW_OPT_TIMING", "TCW_OPT_F0_PER_LANE"):
        m = re.search(rf"\b{name}\s*=\s*(-?\d+)", text)
        assert m, name
        assert int(m.group(1)) == getattr(tcw, name), name


def _sass_of(function: str) -> str:
    """SASS of one kernel of the built library (cuobjdump prints every function; split by name)."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump) and not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not available")
    if not hasattr(_sass_of, "text"):
        _sass_of.text = subprocess.run([cuobjdump, "-sass", tcw.library_path()], capture_output=True, text=True).stdout
    parts = re.split(r"\n\s*Function : ", _sass_of.text)
    for part in parts[1:]:
        if part.split("\n", 1)[0].strip() == function:
            return part
    raise AssertionError(f"{function} not found in {tcw.library_path()}")


def test_library_is_sm100a_and_has_tma_bulk_copies():
    """The .so carries sm_100a SASS and the staged kernel's TMA bulk copies (UBLKCP)."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump) and not shutil.which("cuobjdump"):
        pytest.skip("cuobjdump not available")
    elf = subprocess.run([cuobjdump, "-lelf", tcw.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in elf
    for wgt in ("0", "1"):               # plain and weighted instantiations
        sass = _sass_of(f"_ZN3tcw17sum_staged_kernelILi0ELi8ELb1ELb{wgt}ELb0EEEvNS_9SumParamsE")
        assert "UBLKCP" in sass and "SYNCS" in sass
        # the fast index is ONE fused multiply-add per lookup (8 templates per lane x 4 rows per ring slot)
        # and the defining chain (DMUL, DMUL, DADD) stays in the kernel as the guard band's fallback
        assert sass.count("DFMA") >= 32
        assert "DMUL" in sass and "DADD" in sass
        # ring slots of four SFT rows travel by one tensor-map TMA copy (cp.async.bulk.tensor.3d)
        assert "UTMALDG.3D" in sass
        assert ("FFMA" in sass) == (wgt == "1")   # only the weighted sum fuses weight * element + acc
    # the headline instantiation (float32, 16 templates per lane, equally spaced f0) adds row pairs with packed
    # float32 adds
    head = _sass_of("_ZN3tcw17sum_staged_kernelILi0ELi16ELb1ELb0ELb1EEEvNS_9SumParamsE")
    assert "UTMALDG.3D" in head and "UBLKCP" in head and head.count("FADD2") >= 32


def test_defining_chain_is_never_contracted():
    """The kernels that DEFINE the bins for the rest of the library -- the gather kernel and the
    index export, both straight bin_lo chains -- contain no fused multiply-add: every step of
    ((f0*g)*D)*T is one IEEE operation (build flag -fmad=false plus __dmul_rn / __dadd_rn)."""
    for fn in ("_ZN3tcw17sum_gather_kernelILi0ELb1ELb0EEEvNS_9SumParamsE",
               "_ZN3tcw17sum_gather_kernelILi1ELb0ELb0EEEvNS_9SumParamsE",
               "_ZN3tcw18track_index_kernelILb1EEEvNS_9SumParamsEPKlliPi",
               "_ZN3tcw18track_index_kernelILb0EEEvNS_9SumParamsEPKlliPi"):
        sass = _sass_of(fn)
        assert "DFMA" not in sass and "FFMA" not in sass, fn
        assert "DMUL" in sass and "DADD" in sass, fn


def _create_args(n_sft=4, n_bins=8):
    spec = np.zeros((n_sft, n_bins), dtype=np.float32)
    ts = 8.0 * np.arange(n_sft) + 4.0
    vel = np.zeros((n_sft, 3))
    return spec, ts, vel


def _create(lib, spec, fmt, pitch, n_sft, n_bins, f_min, T, ts, vel):
    h = ctypes.c_void_p()
    dp = ctypes.POINTER(ctypes.c_double)
    rc = lib.tcw_create(ctypes.byref(h), spec.ctypes.data if spec is not None else None, fmt, pitch, n_sft, n_bins,
                        f_min, T, ts.ctypes.data_as(dp) if ts is not None else None,
                        vel.ctypes.data_as(dp) if vel is not None else None, None)
    return rc, h


def test_create_rejects_bad_arguments_without_cuda(lib):
    spec, ts, vel = _create_args()
    bad = [
        dict(spec=None),
        dict(ts=None),
        dict(vel=None),
        dict(fmt=7),
        dict(n_sft=0),
        dict(n_bins=-1),
        dict(pitch=16),                                   # smaller than a row of 8 floats
        dict(T=0.0),
        dict(f_min=500.03),                               # f_min*T_sft not an integer
        dict(ts=np.array([4.0, 12.0, 12.0, 28.0])),       # not strictly increasing
        dict(ts=np.array([4.0, np.nan, 20.0, 28.0])),
        dict(vel=np.full((4, 3), 3e8)),                   # not a physical detector velocity
    ]
    for kw in bad:
        a = dict(spec=spec, fmt=0, pitch=32, n_sft=4, n_bins=8, f_min=500.0, T=8.0, ts=ts, vel=vel)
        a.update(kw)
        rc, h = _create(lib, a["spec"], a["fmt"], a["pitch"], a["n_sft"], a["n_bins"], a["f_min"], a["T"],
                        a["ts"], a["vel"])
        assert rc == tcw.TCW_EINVAL, kw
        assert not h.value
        assert len(lib.tcw_last_error()) > 0
    assert lib.tcw_create(None, None, 0, 0, 0, 0, 0.0, 0.0, None, None, None) == tcw.TCW_EINVAL


def test_null_handle_calls(lib):
    assert lib.tcw_destroy(None) == tcw.TCW_OK
    assert lib.tcw_search(None, None, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_search_host(None, None, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_set_option(None, 0, 0) == tcw.TCW_EINVAL
    assert lib.tcw_get_timing(None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_get_info(None, None) == tcw.TCW_EINVAL
    assert lib.tcw_tables(None, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_track_indices(None, None, 0, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_search_weighted(None, None, None, None, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_search_bank(None, None, None, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_topk(None, None, 0, 1, 1, None, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_select_above(None, None, 0, 1, 0.0, 0, None, None, None) == tcw.TCW_EINVAL
    assert lib.tcw_get_counter(None, 0, None) == tcw.TCW_EINVAL
    assert lib.tcw_upload_wait(None) == tcw.TCW_EINVAL
    assert isinstance(lib.tcw_last_error(), bytes)


def test_prepare_rejects_bad_arguments_without_cuda(lib):
    """tcw_prepare validates sizes before the first CUDA call (no handle is involved)."""
    from paper_2507_07816_b200 import _CPrep
    x = np.zeros(4096, dtype=np.float32)
    n = ctypes.c_int(0)
    good = dict(fs=64.0, T_sft=8.0, f_min=8.0, n_bins=64, median_bins=9, threshold=1.6)
    def call(**kw):
        a = dict(good); a.update(kw)
        cp = _CPrep(a["fs"], a["T_sft"], a["f_min"], a["n_bins"], a["median_bins"], a["threshold"])
        return lib.tcw_prepare(x.ctypes.data, x.size, ctypes.byref(cp), 0, 1, 4 * a["n_bins"], ctypes.byref(n), None)
    for kw in (dict(fs=0.0), dict(fs=63.9), dict(n_bins=0), dict(median_bins=4), dict(f_min=0.05),
               dict(f_min=31.0, n_bins=40), dict(f_min=0.0)):
        assert call(**kw) == tcw.TCW_EINVAL, kw
    assert lib.tcw_prepare(None, 0, None, 0, None, 0, None, None) == tcw.TCW_EINVAL


def test_create_async_rejects_bad_arguments_without_cuda(lib):
    spec, ts, vel = _create_args()
    h = ctypes.c_void_p()
    dp = ctypes.POINTER(ctypes.c_double)
    rc = lib.tcw_create_async(ctypes.byref(h), spec.ctypes.data, 7, 32, 4, 8, 500.0, 8.0, ts.ctypes.data_as(dp),
                              vel.ctypes.data_as(dp), None)
    assert rc == tcw.TCW_EINVAL and not h.value


def test_no_cuda_device_fails_loudly(lib):
    """On a box without a GPU a valid tcw_create must fail with TCW_ECUDA, never fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    spec, ts, vel = _create_args()
    rc, h = _create(lib, spec, 0, 32, 4, 8, 500.0, 8.0, ts, vel)
    assert rc == tcw.TCW_ECUDA and not h.value
    with pytest.raises((tcw.TcwError, RuntimeError, AssertionError)):
        tcw.Handle(spec, "f32", 8, 500.0, 8.0, ts, vel)


def test_grid_marshalling_and_sharding():
    g = tcw.Grid([500.0, 500.125], [3500.0], [3, 5, 7], [[1, 0, 0], [0, 1, 0]], T0=12.0)
    c = g._c()
    assert (c.n_f0, c.n_tau, c.n_brk, c.n_sky, c.T0) == (2, 1, 3, 2, 12.0)
    assert c.brk[2] == 7.0 and c.sky[4] == 1.0
    assert g.n_groups == 6 and g.n_templates == 12
    for n_groups, world in [(160, 8), (7, 3), (2, 4), (98304, 5), (576, 7)]:
        parts = [tcw.shard_groups(n_groups, r, world) for r in range(world)]
        assert parts[0][0] == 0 and parts[-1][1] == n_groups
        assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
        sizes = [hi - lo for lo, hi in parts]
        assert max(sizes) - min(sizes) <= 1


def test_split_groups_tiles_every_range_in_order():
    """tcw_split_groups (host-only): any contiguous range of the flattened (sky, tau, n) index is
    tiled, in ascending order and without overlap, by at most seven sub-grids whose own order is a
    contiguous run of the flattened index."""
    rng = np.random.default_rng(5)
    for n_sky, n_tau, n_brk in [(1, 32, 5), (1, 64, 9), (5, 4, 3), (3, 1, 7), (4, 6, 1), (256, 16, 5)]:
        n_groups = n_sky * n_tau * n_brk
        flat = np.arange(n_groups).reshape(n_sky, n_tau, n_brk)
        ranges = [(0, n_groups), (0, 1), (n_groups - 1, n_groups), (3, 3)]
        ranges += [tuple(sorted(rng.integers(0, n_groups + 1, size=2))) for _ in range(60)]
        for g0, g1 in ranges:
            rects = tcw.split_groups(n_tau, n_brk, int(g0), int(g1))
            assert len(rects) <= 7
            got = [flat[s, a, b].reshape(-1) for s, a, b in rects]
            got = np.concatenate(got) if got else np.empty(0, dtype=int)
            assert np.array_equal(got, np.arange(g0, g1)), (n_sky, n_tau, n_brk, g0, g1)
