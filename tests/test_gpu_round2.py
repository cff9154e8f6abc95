"""Round-2 GPU parity: the one-FMA fast index against the defining chain and the oracle, wide
bands, the device status word as an error, group ranges (multi-GPU unit), the overlapped host
read-back, and cfg2 / cfg3 at BASELINE.json's full sizes in the bench's launch configuration."""
import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload, detector_velocity, sky_vector

from test_gpu_parity import TOL, assert_best_parity, assert_stat_parity, tcw  # noqa: F401
from test_gpu_full_size import _device_group_parity

pytestmark = pytest.mark.gpu


def _search_with(tcw, w, options, host=False):
    import torch
    with tcw.Handle.from_workload(w, host=host) as h:
        for k, v in options.items():
            h.set_option(k, v)
        stat, best = h.search(tcw.Grid.of(w))
        torch.cuda.synchronize()
        info = h.info()
        return stat.cpu().numpy(), best.cpu().numpy(), info


def _random_workload(rng, fmt, n_sft, n_bins, n_f0, df_bins, T=8.0, f_min=500.0, n_sky=1, uniform=True):
    ts = T * np.arange(n_sft) + T / 2
    keep = rng.random(n_sft) > 0.1
    keep[0] = True
    ts = ts[keep]
    rho = rng.standard_exponential((len(ts), n_bins), dtype=np.float32)
    spec = rho if fmt == "f32" else (rho > 1.6).astype(np.uint8)
    f0 = f_min + (df_bins / T) * np.arange(n_f0) + rng.uniform(0, 20.0)
    if not uniform:
        f0 = np.sort(f0 + rng.uniform(-0.3, 0.3, n_f0) * df_bins / T)
    sky = tcw_inputs.fibonacci_cap(n_sky, 1.0, 0.3, 10.0) if n_sky > 1 else sky_vector(1.0, 0.3)[None]
    return Workload("rnd", fmt, spec, len(ts), n_bins, f_min, T, ts, detector_velocity(ts), float(ts[0]) - 3.0,
                    f0, np.array([3500.0, 9000.0, 30000.0]), np.array([3.0, 4.5, 7.0]), sky)


@pytest.mark.parametrize("fmt", ["f32", "u8"])
def test_fast_index_is_bit_identical_to_the_defining_chain(tcw, fmt):
    """The staged kernel's one-FMA index with its guard band selects the bins of
    the defining chain: whole searches agree bit for bit between the default build path, the path with
    TCW_OPT_EXACT_INDEX (every bin by bin_lo) and the general-f0 instantiation, and all agree with the
    oracle -- on cfg1 and on random shapes (holes, T0 inside the data, SFT lengths 8 and 10 s, f0
    spacings of half, one and two bins, uniform and jittered f0 axes)."""
    rng = np.random.default_rng(20250707)
    cases = [tcw_inputs.make_workload("cfg1") if fmt == "f32" else tcw_inputs.make_workload("cfg1").with_format("u8")]
    for trial in range(10):
        cases.append(_random_workload(rng, fmt, int(rng.integers(70, 400)), int(rng.integers(600, 5000)),
                                      int(rng.integers(40, 1500)), float(rng.choice([0.5, 1.0, 2.0])),
                                      T=float(rng.choice([8.0, 10.0])), uniform=bool(trial % 2)))
    for w in cases:
        ref = oracle.evaluate(w)
        # the two instantiations (equally spaced f0 / general f0) add a row pair in different orders, so their
        # float32 sums may differ in the last bits; inside one instantiation the fast index and the defining
        # chain must give identical bits, and counts are identical everywhere
        for inst in ({}, {tcw.TCW_OPT_GENERAL_F0: 1}):
            base, bbest, info = _search_with(tcw, w, {tcw.TCW_OPT_KERNEL: 2, **inst})
            assert info["kernel"] == "staged"
            assert_stat_parity(w, base.reshape(-1), ref.stat)
            got, gbest, _ = _search_with(tcw, w, {tcw.TCW_OPT_KERNEL: 2, tcw.TCW_OPT_EXACT_INDEX: 1, **inst})
            assert np.array_equal(got.view(np.int32), base.view(np.int32)), inst
            assert np.array_equal(gbest, bbest), inst
            for r in (8, 4):
                got, _, _ = _search_with(tcw, w, {tcw.TCW_OPT_KERNEL: 2, tcw.TCW_OPT_F0_PER_LANE: r, **inst})
                ex, _, _ = _search_with(tcw, w, {tcw.TCW_OPT_KERNEL: 2, tcw.TCW_OPT_F0_PER_LANE: r,
                                                 tcw.TCW_OPT_EXACT_INDEX: 1, **inst})
                assert np.array_equal(got.view(np.int32), ex.view(np.int32)), (inst, r)
                assert_stat_parity(w, got.reshape(-1), ref.stat)
                if fmt == "u8":
                    assert np.array_equal(got, base), (inst, r)


def test_fast_index_exact_ties_and_near_ties(tcw):
    """Tracks constructed to sit exactly on half-integers (zero velocity, t_j = T0 so g = 1, f0*T =
    k + 1/2) and one ulp either side of them: the guard band must hand these lookups to the defining
    chain, which rounds half to even like the oracle."""
    n_sft, n_bins, T = 96, 2048, 8.0
    ts = T * np.arange(n_sft) + 4.0
    rng = np.random.default_rng(3)
    spec = rng.integers(0, 200, size=(n_sft, n_bins)).astype(np.uint8)
    k = 4000 + np.arange(10, 1500, 3)
    f0 = (k + 0.5) / T
    f0 = np.unique(np.concatenate([f0, np.nextafter(f0, 0), np.nextafter(f0, 1e9), (k + 1.0) / T]))
    w = Workload("ties", "u8", spec, n_sft, n_bins, 500.0, T, ts, np.zeros((n_sft, 3)), 4.0,
                 f0, np.array([3500.0, 1e9]), np.array([3.0, 5.0]), sky_vector(0.3, -0.2)[None])
    got, _, info = _search_with(tcw, w, {tcw.TCW_OPT_KERNEL: 2})
    assert info["kernel"] == "staged"
    ref = oracle.evaluate(w)
    assert ref.n_ambig.sum() > 0          # the oracle flags the exact ties ...
    clean = ref.n_ambig == 0
    assert np.array_equal(got.reshape(-1)[clean].astype(np.int64), ref.stat[clean])
    # ... and, rounding half to even in the same precision, the GPU agrees on them as well
    assert np.array_equal(got.reshape(-1).astype(np.int64), ref.stat)


def test_wide_float32_band_above_131072_bins(tcw):
    """A float32 band of 150 000 bins (window starts beyond 512 KiB of a row once overflowed
    a 16-bit metadata field).  Templates near the top of the band, staged kernel, against the oracle."""
    n_sft, n_bins, T = 48, 150000, 8.0
    ts = T * np.arange(n_sft) + 4.0
    rng = np.random.default_rng(9)
    rho = rng.standard_exponential((n_sft, n_bins), dtype=np.float32)
    f0 = 100.0 + 0.125 * (n_bins - 2600 + np.arange(2500))
    w = Workload("wide", "f32", rho, n_sft, n_bins, 100.0, T, ts, detector_velocity(ts), 0.0,
                 f0, np.array([3500.0, 35000.0]), np.array([3.0, 7.0]), sky_vector(1.0, 0.3)[None])
    got, best, info = _search_with(tcw, w, {})
    assert info["kernel"] == "staged"
    ref = oracle.evaluate(w)
    assert ref.n_inband.min() > 0
    assert_stat_parity(w, got.reshape(-1), ref.stat)


@pytest.mark.parametrize("fmt,kernel", [("f32", "staged"), ("u8", "skyblock")])
def test_violated_window_bound_is_reported_not_silent(tcw, fmt, kernel):
    """a violated window bound used to give silently wrong sums.  The test hook lowers the
    kernels' own bound so that every staged row trips it; tcw_search_host, tcw_check, tcw_get_timing and
    tcw_get_info must then fail with TCW_EINTERNAL, and a following good search must clear the state."""
    import torch
    w = tcw_inputs.make_workload("cfg1")
    if fmt == "u8":
        w = w.with_format("u8")
        w.sky = tcw_inputs.fibonacci_cap(64, 1.0, 0.3, 10.0)
    grid = tcw.Grid.of(w)
    with tcw.Handle.from_workload(w) as h:
        h.set_option(tcw.TCW_OPT_DEBUG_SHRINK_SLOT, 1 << 19)
        with pytest.raises(tcw.TcwError) as e:
            h.search_host(grid)
        assert e.value.code == tcw.TCW_EINTERNAL
        h.search(grid)
        with pytest.raises(tcw.TcwError) as e:
            h.check()
        assert e.value.code == tcw.TCW_EINTERNAL
        with pytest.raises(tcw.TcwError):
            h.info()
        info = h.info(check=False)
        assert info["status"] != 0 and info["kernel"] == kernel
        h.set_option(tcw.TCW_OPT_TIMING, 1)
        h.search(grid)
        with pytest.raises(tcw.TcwError):
            h.timing()
        h.set_option(tcw.TCW_OPT_TIMING, 0)
        h.set_option(tcw.TCW_OPT_DEBUG_SHRINK_SLOT, 0)
        stat, _ = h.search(grid)
        h.check()
        torch.cuda.synchronize()
        ref = oracle.evaluate(w)
        assert_stat_parity(w, stat.cpu().numpy().reshape(-1), ref.stat)


def test_search_groups_equals_slices_of_the_whole_search(tcw):
    """tcw_search_groups over any contiguous range of the flattened (sky, tau, n) index reproduces the
    slice of tcw_search bit for bit (the multi-GPU unit); n_sky = 1 and n_sky = 3."""
    import torch
    rng = np.random.default_rng(11)
    base = tcw_inputs.make_workload("cfg1")
    for n_sky in (1, 3):
        w = base.subgrid()
        if n_sky > 1:
            w.sky = tcw_inputs.fibonacci_cap(n_sky, 1.0, 0.3, 10.0)
        grid = tcw.Grid.of(w)
        n_f0 = len(w.f0)
        with tcw.Handle.from_workload(w) as h:
            stat, best = h.search(grid)
            torch.cuda.synchronize()
            stat = stat.reshape(-1, n_f0).cpu().numpy()
            best = best.cpu().numpy()
            ranges = [(0, grid.n_groups), (0, 1), (grid.n_groups - 1, grid.n_groups)]
            ranges += [tuple(sorted(rng.choice(grid.n_groups + 1, size=2, replace=False))) for _ in range(12)]
            for g0, g1 in ranges:
                s, b = h.search_groups(grid, int(g0), int(g1))
                h.check()
                assert np.array_equal(s.cpu().numpy().view(np.int32), stat[g0:g1].view(np.int32)), (n_sky, g0, g1)
                assert np.array_equal(b.cpu().numpy(), best[g0:g1]), (n_sky, g0, g1)
            # an empty in-range interval is a rank with nothing to do (no-op); the C call itself still
            # refuses it, as tcw.h says, and anything outside 0..n_groups is an error either way
            assert h.search_groups(grid, 3, 3)[0].shape[0] == 0
            cg = grid._c()
            import ctypes
            assert tcw.load_library().tcw_search_groups(h._h, ctypes.byref(cg), 3, 3, s.data_ptr(), b.data_ptr(), None) == tcw.TCW_EINVAL
            with pytest.raises(tcw.TcwError):
                h.search_groups(grid, 0, grid.n_groups + 1)
    ref = oracle.evaluate(w)
    assert_stat_parity(w, stat.reshape(-1), ref.stat)


def test_search_groups_count_formats_across_sky_blocks(tcw):
    """Group ranges of a 40-sky-point uint8 grid: the whole search runs on the sky-block kernel, a range is
    served by whole-sky sub-grids (sky-block kernel) plus partial sky points (staged kernel); counts are exact
    integers, so every slice must be identical whichever kernels produced it."""
    import torch
    rng = np.random.default_rng(17)
    w = tcw_inputs.make_workload("cfg1").with_format("u8")
    w.sky = tcw_inputs.fibonacci_cap(40, 1.0, 0.3, 10.0)
    grid = tcw.Grid.of(w)
    with tcw.Handle.from_workload(w) as h:
        stat, best = h.search(grid)
        torch.cuda.synchronize()
        assert h.info()["kernel"] == "skyblock"
        stat = stat.reshape(-1, len(w.f0)).cpu().numpy()
        best = best.cpu().numpy()
        for g0, g1 in [(0, grid.n_groups), (5, 12 * 30 + 7), (12 * 3, 12 * 29)] + \
                [tuple(sorted(rng.choice(grid.n_groups + 1, size=2, replace=False))) for _ in range(6)]:
            s, b = h.search_groups(grid, int(g0), int(g1))
            h.check()
            assert np.array_equal(s.cpu().numpy(), stat[g0:g1]) and np.array_equal(b.cpu().numpy(), best[g0:g1]), (g0, g1)
    ref = oracle.evaluate(w, sel=oracle.group_templates(w, np.array([0, 77, grid.n_groups - 1])))
    assert np.array_equal(stat[[0, 77, grid.n_groups - 1]].reshape(-1).astype(np.int64), ref.stat)


def test_search_host_overlapped_read_back_is_bit_identical(tcw):
    """An out_stat of more than 64 MiB goes to the host tau range by tau range while the later ranges are
    still being searched (tcw_search_host: per-range progress counters + cuStreamWaitValue32); the host
    arrays must equal the plain device search exactly, also when the call is repeated on the handle.
    cfg3 data, 4000 f0 x 16 tau x 5 n x 56 sky points = 17.9 M templates (72 MB), pinned host buffers."""
    import torch
    w = tcw_inputs.make_workload("cfg3", fmt="u8").subgrid(sky=np.arange(0, 256, 256 // 56)[:56])
    grid = tcw.Grid.of(w)
    assert grid.n_templates * 4 > (64 << 20)
    with tcw.Handle.from_workload(w) as h:
        stat, best = h.search(grid)
        torch.cuda.synchronize()
        out = torch.empty(stat.shape, dtype=torch.int32).pin_memory()
        bout = torch.empty((grid.n_groups, 2), dtype=torch.int32).pin_memory()
        h.search_host(grid, out.numpy(), bout.numpy())
        info = h.info()
        assert info["readback_parts"] > 1     # the progressive read-back was taken
        assert torch.equal(out, stat.cpu()) and torch.equal(bout, best.cpu())
        # pageable host arrays take the same path; so does a repeated call (the counters are cleared per search)
        for _ in range(2):
            o2, b2 = h.search_host(grid)
            assert np.array_equal(o2, out.numpy()) and np.array_equal(b2, bout.numpy())
    groups = np.array([0, 17, grid.n_groups - 1])
    ref = oracle.evaluate(w, sel=oracle.group_templates(w, groups))
    assert np.array_equal(out.numpy().reshape(-1, len(w.f0))[groups].reshape(-1).astype(np.int64), ref.stat)


def test_async_uint8_handle_takes_the_two_level_kernel(tcw):
    """a uint8 handle made by tcw_create_async assumed counts up to 255 and never took the
    256-point sky-block kernel.  The first search now scans the uploaded rows."""
    import torch
    w = tcw_inputs.make_workload("cfg3", fmt="u8").subgrid(tau=[0, 9], brk=[1])
    grid = tcw.Grid.of(w)
    spec = torch.from_numpy(np.ascontiguousarray(w.spectrogram)).pin_memory()
    with tcw.Handle(spec, "u8", w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities, async_upload=True) as h:
        stat, best = h.search(grid)
        torch.cuda.synchronize()
        info = h.info()
        assert info["kernel"] == "skyblock" and info["sky_block"] == 256
    with tcw.Handle.from_workload(w) as h2:
        s2, b2 = h2.search(grid)
        torch.cuda.synchronize()
    assert torch.equal(stat, s2) and torch.equal(best, b2)


def test_cfg2_full_grid_every_group(tcw):
    """'cfg1 and cfg2 are checked in full'.  All 640 000 templates x 10 800 SFTs
    of cfg2 against the oracle (6.9e9 lookups: a few seconds on the box's cores), every statistic and
    every per-group best; bin indices of 3000 sampled templates identical wherever the oracle does
    not flag a tie."""
    import torch
    w = tcw_inputs.make_workload("cfg2")
    grid = tcw.Grid.of(w)
    with tcw.Handle.from_workload(w) as h:
        stat, best = h.search(grid)
        torch.cuda.synchronize()
        info = h.info()
        assert info["kernel"] == "staged" and info["chunks"] > 1
        bs, bi = h.best_fields(best)
        rng = np.random.default_rng(2)
        sel = np.sort(rng.choice(w.n_templates, size=3000, replace=False))
        k = h.track_indices(grid, sel).cpu().numpy()
    ref = oracle.evaluate(w)
    assert_stat_parity(w, stat.cpu().numpy().reshape(-1), ref.stat)
    assert_best_parity(w, len(w.f0), bs, bi, ref.stat)
    rk = oracle.evaluate(w, sel=sel, want_k=True)
    clean = rk.n_ambig == 0
    assert clean.sum() >= 2990 and np.array_equal(k[clean], rk.k[clean])


@pytest.mark.parametrize("fmt", ["u8", "bits"])
def test_cfg3_full_size_sampled_groups(tcw, fmt):
    """cfg3 exactly as bench.py times it: 81.92 M templates (4000 f0 x 16 tau x 5 n x 256 sky points),
    number counts as uint8 and bit-packed, automatic kernel choice = the two-level 256-point sky-block
    kernel; counts of sampled whole groups bit-exact against the oracle, per-group best exact, and
    size-independent properties on the whole output."""
    import torch
    w = tcw_inputs.make_workload("cfg3", fmt=fmt)
    with tcw.Handle.from_workload(w) as h:
        stat, best = h.search(tcw.Grid.of(w))
        torch.cuda.synchronize()
        info = h.info()
        assert info["kernel"] == "skyblock" and info["sky_block"] == 256 and info["status"] == 0
        n_ab = len(w.tau) * len(w.brk)
        # first and last group plus 32 seeded-random ones (no hand-picked lists)
        groups = np.unique(np.concatenate(([0, 256 * n_ab - 1], np.random.default_rng(303).integers(0, 256 * n_ab, size=32))))
        _device_group_parity(tcw, w, groups, stat, best, h)
        st = stat.reshape(-1, len(w.f0))
        bmax = st.max(dim=1)
        b = best.cpu().numpy()
        assert np.array_equal(b[:, 0], bmax.values.cpu().numpy())
        idx = torch.as_tensor(b[:, 1], device=st.device).long()
        first = (st == bmax.values[:, None]).int().argmax(dim=1)
        assert torch.equal(first, idx)
        assert (stat >= 0).all().item() and (stat <= w.n_sft).all().item()


@pytest.mark.parametrize("fmt", ["f32", "u8"])
def test_box_copies_are_bit_identical_to_row_copies(tcw, fmt):
    """The staged kernel fetches a ring slot (four consecutive SFT rows) with ONE tensor-map copy where the rows'
    windows fit one box, and with one 1-D bulk copy per row otherwise (band edges, gaps in the data, the steep
    start of a fast spin-down).  Both stagings feed the same arithmetic in the same order, so whole searches must
    agree bit for bit with TCW_OPT_ROW_COPIES, and with the oracle: on cfg1, on random shapes with holes (rows of
    one slot far apart in time), on a steep track (3000 Hz, tau = 3500 s, n = 3: 27 bins per SFT at the start) and
    on an SFT-chunked search."""
    rng = np.random.default_rng(20251105)
    base = tcw_inputs.make_workload("cfg1")
    cases = [(base if fmt == "f32" else base.with_format("u8"), {})]
    for trial in range(6):
        w = _random_workload(rng, fmt, int(rng.integers(70, 400)), int(rng.integers(600, 5000)),
                             int(rng.integers(40, 1500)), float(rng.choice([0.5, 1.0, 2.0])),
                             T=float(rng.choice([8.0, 10.0])), uniform=bool(trial % 2))
        cases.append((w, {tcw.TCW_OPT_CHUNK_ROWS: 64} if trial % 3 == 0 else {}))
    # steep: a band of 2600 bins below 3000 Hz, 600 templates, short tau, low braking index, and a gap of two hours
    T, n_bins, f_min = 8.0, 2600, 2700.0
    ts = np.concatenate([T * np.arange(300) + T / 2, 7200.0 + T * np.arange(300, 520) + T / 2])
    rho = rng.standard_exponential((len(ts), n_bins), dtype=np.float32)
    spec = rho if fmt == "f32" else (rho > 1.6).astype(np.uint8)
    steep = Workload("steep", fmt, spec, len(ts), n_bins, f_min, T, ts, detector_velocity(ts), 0.0,
                     f_min + 150.0 + 0.125 * np.arange(600), np.array([3500.0, 5000.0]), np.array([3.0, 5.0]),
                     sky_vector(1.0, 0.3)[None])
    cases.append((steep, {}))
    n_box = 0
    for w, opts in cases:
        ref = oracle.evaluate(w)
        s_box, b_box, i_box = _search_with(tcw, w, {tcw.TCW_OPT_KERNEL: 2, **opts})
        s_row, b_row, i_row = _search_with(tcw, w, {tcw.TCW_OPT_KERNEL: 2, tcw.TCW_OPT_ROW_COPIES: 1, **opts})
        assert i_row["box_copies"] == 0 and i_box["status"] == 0 and i_row["status"] == 0
        n_box += i_box["box_copies"]
        assert np.array_equal(s_box.view(np.uint32), s_row.view(np.uint32)), w.name
        assert np.array_equal(b_box.view(np.uint8), b_row.view(np.uint8)), w.name
        assert_stat_parity(w, s_box.reshape(-1), ref.stat)
    assert n_box > 0, "no case exercised the tensor-map copies"


def test_measured_peaks_are_sane(tcw):
    """tcw_measure_peaks: every rate is positive and in the order the hardware imposes -- FP64 at about half the
    issue rate, the shipped lookup chain below 32 lookups per issued instruction, a tensor-map copy per slot staging
    at least as fast as four bulk copies per slot (within noise), bit-packed gathers slower than byte gathers."""
    import torch
    torch.cuda.set_device(0)
    p = tcw.measure_peaks()
    assert all(v > 0 for v in p.values()), p
    assert 0.35 < p["fp64_dfma_winst_per_s"] / p["issue_winst_per_s"] < 0.6
    assert p["chain_lookups_per_s"] < 32 * p["issue_winst_per_s"] / 3.5
    assert p["stage_box_copies_bytes_per_s"] > 0.9 * p["stage_row_copies_bytes_per_s"] > 5e12
    assert p["count_chain_bitpacked_lookups_per_s"] < p["count_chain_u8_lookups_per_s"]


def test_bank_search_clears_the_status_word(tcw, cfg1):
    """tcw.h says every search starts with a clear status word and lists tcw_search_bank among the
    calls tcw_check reports on; a bank search after an invalid grid search must therefore check clean."""
    import torch
    w = cfg1
    f0, tau, brk, sky = tcw_inputs.random_bank(200, 480.0, 640.0, 5, sky=w.sky[0])
    with tcw.Handle.from_workload(w) as h:
        h.set_option(tcw.TCW_OPT_DEBUG_SHRINK_SLOT, 1 << 19)
        h.search(tcw.Grid.of(w))
        with pytest.raises(tcw.TcwError):
            h.check()
        h.set_option(tcw.TCW_OPT_DEBUG_SHRINK_SLOT, 0)
        stat, inband, _ = h.search_bank(f0, tau, brk, sky, T0=w.T0)
        h.check()
        assert h.info()["status"] == 0
        torch.cuda.synchronize()
    ref = oracle.evaluate_bank(w, f0, tau, brk, sky)
    clean = ref.n_ambig == 0
    assert np.array_equal(inband.cpu().numpy()[clean], ref.n_inband[clean])


def test_search_groups_of_an_empty_range_is_a_no_op(tcw, cfg1):
    """shard_groups hands a rank an empty range when world_size > n_groups; that rank must get
    empty outputs, not an error."""
    grid = tcw.Grid.of(cfg1)
    with tcw.Handle.from_workload(cfg1) as h:
        for r in range(16):
            lo, hi = tcw.shard_groups(grid.n_groups, r, 16)          # 12 groups over 16 ranks
            stat, best = h.search_groups(grid, lo, hi)
            assert stat.shape == (hi - lo, len(grid.f0)) and best.shape == (hi - lo, 2)
        with pytest.raises(tcw.TcwError):
            h.search_groups(grid, grid.n_groups + 1, grid.n_groups + 1)


@pytest.mark.parametrize("fail_part", [1, 2, 3])
def test_read_back_survives_a_refused_stream_wait(tcw, fail_part):
    """if the driver refuses cuStreamWaitValue32 for some part of tcw_search_host's progressive
    read-back, the finished search must still be delivered whole (remaining parts by plain copies after the
    search) and nothing may hang.  The hook makes part (fail_part - 1) report CUDA_ERROR_NOT_SUPPORTED."""
    import torch
    w = tcw_inputs.make_workload("cfg3", fmt="u8").subgrid(sky=np.arange(0, 256, 256 // 56)[:56])
    grid = tcw.Grid.of(w)
    with tcw.Handle.from_workload(w) as h:
        stat, best = h.search(grid)
        torch.cuda.synchronize()
        want, bwant = stat.cpu().numpy(), best.cpu().numpy()
        h.set_option(tcw.TCW_OPT_DEBUG_FAIL_WAIT, fail_part)
        got, bgot = h.search_host(grid)
        assert h.info()["readback_parts"] == fail_part - 1           # parts that went back under the search
        assert np.array_equal(got, want) and np.array_equal(bgot, bwant)
        h.set_option(tcw.TCW_OPT_DEBUG_FAIL_WAIT, 0)
        got, bgot = h.search_host(grid)                              # and the handle is healthy afterwards
        assert h.info()["readback_parts"] > 1
        assert np.array_equal(got, want) and np.array_equal(bgot, bwant)


def test_group_range_takes_the_whole_grids_chunk_plan(tcw, cfg1):
    """whether the SFT axis is chunked fixes the float32 summation order, and the decision has two
    size limits that depend on the number of groups.  A range of groups must decide as its whole grid does, or
    tcw_search_groups would not be the slice of tcw_search bit for bit.  The hook lowers the scratch cap so that
    cfg1's whole grid (12 groups) is over it while a 6-group range alone would be under it."""
    import torch
    w = cfg1
    grid = tcw.Grid.of(w)
    with tcw.Handle.from_workload(w) as h:
        h.set_option(tcw.TCW_OPT_KERNEL, 2)
        h.set_option(tcw.TCW_OPT_CHUNK_ROWS, 64)                     # 256 SFTs -> 4 chunks where chunking is allowed
        stat_c, _ = h.search(grid)
        assert h.info()["chunks"] == 4
        h.set_option(tcw.TCW_OPT_DEBUG_CHUNK_SCRATCH, 4 * 9 * len(w.f0) * 4)      # room for 9 groups of partial sums
        stat, best = h.search(grid)
        assert h.info()["chunks"] <= 1                               # the whole grid does not chunk under the cap
        s, b = h.search_groups(grid, 3, 9)
        assert h.info()["chunks"] <= 1                               # ... so neither does a 6-group range
        torch.cuda.synchronize()
        assert torch.equal(s, stat.reshape(-1, len(w.f0))[3:9]) and torch.equal(b, best[3:9])
        # the two plans do differ in the last bits (else this test would prove nothing), within the float32 bar
        assert not torch.equal(stat_c, stat)
        assert torch.allclose(stat_c, stat, rtol=2e-6, atol=0)
