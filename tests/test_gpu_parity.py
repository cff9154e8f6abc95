"""GPU parity: the CUDA path (through the C ABI of libtcw.so) against oracle/, element by element.

Bars (BASELINE.json north_star):
  * tables g, D and bin indices k_j: bit-identical to the oracle
  * counts (u8 / bit-packed): bit-exact
  * power sums: |gpu - oracle| <= 1e-4 * max(1, |oracle|)
  * best per group: identical f0 index, except that where the two leading statistics differ by
    less than the tolerance either is accepted (checked as oracle_stat[gpu_argmax] >= max - tol)
"""
import dataclasses

import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload, detector_velocity, sky_vector

pytestmark = pytest.mark.gpu

TOL = 1e-4
KERNELS = {"auto": 0, "gather": 1, "staged": 2, "skyblock": 3}


@pytest.fixture(scope="module")
def tcw():
    import torch
    assert torch.cuda.is_available()
    import paper_2507_07816_b200 as pkg
    pkg.load_library()
    return pkg


def gpu_search(tcw, w, kernel="auto", f0_per_lane=0, host=False, sky_block=0, chunk_rows=0):
    import torch
    with tcw.Handle.from_workload(w, host=host) as h:
        h.set_option(tcw.TCW_OPT_KERNEL, KERNELS[kernel])
        h.set_option(tcw.TCW_OPT_CHUNK_ROWS, chunk_rows)
        h.set_option(tcw.TCW_OPT_F0_PER_LANE, f0_per_lane)
        h.set_option(tcw.TCW_OPT_SKY_BLOCK, sky_block)
        grid = tcw.Grid.of(w)
        stat, best = h.search(grid)
        torch.cuda.synchronize()
        info = h.info()
        assert info["status"] == 0
        if kernel != "auto":
            assert info["kernel"] == kernel
        bs, bi = h.best_fields(best)
        return stat.cpu().numpy().reshape(-1), bs, bi, info


def assert_stat_parity(w, got, want):
    if w.fmt == "f32":
        err = np.abs(got.astype(np.float64) - want)
        bound = TOL * np.maximum(1.0, np.abs(want))
        bad = np.nonzero(err > bound)[0]
        assert bad.size == 0, (bad[:5], got[bad[:5]], want[bad[:5]])
    else:
        assert got.dtype == np.int32
        assert np.array_equal(got.astype(np.int64), want), np.nonzero(got != want)[0][:5]


def assert_best_parity(w, n_f0, bs, bi, want_stat):
    """want_stat: oracle statistics [n_groups * n_f0] of the same groups, in order."""
    val, idx = oracle.best(want_stat, n_f0)
    ws = want_stat.reshape(-1, n_f0)
    assert np.all((bi >= 0) & (bi < n_f0))
    if w.fmt == "f32":
        tol = TOL * np.maximum(1.0, np.abs(val))
        assert np.all(np.abs(bs.astype(np.float64) - val) <= tol)
        at_gpu = ws[np.arange(len(bi)), bi]
        assert np.all(at_gpu >= val - tol)
        clear = np.array([np.sum(ws[g] >= val[g] - 2 * tol[g]) == 1 for g in range(len(val))])
        assert np.array_equal(bi[clear], idx[clear])
    else:
        assert np.array_equal(bs.astype(np.int64), val)
        assert np.array_equal(bi, idx)


def full_parity(tcw, w, kernel="auto", f0_per_lane=0, host=False, sky_block=0, chunk_rows=0):
    got, bs, bi, info = gpu_search(tcw, w, kernel, f0_per_lane, host, sky_block, chunk_rows)
    ref = oracle.evaluate(w)
    assert_stat_parity(w, got, ref.stat)
    assert_best_parity(w, len(w.f0), bs, bi, ref.stat)
    return got, ref, info


# ------------------------------------------------------------------ tables and indices
def test_tables_bit_identical_cfg1(tcw, cfg1):
    import torch
    with tcw.Handle.from_workload(cfg1) as h:
        grid = tcw.Grid.of(cfg1)
        h.search(grid)
        g, d = h.tables(grid)
    assert np.array_equal(g, oracle.spindown_table(cfg1.timestamps, cfg1.T0, cfg1.tau, cfg1.brk))
    assert np.array_equal(d, oracle.doppler_table(cfg1.velocities, cfg1.sky))


def test_spindown_table_bit_identical_large(tcw):
    """The whole g table of a cfg4-sized grid (64 tau x 9 n x 22.7k SFTs with gaps, ~13 M
    entries) against the oracle's correctly rounded values; D for 64 sky points."""
    rng = np.random.default_rng(5)
    present = np.ones(32400, dtype=bool)
    for _ in range(6):
        s = int(rng.integers(0, 30000))
        present[s:s + int(rng.integers(450, 2700))] = False
    ts = (8.0 * np.arange(32400) + 4.0)[present]
    vel = detector_velocity(ts)
    tau = np.geomspace(3500.0, 35000.0, 64)
    brk = 3.0 + 0.5 * np.arange(9)
    sky = tcw_inputs.fibonacci_sphere(64)
    spec = np.zeros((len(ts), 8), dtype=np.float32)
    w = Workload("tab", "f32", spec, len(ts), 8, 500.0, 8.0, ts, vel, 0.0, np.array([500.0]), tau, brk, sky)
    with tcw.Handle.from_workload(w) as h:
        grid = tcw.Grid.of(w)
        h.search(grid)
        g, d = h.tables(grid)
    want = oracle.spindown_table(ts, 0.0, tau, brk)
    diff = np.nonzero(g != want)
    assert diff[0].size == 0, (diff[0].size, g[diff][:3], want[diff][:3])
    assert np.array_equal(d, oracle.doppler_table(vel, sky))


def test_indices_identical_cfg1(tcw, cfg1):
    import torch
    ref = oracle.evaluate(cfg1, want_k=True)
    with tcw.Handle.from_workload(cfg1) as h:
        k = h.track_indices(tcw.Grid.of(cfg1), np.arange(cfg1.n_templates))
        torch.cuda.synchronize()
    assert np.array_equal(k.cpu().numpy(), ref.k)                     # all 196 608 lookups


def test_indices_with_exact_ties_zero_velocity(tcw, cfg1):
    """Zero velocity puts 11 lookups of cfg1 exactly on half-integers (tests/test_oracle_pins.py).
    Reading Q10: identical where unmasked, either neighbour where masked."""
    import torch
    w = dataclasses.replace(cfg1, velocities=np.zeros_like(cfg1.velocities))
    ref = oracle.evaluate(w, want_k=True)
    with tcw.Handle.from_workload(w) as h:
        k = h.track_indices(tcw.Grid.of(w), np.arange(w.n_templates))
        torch.cuda.synchronize()
    k = k.cpu().numpy()
    clean = ref.n_ambig == 0
    assert np.array_equal(k[clean], ref.k[clean])
    d = np.abs(k[~clean].astype(np.int64) - ref.k[~clean])
    assert d.max(initial=0) <= 1 and np.all((d != 0).sum(axis=1) <= ref.n_ambig[~clean])


def test_indices_T0_and_non_pow2_tsft(tcw):
    """T0 in the middle of the data (earlier SFTs are INT32_MIN) and T_sft = 10 s, which takes
    the three-multiply index path instead of the folded D*T one."""
    import torch
    rng = np.random.default_rng(9)
    n_sft, n_bins = 300, 900
    ts = 10.0 * np.arange(n_sft) + 5.0
    vel = detector_velocity(ts)
    rho = rng.standard_exponential((n_sft, n_bins)).astype(np.float32)
    w = Workload("t10", "f32", rho, n_sft, n_bins, 700.0, 10.0, ts, vel, 1000.0,
                 700.0 + 0.1 * np.arange(333), np.array([3500.0, 20000.0]), np.array([3.0, 4.5, 7.0]),
                 np.stack([sky_vector(1.0, 0.3), sky_vector(4.0, -1.1)]))
    ref = oracle.evaluate(w, want_k=True)
    with tcw.Handle.from_workload(w) as h:
        k = h.track_indices(tcw.Grid.of(w), np.arange(w.n_templates))
        torch.cuda.synchronize()
    assert np.array_equal(k.cpu().numpy(), ref.k)
    assert np.all(ref.k[:, :100] == np.iinfo(np.int32).min)
    for kernel in ("gather", "staged"):
        full_parity(tcw, w, kernel)
        full_parity(tcw, w.with_format("bits"), kernel)


# ------------------------------------------------------------------ the sum, every format and kernel
@pytest.mark.parametrize("kernel,r", [("gather", 0), ("staged", 8), ("staged", 4), ("auto", 0)])
@pytest.mark.parametrize("fmt", ["f32", "u8", "bits"])
def test_cfg1_full_parity(tcw, cfg1, fmt, kernel, r):
    full_parity(tcw, cfg1.with_format(fmt), kernel, r)


def test_u8_values_above_one_are_added_as_integers(tcw, cfg1):
    rng = np.random.default_rng(2)
    spec = rng.integers(0, 256, size=cfg1.spectrogram.shape).astype(np.uint8)
    w = dataclasses.replace(cfg1, fmt="u8", spectrogram=spec)
    for kernel in ("gather", "staged"):
        full_parity(tcw, w, kernel)


def ragged_workload(fmt="f32", seed=3):
    """Several f0 tiles with a ragged tail, an SFT count that is not a multiple of 32, gaps in
    the timestamps, f0 below and above the band, two sky points, T0 > first timestamp."""
    rng = np.random.default_rng(seed)
    slots = np.ones(1500, dtype=bool)
    slots[200:450] = False
    slots[900:1000] = False
    ts = (8.0 * np.arange(1500) + 4.0)[slots][:1131]
    n_sft, n_bins = len(ts), 1500
    rho = rng.standard_exponential((n_sft, n_bins)).astype(np.float32)
    f0 = 590.0 + 0.125 * np.arange(1900)                      # band is 600 .. 787.5 Hz
    w = Workload("ragged", "f32", rho, n_sft, n_bins, 600.0, 8.0, ts, detector_velocity(ts), 100.0,
                 f0, np.array([3500.0, 9000.0, 35000.0]), np.array([3.0, 5.0, 6.5]),
                 np.stack([sky_vector(1.0, 0.3), sky_vector(3.45, -0.41)]))
    return w.with_format(fmt)


@pytest.mark.parametrize("kernel,r", [("gather", 0), ("staged", 8), ("staged", 4)])
@pytest.mark.parametrize("fmt", ["f32", "u8", "bits"])
def test_ragged_edges_parity(tcw, fmt, kernel, r):
    w = ragged_workload(fmt)
    got, ref, info = full_parity(tcw, w, kernel, r)
    assert (ref.n_inband == 0).any() and (ref.n_inband > 500).any()
    if kernel == "staged":
        assert info["tile"] == 32 * r and info["ctas"] == w.n_groups * -(-len(w.f0) // (32 * r))


@pytest.mark.parametrize("fmt", ["f32", "u8", "bits"])
@pytest.mark.parametrize("chunk_rows,r", [(64, 8), (128, 4), (320, 16), (4096, 8)])
def test_sft_chunked_staged_parity(tcw, fmt, chunk_rows, r):
    """TCW_OPT_CHUNK_ROWS: (chunk, group, tile) CTAs + chunk_reduce_kernel.  The ragged workload has
    tiles that leave the band after a few chunks (dead CTAs), tiles never in band, a last chunk
    shorter than the others, and T0 > 0."""
    w = ragged_workload(fmt)
    got, ref, info = full_parity(tcw, w, "staged", r, chunk_rows=chunk_rows)
    rows = w.n_sft - int(np.searchsorted(w.timestamps, w.T0))
    want_chunks = -(-rows // chunk_rows) if chunk_rows < rows else 1
    assert info["chunks"] == want_chunks and info["ctas"] == want_chunks * w.n_groups * -(-len(w.f0) // (32 * r))
    assert info["launches"] == (5 if want_chunks > 1 else 4)
    # counts do not depend on the chunking at all; chunked power sums are run-to-run identical
    again, _, _, _ = gpu_search(tcw, w, "staged", r, chunk_rows=chunk_rows)
    assert np.array_equal(got, again)
    if fmt != "f32":
        plain, _, _, _ = gpu_search(tcw, w, "staged", r, chunk_rows=-1)
        assert np.array_equal(got, plain)


def test_sft_chunking_auto_only_for_large_spectrograms(tcw, cfg1):
    _, _, _, info = gpu_search(tcw, cfg1, "staged")
    assert info["chunks"] == 1
    with tcw.Handle.from_workload(cfg1) as h:
        with pytest.raises(tcw.TcwError):
            h.set_option(tcw.TCW_OPT_CHUNK_ROWS, -2)


def test_odd_band_start_and_tiny_sizes(tcw):
    """k_min odd and not a multiple of 4/16/128 (alignment of the staged window), n_bins not a
    multiple of 32, a single SFT, a single template."""
    rng = np.random.default_rng(4)
    ts = 8.0 * np.arange(77) + 4.0
    rho = rng.standard_exponential((77, 203)).astype(np.float32)
    w = Workload("odd", "f32", rho, 77, 203, 500.875, 8.0, ts, detector_velocity(ts), 0.0,
                 500.0 + 0.125 * np.arange(230), np.array([5000.0]), np.array([5.0]), sky_vector(0.2, 0.1)[None])
    for fmt in ("f32", "u8", "bits"):
        for kernel in ("gather", "staged"):
            full_parity(tcw, w.with_format(fmt), kernel)
    one = dataclasses.replace(w, spectrogram=rho[:1], n_sft=1, timestamps=ts[:1], velocities=w.velocities[:1],
                              f0=np.array([505.0]))
    for kernel in ("gather", "staged"):
        got, ref, _ = full_parity(tcw, one, kernel)
        assert got.shape == (1,)


def test_all_out_of_band_gives_zero_and_index_zero(tcw, cfg1):
    w = dataclasses.replace(cfg1, f0=400.0 + 0.125 * np.arange(40))       # entirely below the band
    for fmt in ("f32", "bits"):
        for kernel in ("gather", "staged"):
            got, bs, bi, _ = gpu_search(tcw, w.with_format(fmt), kernel)
            assert np.all(got == 0) and np.all(bs == 0) and np.all(bi == 0)
    w = dataclasses.replace(cfg1, f0=900.0 + 0.125 * np.arange(40))       # above the band for all 256 SFTs
    got, bs, bi, _ = gpu_search(tcw, w, "staged")
    assert np.all(got == 0) and np.all(bi == 0)


def test_sparse_f0_axis_falls_back_to_gather(tcw, cfg1):
    w = dataclasses.replace(cfg1, f0=505.0 + 25.0 * np.arange(5))         # 200 bins between templates
    w = dataclasses.replace(w, f0=np.concatenate([w.f0, 700.0 + 60.0 * np.arange(60)]))
    got, ref, info = full_parity(tcw, w, "auto")
    assert info["kernel"] == "gather"
    with tcw.Handle.from_workload(w) as h:
        h.set_option(tcw.TCW_OPT_KERNEL, 2)
        with pytest.raises(tcw.TcwError) as e:
            h.search(tcw.Grid.of(w))
        assert e.value.code == tcw.TCW_EUNSUPPORTED


def test_half_bin_f0_spacing_and_two_bin_spacing(tcw, cfg1):
    for step in (0.0625, 0.25, 0.3):
        w = dataclasses.replace(cfg1, f0=515.0 + step * np.arange(301))
        for fmt in ("f32", "bits"):
            full_parity(tcw, w.with_format(fmt), "staged")


def test_constant_spectrogram_counts_inband_sfts(tcw, cfg1):
    w = dataclasses.replace(cfg1, spectrogram=np.ones_like(cfg1.spectrogram))
    got, ref, _ = full_parity(tcw, w, "staged")
    assert np.array_equal(got, ref.n_inband.astype(np.float32))          # small integers: exact in float32


def test_injection_recovered_on_gpu(tcw, cfg1):
    f0 = np.sort(np.append(cfg1.f0, 550.0 + 0.125 * np.arange(-8, 9)))
    w = dataclasses.replace(cfg1, f0=f0, tau=np.array([3500.0, 5000.0, 9000.0]), brk=np.array([3.0, 5.0, 7.0]))
    got, bs, bi, _ = gpu_search(tcw, w)
    top = int(np.argmax(bs))
    assert top == 4 and f0[bi[top]] == 550.0


def test_outputs_optional_and_deterministic(tcw, cfg1):
    import torch
    with tcw.Handle.from_workload(cfg1) as h:
        grid = tcw.Grid.of(cfg1)
        s1, b1 = h.search(grid)
        s2, b2 = h.search(grid)
        s3, none_b = h.search(grid, want_best=False)
        none_s, b3 = h.search(grid, want_stat=False)
        torch.cuda.synchronize()
        assert none_b is None and none_s is None
        assert torch.equal(s1, s2) and torch.equal(b1, b2) and torch.equal(s1, s3) and torch.equal(b1, b3)
        with pytest.raises(tcw.TcwError) as e:
            h.search(grid, want_stat=False, want_best=False)
        assert e.value.code == tcw.TCW_EINVAL
        # a second, different grid on the same handle (scratch is reused / grown)
        g2 = tcw.Grid(cfg1.f0[:40], np.array([4000.0, 6000.0, 8000.0, 1e4, 2e4]), cfg1.brk, cfg1.sky, 0.0)
        s4, b4 = h.search(g2)
        torch.cuda.synchronize()
    w2 = dataclasses.replace(cfg1, f0=g2.f0, tau=g2.tau)
    assert_stat_parity(w2, s4.cpu().numpy().reshape(-1), oracle.evaluate(w2).stat)


def test_host_buffers_end_to_end(tcw, cfg1):
    """tcw_create from a HOST spectrogram and tcw_search_host into HOST outputs."""
    for fmt in ("f32", "bits"):
        w = cfg1.with_format(fmt)
        with tcw.Handle.from_workload(w, host=True) as h:
            stat, best = h.search_host(tcw.Grid.of(w))
        ref = oracle.evaluate(w)
        assert_stat_parity(w, stat.reshape(-1), ref.stat)
        bs, bi = h.best_fields(best)
        assert_best_parity(w, len(w.f0), bs, bi, ref.stat)


def test_strided_device_spectrogram(tcw, cfg1):
    """row_pitch_bytes larger than a row: the library re-lays the rows into its own pitch."""
    import torch
    wide = torch.full((cfg1.n_sft, cfg1.n_bins + 37), 1e9, dtype=torch.float32, device="cuda")
    wide[:, :cfg1.n_bins] = torch.from_numpy(cfg1.spectrogram).cuda()
    view = wide[:, :cfg1.n_bins]
    with tcw.Handle(view, "f32", cfg1.n_bins, cfg1.f_min, cfg1.T_sft, cfg1.timestamps, cfg1.velocities) as h:
        stat, _ = h.search(tcw.Grid.of(cfg1))
        torch.cuda.synchronize()
    assert_stat_parity(cfg1, stat.cpu().numpy().reshape(-1), oracle.evaluate(cfg1).stat)


@pytest.mark.parametrize("fmt", ["f32", "u8"])
def test_T0_after_the_last_sft_gives_empty_spans(tcw, cfg1, fmt):
    """Degenerate span: every SFT is before T0 (reading Q2), so every statistic is 0, the best index 0,
    Psi 0 and every bank template has no in-band SFT -- for each entry point and kernel."""
    import torch
    w = dataclasses.replace(cfg1.with_format(fmt), T0=float(cfg1.timestamps[-1]) + 1.0)
    ref = oracle.evaluate(w)
    assert not ref.stat.any() and not ref.n_inband.any()
    for kernel in ("staged", "gather"):
        got, bs, bi, _ = gpu_search(tcw, w, kernel=kernel)
        assert not got.any() and not bs.any() and not bi.any()
    many = dataclasses.replace(w, sky=tcw_inputs.fibonacci_cap(20, 1.0, 0.3, 5.0))
    if fmt == "u8":
        got, bs, bi, info = gpu_search(tcw, many)
        assert info["kernel"] == "skyblock" and not got.any() and not bi.any()
    with tcw.Handle.from_workload(w) as h:
        psi, stat, best = h.search_weighted(tcw.Grid.of(w), None, 1.0, 1.0)
        bstat, inband, _ = h.search_bank(w.f0, np.full(len(w.f0), 5000.0), np.full(len(w.f0), 5.0), w.sky[0], T0=w.T0)
        torch.cuda.synchronize()
        assert not psi.any().item() and not stat.any().item() and not best[:, 1].any().item()
        assert not bstat.any().item() and not inband.any().item()


@pytest.mark.parametrize("fmt", ["f32", "u8", "bits"])
def test_async_upload_gives_identical_results(tcw, fmt):
    """tcw_create_async: the first search runs chunk by chunk behind the upload pieces; results are
    bit-identical to a handle made by tcw_create, for the first search and for later ones, and for
    the other entry points whose first call has to wait for the whole upload."""
    import torch
    rng = np.random.default_rng(31)
    n_sft, n_bins = 1500, 6000            # 36 MB of float32: several 16 MB upload pieces
    ts = 8.0 * np.arange(n_sft) + 4.0
    rho = rng.standard_exponential((n_sft, n_bins)).astype(np.float32)
    w = tcw_inputs.Workload("async", "f32", rho, n_sft, n_bins, 500.0, 8.0, ts, tcw_inputs.detector_velocity(ts), 0.0,
                            500.0 + 0.125 * np.arange(3000), np.geomspace(3500.0, 35000.0, 3), np.array([3.0, 5.0]),
                            tcw_inputs.sky_vector(1.0, 0.3)[None]).with_format(fmt)
    grid = tcw.Grid.of(w)
    arr = np.ascontiguousarray(w.spectrogram)
    if arr.dtype == np.uint32:
        arr = arr.view(np.int32)
    pinned = torch.from_numpy(arr).pin_memory()
    with tcw.Handle(pinned, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities) as h0:
        h0.set_option(tcw.TCW_OPT_CHUNK_ROWS, 256)
        ref_stat, ref_best = h0.search(grid)
        ref_bank, _, _ = h0.search_bank(w.f0[:200], np.full(200, 9000.0), np.full(200, 4.0), w.sky[0])
        torch.cuda.synchronize()
    for first in ("search", "bank"):
        with tcw.Handle(pinned, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities, async_upload=True) as h:
            h.set_option(tcw.TCW_OPT_CHUNK_ROWS, 256)
            if first == "bank":
                bank, _, _ = h.search_bank(w.f0[:200], np.full(200, 9000.0), np.full(200, 4.0), w.sky[0])
                torch.cuda.synchronize()
                assert torch.equal(bank, ref_bank)
            stat, best = h.search(grid)
            torch.cuda.synchronize()
            info = h.info()
            assert info["chunks"] == 6 and info["status"] == 0
            assert torch.equal(stat, ref_stat) and torch.equal(best, ref_best)
            stat2, best2 = h.search(grid)             # upload long finished: single launch again
            torch.cuda.synchronize()
            assert torch.equal(stat2, ref_stat) and torch.equal(best2, ref_best)
            h.upload_wait()
    # a handle destroyed while its upload may still be in flight
    h = tcw.Handle(pinned, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities, async_upload=True)
    h.close()
