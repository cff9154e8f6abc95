"""GPU parity of the sky-block kernel (csrc/tcw_skyblock.cuh): exact sharing of lookups between
neighbouring sky points for the count formats.

The kernel's claim is bit-exactness: monotonicity of rint(a*d) in d lets one lookup serve every sky
point of a block whose two extreme Doppler factors select the same bin, and the rest is resolved
per sky point in integer arithmetic.  So every comparison here is array equality -- against the
oracle at sizes it finishes in seconds, and against the per-sky staged kernel at full size.
"""
import dataclasses

import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload, detector_velocity, fibonacci_cap, fibonacci_sphere

from test_gpu_parity import assert_best_parity, assert_stat_parity, full_parity, gpu_search, ragged_workload, tcw  # noqa: F401

pytestmark = pytest.mark.gpu


def sky_workload(cfg1, sky, fmt="u8", **kw):
    return dataclasses.replace(cfg1, sky=np.ascontiguousarray(sky), **kw).with_format(fmt)


@pytest.mark.parametrize("sky_block", [64, 128])
@pytest.mark.parametrize("fmt", ["u8", "bits"])
def test_cfg1_cap_of_70_sky_points(tcw, cfg1, fmt, sky_block):
    """70 sky points (a ragged block: 64 + 6, or 70 of 128) in a 10-degree cap."""
    w = sky_workload(cfg1, fibonacci_cap(70, 3.45, -0.41, 10.0), fmt)
    got, ref, info = full_parity(tcw, w, "skyblock", sky_block=sky_block)
    assert info["sky_block"] == sky_block and info["ctas"] == -(-70 // sky_block) * 12 * 1


def test_cfg1_full_sphere_unsorted_sky(tcw, cfg1):
    """150 points over the whole sphere in random order (Doppler spread +-0.4 bin at 520 Hz).
    Blocks are formed by the library's own sort, so the caller's order must not matter."""
    rng = np.random.default_rng(11)
    sky = fibonacci_sphere(150)[rng.permutation(150)]
    w = sky_workload(cfg1, sky, "u8")
    full_parity(tcw, w, "skyblock")
    # the same search in the caller's sorted order gives the same numbers at permuted places
    order = np.argsort(sky[:, 2])
    got_a, _, _, _ = gpu_search(tcw, w, "skyblock")
    got_b, _, _, _ = gpu_search(tcw, dataclasses.replace(w, sky=np.ascontiguousarray(sky[order])), "skyblock")
    n = len(w.tau) * len(w.brk) * len(w.f0)
    assert np.array_equal(got_a.reshape(150, n)[order], got_b.reshape(150, n))


def test_wide_doppler_spread_many_bins_apart(tcw):
    """High band (k_min = 80 000, i.e. 10 kHz) so that the full-sphere Doppler spread is +-8 bins:
    the two ends of a block are several bins apart and the generic per-sky resolve path runs."""
    rng = np.random.default_rng(12)
    n_sft, n_bins = 200, 1500
    ts = 8.0 * np.arange(n_sft) + 4.0
    nu = (rng.random((n_sft, n_bins)) < 0.3).astype(np.uint8)
    w = Workload("wide", "u8", nu, n_sft, n_bins, 10000.0, 8.0, ts, detector_velocity(ts), 0.0,
                 10020.0 + 0.125 * np.arange(700), np.array([4000.0, 30000.0]), np.array([3.0, 5.0]),
                 fibonacci_sphere(40))
    full_parity(tcw, w, "skyblock")
    full_parity(tcw, w, "skyblock", sky_block=128)


def test_u8_values_above_one_and_ragged_edges(tcw):
    """General uint8 values (reading Q20), several f0 tiles with a ragged tail, gaps in the
    timestamps, T0 > first timestamp, templates below and above the band, 33 sky points."""
    w = ragged_workload("u8")
    rng = np.random.default_rng(13)
    spec = rng.integers(0, 256, size=w.spectrogram.shape).astype(np.uint8)
    w = dataclasses.replace(w, spectrogram=spec, sky=fibonacci_cap(33, 1.0, 0.3, 25.0))
    got, ref, info = full_parity(tcw, w, "skyblock")
    assert info["tile"] == 512 and (ref.n_inband == 0).any()
    full_parity(tcw, w, "skyblock", sky_block=128)


def test_non_pow2_tsft_and_single_sky_point(tcw):
    """T_sft = 10 s takes the unfolded ((f0*g)*D)*T path; one sky point is a block of duplicates."""
    rng = np.random.default_rng(14)
    n_sft, n_bins = 300, 900
    ts = 10.0 * np.arange(n_sft) + 5.0
    nu = (rng.random((n_sft, n_bins)) < 0.2).astype(np.uint8)
    w = Workload("t10", "u8", nu, n_sft, n_bins, 700.0, 10.0, ts, detector_velocity(ts), 1000.0,
                 700.0 + 0.1 * np.arange(333), np.array([3500.0, 20000.0]), np.array([3.0, 4.5, 7.0]),
                 fibonacci_cap(20, 4.0, -1.1, 15.0))
    full_parity(tcw, w, "skyblock")
    full_parity(tcw, dataclasses.replace(w, sky=w.sky[:1].copy()), "skyblock")


def test_auto_picks_skyblock_for_counts_only(tcw, cfg1):
    sky = fibonacci_cap(16, 1.0, 0.3, 5.0)
    _, _, info = full_parity(tcw, sky_workload(cfg1, sky, "bits"), "auto")
    assert info["kernel"] == "skyblock"
    _, _, info = full_parity(tcw, sky_workload(cfg1, sky[:15], "bits"), "auto")
    assert info["kernel"] == "staged"
    _, _, info = full_parity(tcw, sky_workload(cfg1, sky, "f32"), "auto")
    assert info["kernel"] == "staged"
    with tcw.Handle.from_workload(sky_workload(cfg1, sky, "f32")) as h:
        h.set_option(tcw.TCW_OPT_KERNEL, 3)
        with pytest.raises(tcw.TcwError) as e:
            h.search(tcw.Grid.of(cfg1))
        assert e.value.code == tcw.TCW_EUNSUPPORTED


def test_constant_spectrogram_counts_inband_sfts(tcw, cfg1):
    w = sky_workload(cfg1, fibonacci_cap(64, 1.0, 0.3, 10.0), "u8")
    w = dataclasses.replace(w, spectrogram=np.ones_like(w.spectrogram))
    got, ref, _ = full_parity(tcw, w, "skyblock")
    assert np.array_equal(got, ref.n_inband)


def staged_vs_skyblock(tcw, w, sky_block=0):
    got_s, bs_s, bi_s, _ = gpu_search(tcw, w, "staged")
    got_b, bs_b, bi_b, info = gpu_search(tcw, w, "skyblock", sky_block=sky_block)
    assert np.array_equal(got_s, got_b)
    assert np.array_equal(bs_s, bs_b) and np.array_equal(bi_s, bi_b)
    return got_b, bs_b, bi_b, info


@pytest.mark.parametrize("sky_block", [64, 128])
def test_cfg3_whole_sky_patch_equals_per_sky_kernel(tcw, sky_block):
    """cfg3's data and all 256 sky points of its cap, all 4000 f0, a 2 x 2 slice of (tau, n):
    4.1 M templates x 10 800 SFTs.  Bit-identical to the per-sky staged kernel everywhere, and to
    the oracle on sampled whole groups."""
    w = tcw_inputs.make_workload("cfg3", fmt="u8").subgrid(tau=[0, 15], brk=[0, 3])
    got, bs, bi, info = staged_vs_skyblock(tcw, w, sky_block)
    assert info["ctas"] == (256 // sky_block) * 4 * -(-4000 // info["tile"])
    groups = np.array([0, 3, 517, 1023])
    ref = oracle.evaluate(w, sel=oracle.group_templates(w, groups))
    assert_stat_parity(w, got.reshape(-1, 4000)[groups].reshape(-1), ref.stat)
    assert_best_parity(w, 4000, bs[groups], bi[groups], ref.stat)


def test_cfg5_all_sky_subset_equals_per_sky_kernel(tcw):
    """cfg5's data (band from 1000 Hz, non-stationary floor, bit-packed) with 300 of its 4096
    full-sphere sky points in the generator's (unsorted) order, one tau, two n."""
    w = tcw_inputs.make_workload("cfg5").subgrid(tau=[3], brk=[0, 2], sky=np.arange(0, 4096, 13)[:300])
    got, bs, bi, info = staged_vs_skyblock(tcw, w)
    groups = np.array([0, 299, 598])
    ref = oracle.evaluate(w, sel=oracle.group_templates(w, groups))
    assert_stat_parity(w, got.reshape(-1, 4000)[groups].reshape(-1), ref.stat)


def _sky_search(tcw, w, sky_block):
    import torch
    with tcw.Handle.from_workload(w) as h:
        h.set_option(tcw.TCW_OPT_KERNEL, 3)
        h.set_option(tcw.TCW_OPT_SKY_BLOCK, sky_block)
        stat, best = h.search(tcw.Grid.of(w))
        torch.cuda.synchronize()
        info = h.info()
        assert info["status"] == 0 and info["kernel"] == "skyblock" and info["sky_block"] == sky_block
        return stat.cpu().numpy(), best.cpu().numpy()


def test_two_level_blocks_of_256_equal_blocks_of_64_and_the_oracle(tcw, cfg1):
    """The two-level kernel (256 sky points = 4 sub-blocks of 64, packed int16 corrections) on
    bit-packed input: bit-identical to the 64-point kernel and to the oracle -- a 10-degree cap
    (mostly level-0 agreement), the full sphere in arbitrary order (levels 1 and 2 busy), a ragged
    block (300 sky points) and a ragged f0 tile."""
    import oracle
    for sky in (tcw_inputs.fibonacci_cap(300, 3.45, -0.41, 10.0),
                tcw_inputs.fibonacci_sphere(512)[np.random.default_rng(3).permutation(512)]):
        w = dataclasses.replace(cfg1.with_format("bits"), sky=sky, f0=520.0 + 0.125 * np.arange(300),
                                tau=cfg1.tau[:2], brk=cfg1.brk[:2])
        s256, b256 = _sky_search(tcw, w, 256)
        s64, b64 = _sky_search(tcw, w, 64)
        assert np.array_equal(s256, s64) and np.array_equal(b256, b64)
        groups = np.array([0, 3, w.n_groups // 2, w.n_groups - 1])
        ref = oracle.evaluate(w, sel=oracle.group_templates(w, groups))
        got = s256.reshape(-1, len(w.f0))[groups].reshape(-1)
        assert np.array_equal(got.astype(np.int64), ref.stat)


def test_two_level_blocks_need_small_counts(tcw, cfg1):
    """The packed int16 corrections are exact while n_sft * (largest count) < 2^15: uint8 data with 0/1
    values take the two-level kernel like bit-packed data; large counts are refused (and auto falls
    back to 64-point blocks)."""
    import torch
    sky = tcw_inputs.fibonacci_cap(300, 3.45, -0.41, 10.0)
    w = dataclasses.replace(cfg1.with_format("u8"), sky=sky)
    s256, b256 = _sky_search(tcw, w, 256)
    s64, b64 = _sky_search(tcw, w, 64)
    assert np.array_equal(s256, s64) and np.array_equal(b256, b64)
    big = dataclasses.replace(w, spectrogram=(w.spectrogram * 200).astype(np.uint8))      # 256 SFTs x 200 > 32767
    with tcw.Handle.from_workload(big) as h:
        h.set_option(tcw.TCW_OPT_SKY_BLOCK, 256)
        with pytest.raises(tcw.TcwError) as e:
            h.search(tcw.Grid.of(big))
        assert e.value.code == tcw.TCW_EUNSUPPORTED
        h.set_option(tcw.TCW_OPT_SKY_BLOCK, 0)
        stat, _ = h.search(tcw.Grid.of(big))
        torch.cuda.synchronize()
        assert h.info()["sky_block"] == 64
        assert np.array_equal(stat.cpu().numpy(), 200 * s64)


def test_cfg3_bits_whole_patch_two_level_equals_64(tcw):
    """cfg3's whole sky patch (256 points = one block) on a slice of the (tau, n) axes, 4000 f0."""
    w = tcw_inputs.make_workload("cfg3", fmt="bits").subgrid(tau=slice(0, 16, 5), brk=slice(0, 5, 2))
    s256, b256 = _sky_search(tcw, w, 256)
    s64, b64 = _sky_search(tcw, w, 64)
    assert np.array_equal(s256, s64) and np.array_equal(b256, b64)
