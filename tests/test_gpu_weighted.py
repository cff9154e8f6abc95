"""GPU parity of tcw_search_weighted (weighted statistic, critical ratio Psi of eq. (4),
PAPER.md:57-61) against oracle.evaluate_weighted, through the C ABI.

Bars:
  * s:   |gpu - oracle| <= 1e-4 * max(1, |oracle|)            (north_star's power tolerance)
  * Psi: |gpu - oracle| <= (1e-4 * max(1, |s|) + 1e-5 * |mean1| * W1) / sigma_s + 1e-5 * |Psi|
         -- the s tolerance carried through eq. (4), plus the float32 share of the weight sums
         (rows in which a tile straddles a band edge; per-chunk partial sums): both at most
         ~N_inband * 2^-24 relative, bounded here by 1e-5
  * best: max over f0 of Psi within the Psi tolerance; index identical unless another template
         lies within twice the tolerance of the maximum
"""
import dataclasses
import math

import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload, detector_velocity, sky_vector

from test_gpu_parity import KERNELS, tcw  # noqa: F401

pytestmark = pytest.mark.gpu

P_NU = math.exp(-1.6)
MOMENTS = {"f32": (1.0, 1.0), "u8": (P_NU, P_NU * (1 - P_NU)), "bits": (P_NU, P_NU * (1 - P_NU))}


def gpu_weighted(tcw, w, weights, mean1, var1, kernel="auto", f0_per_lane=0, chunk_rows=0, device_weights=False):
    import torch
    with tcw.Handle.from_workload(w) as h:
        h.set_option(tcw.TCW_OPT_KERNEL, KERNELS[kernel])
        h.set_option(tcw.TCW_OPT_CHUNK_ROWS, chunk_rows)
        h.set_option(tcw.TCW_OPT_F0_PER_LANE, f0_per_lane)
        grid = tcw.Grid.of(w)
        wts = torch.from_numpy(weights).cuda() if (device_weights and weights is not None) else weights
        psi, stat, best = h.search_weighted(grid, wts, mean1, var1)
        torch.cuda.synchronize()
        info = h.info()
        assert info["status"] == 0
        if kernel != "auto":
            assert info["kernel"] == kernel
        b = best.cpu().numpy()
        return (psi.cpu().numpy().reshape(-1), stat.cpu().numpy().reshape(-1),
                b[:, 0].copy().view(np.float32), b[:, 1].copy(), info)


def psi_tolerance(ref, mean1, var1):
    sigma = np.sqrt(var1 * ref.w2)
    with np.errstate(divide="ignore", invalid="ignore"):
        tol = (1e-4 * np.maximum(1.0, np.abs(ref.s)) + 1e-5 * abs(mean1) * ref.w1) / sigma + 1e-5 * np.abs(ref.psi)
    return np.where(ref.w2 > 0, tol, 0.0)


def assert_weighted_parity(w, ref, mean1, var1, psi, stat, bs, bi):
    n_f0 = len(w.f0)
    err = np.abs(stat.astype(np.float64) - ref.s)
    assert np.all(err <= 1e-4 * np.maximum(1.0, np.abs(ref.s))), float(err.max())
    tol = psi_tolerance(ref, mean1, var1)
    perr = np.abs(psi.astype(np.float64) - ref.psi)
    bad = np.nonzero(perr > tol)[0]
    assert bad.size == 0, (bad[:5], psi[bad[:5]], ref.psi[bad[:5]], tol[bad[:5]])
    val, idx = oracle.best(ref.psi, n_f0)
    rp, rt = ref.psi.reshape(-1, n_f0), tol.reshape(-1, n_f0)
    gtol = rt.max(axis=1)
    assert np.all((bi >= 0) & (bi < n_f0))
    assert np.all(np.abs(bs.astype(np.float64) - val) <= gtol)
    assert np.all(rp[np.arange(len(bi)), bi] >= val - gtol)
    clear = np.array([np.sum(rp[g] >= val[g] - 2 * gtol[g]) == 1 for g in range(len(val))])
    assert np.array_equal(bi[clear], idx[clear])
    # the GPU's own outputs are consistent: best is the maximum of its psi, lowest index on ties
    gp = psi.reshape(-1, n_f0)
    assert np.array_equal(bs, gp.max(axis=1)) and np.array_equal(bi, gp.argmax(axis=1))


@pytest.mark.parametrize("fmt", ["f32", "u8", "bits"])
@pytest.mark.parametrize("kernel", ["staged", "gather"])
def test_cfg1_weighted_parity(tcw, cfg1, fmt, kernel):
    w = cfg1.with_format(fmt)
    wt = tcw_inputs.synthetic_weights(w.sky, w.timestamps, w.seed)
    mean1, var1 = MOMENTS[fmt]
    ref = oracle.evaluate_weighted(w, wt, mean1, var1)
    psi, stat, bs, bi, _ = gpu_weighted(tcw, w, wt, mean1, var1, kernel=kernel)
    assert_weighted_parity(w, ref, mean1, var1, psi, stat, bs, bi)


def test_unit_weights_match_the_plain_search_bit_for_bit(tcw, cfg1):
    """weights = NULL: fma(1, v, acc) = acc + v, so s is bit-identical to the statistic of a plain search that
    adds the rows in the same order -- one at a time, which is what tcw_search does in its general-f0
    instantiation (TCW_OPT_GENERAL_F0); the equally-spaced-f0 instantiation adds rows in pairs
    (acc += row_q + row_q+1) and agrees to float32 rounding.
    Psi = (s - N_inband)/sqrt(N_inband)."""
    import torch
    with tcw.Handle.from_workload(cfg1) as h:
        grid = tcw.Grid.of(cfg1)
        paired, _ = h.search(grid)
        paired = paired.clone()
        h.set_option(tcw.TCW_OPT_GENERAL_F0, 1)
        plain, _ = h.search(grid)
        h.set_option(tcw.TCW_OPT_GENERAL_F0, 0)
        psi, stat, _ = h.search_weighted(grid, None, 1.0, 1.0)
        torch.cuda.synchronize()
        assert torch.equal(plain, stat)
        # kernel-vs-kernel, not an oracle tolerance (reason in DESIGN.md section 7, "paired rows"): the two
        # instantiations add the same float32 values in two fixed orders; 2e-6 is a few float32 ulps (2^-24 = 6e-8
        # per add, partial cancellation over the 256 rows of cfg1).  Both are held to 1e-4 against the oracle elsewhere.
        assert torch.allclose(paired, stat, rtol=2e-6, atol=2e-6)
    ref = oracle.evaluate(cfg1)
    n = ref.n_inband.astype(np.float64)
    want = (stat.cpu().numpy().reshape(-1).astype(np.float64) - n) / np.sqrt(n)
    assert np.allclose(psi.cpu().numpy().reshape(-1), want, rtol=2e-6, atol=2e-6)


@pytest.mark.parametrize("f0_per_lane", [4, 8, 16])
def test_ragged_grid_gaps_T0_and_nonpow2_T(tcw, f0_per_lane):
    """n_f0 not a multiple of the tile, timestamps with holes, T0 inside the data, T_sft = 10 s
    (the unfolded index path), three sky points with their own weight rows, tracks leaving the band
    at the bottom and entering it from above (both band edges straddled)."""
    rng = np.random.default_rng(77)
    n_slots, n_bins, T = 700, 1500, 10.0
    keep = np.ones(n_slots, dtype=bool)
    keep[100:180] = False
    keep[400:403] = False
    ts = (T * np.arange(n_slots) + 5.0)[keep]
    rho = rng.standard_exponential((len(ts), n_bins)).astype(np.float32)
    f0 = 500.0 + 0.1 * np.arange(0, 1731)              # up to 673 Hz: the top 230 templates start above the band (650 Hz)
    sky = np.stack([sky_vector(1.0, 0.3), sky_vector(2.5, -0.7), sky_vector(4.0, 1.1)])
    w = Workload("ragged", "f32", rho, len(ts), n_bins, 500.0, T, ts, detector_velocity(ts), 1000.0,
                 f0, np.array([3500.0, 20000.0]), np.array([3.0, 6.5]), sky)
    wt = tcw_inputs.synthetic_weights(sky, ts, 3)
    wt[1, 50:60] = 0.0
    ref = oracle.evaluate_weighted(w, wt, 1.0, 1.0)
    # coverage: templates never in band (W2 = 0 -> Psi = 0), templates entering from above, leaving below
    assert 0 < (ref.w1 == 0).sum() < ref.w1.size // 4
    for dev_w in (False, True):
        psi, stat, bs, bi, info = gpu_weighted(tcw, w, wt, 1.0, 1.0, kernel="staged", f0_per_lane=f0_per_lane,
                                               device_weights=dev_w)
        assert info["tile"] == 32 * f0_per_lane
        assert_weighted_parity(w, ref, 1.0, 1.0, psi, stat, bs, bi)


@pytest.mark.parametrize("fmt", ["f32", "u8"])
def test_chunked_weighted_search(tcw, cfg1, fmt):
    """SFT chunks (the cfg2/cfg4 launch configuration): per-chunk partial s, W1, W2 added in order."""
    w = cfg1.with_format(fmt)
    wt = tcw_inputs.synthetic_weights(w.sky, w.timestamps, 21)
    mean1, var1 = MOMENTS[fmt]
    ref = oracle.evaluate_weighted(w, wt, mean1, var1)
    psi, stat, bs, bi, info = gpu_weighted(tcw, w, wt, mean1, var1, kernel="staged", chunk_rows=64)
    assert info["chunks"] == 4
    assert_weighted_parity(w, ref, mean1, var1, psi, stat, bs, bi)
    # chunking changes only the order of the float32 additions
    psi1, stat1, _, _, info1 = gpu_weighted(tcw, w, wt, mean1, var1, kernel="staged", chunk_rows=-1)
    assert info1["chunks"] == 1
    assert np.allclose(stat, stat1, rtol=1e-5, atol=1e-5)


def test_template_never_in_band_has_zero_psi(tcw):
    rho = np.ones((64, 256), dtype=np.float32)
    ts = 8.0 * np.arange(64) + 4.0
    f0 = 400.0 + 0.125 * np.arange(64)                  # all below the band (500 Hz)
    w = Workload("below", "f32", rho, 64, 256, 500.0, 8.0, ts, np.zeros((64, 3)), 0.0, f0,
                 np.array([5000.0]), np.array([5.0]), sky_vector(1.0, 0.3)[None, :])
    for kernel in ("staged", "gather"):
        psi, stat, bs, bi, _ = gpu_weighted(tcw, w, None, 1.0, 1.0, kernel=kernel)
        assert np.all(psi == 0) and np.all(stat == 0) and bs[0] == 0 and bi[0] == 0


def test_weighted_argument_errors(tcw, cfg1):
    with tcw.Handle.from_workload(cfg1) as h:
        grid = tcw.Grid.of(cfg1)
        for mean1, var1 in ((1.0, 0.0), (1.0, -1.0), (float("nan"), 1.0), (1.0, float("inf"))):
            with pytest.raises(tcw.TcwError) as e:
                h.search_weighted(grid, None, mean1, var1)
            assert e.value.code == tcw.TCW_EINVAL
        with pytest.raises(tcw.TcwError) as e:
            h.search_weighted(grid, None, 1.0, 1.0, want_psi=False, want_stat=False, want_best=False)
        assert e.value.code == tcw.TCW_EINVAL
    with tcw.Handle.from_workload(cfg1.with_format("u8")) as h:
        h.set_option(tcw.TCW_OPT_KERNEL, KERNELS["skyblock"])
        with pytest.raises(tcw.TcwError) as e:
            h.search_weighted(tcw.Grid.of(cfg1), None, 1.0, 1.0)
        assert e.value.code == tcw.TCW_EUNSUPPORTED


def test_cfg2_weighted_full_grid_sampled_groups(tcw):
    """cfg2 at full size in the bench's launch configuration (chunked staged kernel), weighted."""
    w = tcw_inputs.make_workload("cfg2")
    wt = tcw_inputs.synthetic_weights(w.sky, w.timestamps, w.seed)
    psi, stat, bs, bi, info = gpu_weighted(tcw, w, wt, 1.0, 1.0)
    assert info["kernel"] == "staged" and info["chunks"] > 1
    n_f0 = len(w.f0)
    groups = np.array([0, 4, 37, 80, 121, 159])
    ref = oracle.evaluate_weighted(w, wt, 1.0, 1.0, sel=oracle.group_templates(w, groups))
    sel = (groups[:, None] * n_f0 + np.arange(n_f0)[None, :]).reshape(-1)
    assert_weighted_parity(w, ref, 1.0, 1.0, psi[sel], stat[sel], bs[groups], bi[groups])
    gp = psi.reshape(-1, n_f0)
    assert np.array_equal(bs, gp.max(axis=1)) and np.array_equal(bi, gp.argmax(axis=1))
    # the 20 injections (+2.0 per bin) stand far above the noise distribution of Psi (unit variance)
    assert bs.max() > 20.0 and np.isfinite(psi).all()


def test_multi_sky_count_weighted_uses_staged_kernel(tcw):
    """Count format with many sky points: the plain search takes the sky-block kernel, the weighted
    one the per-sky staged kernel (weights differ per sky point)."""
    w = tcw_inputs.make_workload("cfg3", fmt="u8")
    w = w.subgrid(tau=slice(0, 2), brk=slice(0, 2), sky=slice(0, 24), f0=slice(0, 1024))
    wt = tcw_inputs.synthetic_weights(w.sky, w.timestamps, 8)
    mean1, var1 = MOMENTS["u8"]
    psi, stat, bs, bi, info = gpu_weighted(tcw, w, wt, mean1, var1)
    assert info["kernel"] == "staged"
    groups = np.array([0, 5, 50, 95])
    n_f0 = len(w.f0)
    ref = oracle.evaluate_weighted(w, wt, mean1, var1, sel=oracle.group_templates(w, groups))
    sel = (groups[:, None] * n_f0 + np.arange(n_f0)[None, :]).reshape(-1)
    assert_weighted_parity(w, ref, mean1, var1, psi[sel], stat[sel], bs[groups], bi[groups])


@pytest.mark.parametrize("fmt", ["f32", "u8"])
def test_weighted_box_copies_are_bit_identical_to_row_copies(tcw, fmt):
    """The weighted instantiation stages ring slots by one tensor-map copy like the unweighted one (its weights and
    band-edge constants live in a second metadata ring); with TCW_OPT_ROW_COPIES it stages row by row.  Same
    arithmetic in the same order: Psi, s and the best templates must agree bit for bit (cfg1 with and without SFT
    chunks, which exercises whole-tile rows, band-edge rows and rows past the band)."""
    import torch
    w = tcw_inputs.make_workload("cfg1")
    if fmt != "f32":
        w = w.with_format(fmt)
    wts = tcw_inputs.synthetic_weights(w.sky, w.timestamps, 5)
    mean1, var1 = MOMENTS[fmt]
    for chunk in (0, 64):
        out = []
        for row_copies in (0, 1):
            with tcw.Handle.from_workload(w) as h:
                h.set_option(tcw.TCW_OPT_KERNEL, KERNELS["staged"])
                h.set_option(tcw.TCW_OPT_CHUNK_ROWS, chunk)
                h.set_option(tcw.TCW_OPT_ROW_COPIES, row_copies)
                psi, stat, best = h.search_weighted(tcw.Grid.of(w), wts, mean1, var1)
                torch.cuda.synchronize()
                info = h.info()
                assert info["status"] == 0 and info["box_copies"] == 1 - row_copies, info
                out.append((psi.cpu().numpy().view(np.uint32), stat.cpu().numpy().view(np.uint32), best.cpu().numpy().view(np.uint8)))
        for a, b in zip(out[0], out[1]):
            assert np.array_equal(a, b)
