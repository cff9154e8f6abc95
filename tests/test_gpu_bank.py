"""GPU parity of tcw_search_bank (random template bank, PAPER.md:63 (ii)) against
oracle.evaluate_bank, through the C ABI.

Bars: bin indices identical to the oracle (except where the oracle flags a lookup within 1e-9 bin
of a half-integer, reading Q10), counts and in-band counts bit-exact, power sums within
1e-4 * max(1, |oracle|).
"""
import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload, detector_velocity, sky_vector

from test_gpu_parity import TOL, tcw  # noqa: F401

pytestmark = pytest.mark.gpu


def gpu_bank(tcw, w, f0, tau, brk, sky, want_k=True):
    import torch
    with tcw.Handle.from_workload(w) as h:
        stat, inband, k = h.search_bank(f0, tau, brk, sky, T0=w.T0, want_k=want_k)
        torch.cuda.synchronize()
        info = h.info()
        assert info["kernel"] == "bank" and info["status"] == 0
        n_exact = h.counter(0)
        return (stat.cpu().numpy(), inband.cpu().numpy(), k.cpu().numpy() if k is not None else None, n_exact)


def assert_bank_parity(w, ref, stat, inband, k):
    clean = ref.n_ambig == 0
    assert clean.mean() > 0.99
    if k is not None:
        assert np.array_equal(k[clean], ref.k[clean])
    assert np.array_equal(inband[clean], ref.n_inband[clean])
    if w.fmt == "f32":
        err = np.abs(stat.astype(np.float64) - ref.stat)
        assert np.all(err[clean] <= TOL * np.maximum(1.0, np.abs(ref.stat[clean]))), float(err.max())
    else:
        assert stat.dtype == np.int32
        assert np.array_equal(stat[clean].astype(np.int64), ref.stat[clean])


@pytest.mark.parametrize("fmt", ["f32", "u8", "bits"])
@pytest.mark.parametrize("shared", [True, False])
def test_cfg1_random_bank_parity(tcw, cfg1, fmt, shared):
    w = cfg1.with_format(fmt)
    f0, tau, brk, sky = tcw_inputs.random_bank(1500, 480.0, 640.0, 5, sky=w.sky[0] if shared else None)
    ref = oracle.evaluate_bank(w, f0, tau, brk, sky, want_k=True)
    stat, inband, k, n_exact = gpu_bank(tcw, w, f0, tau, brk, sky)
    assert_bank_parity(w, ref, stat, inband, k)
    assert n_exact < 1000                      # the defining chain is the rare path


def test_bank_built_from_the_grid_matches_tcw_search(tcw, cfg1):
    """The same templates through both entry points: identical indices, hence identical counts."""
    import torch
    w = cfg1.with_format("u8")
    s, a, b, i = np.meshgrid(np.arange(len(w.sky)), np.arange(len(w.tau)), np.arange(len(w.brk)),
                             np.arange(len(w.f0)), indexing="ij")
    f0, tau, brk = w.f0[i.ravel()], w.tau[a.ravel()], w.brk[b.ravel()]
    stat, inband, k, _ = gpu_bank(tcw, w, f0, tau, brk, w.sky[0])
    with tcw.Handle.from_workload(w) as h:
        grid = tcw.Grid.of(w)
        gstat, _ = h.search(grid)
        gk = h.track_indices(grid, np.arange(w.n_templates))
        torch.cuda.synchronize()
    assert np.array_equal(k, gk.cpu().numpy())
    assert np.array_equal(stat, gstat.cpu().numpy().reshape(-1))


def test_bank_exact_points_gaps_T0_nonpow2(tcw):
    """Inputs that land exactly on integers and half-integers (the defining chain must decide them),
    T_sft = 10 s, holes in the timestamps, T0 inside the data, templates above and below the band."""
    rng = np.random.default_rng(4)
    # exact powers: base 16 with n = 5 gives g = 1/2, base 4 with n = 3 gives g = 1/2 (zero velocity)
    ts = np.array([0.0, 15000.0, 75000.0, 75008.0, 90000.0])
    rho = rng.standard_exponential((len(ts), 4200)).astype(np.float32)
    w = Workload("exact", "f32", rho, len(ts), 4200, 500.0, 8.0, ts, np.zeros((len(ts), 3)), 0.0,
                 np.array([1000.0]), np.array([5000.0]), np.array([5.0]), np.array([[1.0, 0.0, 0.0]]))
    f0 = np.array([1000.0, 1000.0, 1000.125, 1000.0625, 8000.0625 / 8.0, 400.0, 2000.0])
    tau = np.array([5000.0, 5000.0, 5000.0, 5000.0, 1e9, 5000.0, 5000.0])
    brk = np.array([5.0, 3.0, 5.0, 5.0, 5.0, 5.0, 5.0])
    sky = np.array([1.0, 0.0, 0.0])
    ref = oracle.evaluate_bank(w, f0, tau, brk, sky, want_k=True)
    assert ref.k[0, 2] == 0 and ref.k[1, 1] == 0          # x = 4000 exactly
    stat, inband, k, n_exact = gpu_bank(tcw, w, f0, tau, brk, sky)
    assert n_exact > 0
    ok = ref.n_ambig == 0
    assert np.array_equal(k[ok], ref.k[ok]) and np.array_equal(inband[ok], ref.n_inband[ok])
    # exact ties: x = 4000.5 at (template 2, SFT 2) and x = 8000.5 at (template 3, SFT 0); the
    # defining chain rounds them to even like the oracle
    assert ref.n_ambig[2] == 1 and ref.n_ambig[3] == 1
    assert k[2, 2] == ref.k[2, 2] == 0 and k[3, 0] == ref.k[3, 0] == 4000

    n_slots, n_bins, T = 500, 1200, 10.0
    keep = np.ones(n_slots, dtype=bool)
    keep[60:140] = False
    tsg = (T * np.arange(n_slots) + 5.0)[keep]
    rho = rng.standard_exponential((len(tsg), n_bins)).astype(np.float32)
    wg = Workload("gaps", "f32", rho, len(tsg), n_bins, 500.0, T, tsg, detector_velocity(tsg), 400.0,
                  np.array([500.0]), np.array([5000.0]), np.array([5.0]), sky_vector(1.0, 0.3)[None, :])
    f0, tau, brk, sky = tcw_inputs.random_bank(700, 470.0, 660.0, 12)
    ref = oracle.evaluate_bank(wg, f0, tau, brk, sky, want_k=True)
    assert (ref.n_inband == 0).any() and (ref.k[:, 80] >= n_bins).any()
    stat, inband, k, _ = gpu_bank(tcw, wg, f0, tau, brk, sky)
    assert_bank_parity(wg, ref, stat, inband, k)


def test_bank_argument_errors(tcw, cfg1):
    with tcw.Handle.from_workload(cfg1) as h:
        good = dict(f0=[600.0], tau=[5000.0], brk=[5.0], sky=[1.0, 0.0, 0.0])
        for key, val in (("f0", [-1.0]), ("tau", [0.0]), ("brk", [1.0]), ("sky", [1.0, 1.0, 0.0]), ("f0", [1e12])):
            args = dict(good)
            args[key] = val
            with pytest.raises(tcw.TcwError) as e:
                h.search_bank(**args)
            assert e.value.code == tcw.TCW_EINVAL


def test_cfg2_bank_sampled_parity(tcw):
    """A 200 000-template bank on the cfg2 data (one day, 500-1000 Hz) at the injection sky point,
    as in the paper's search; the oracle recomputes a seeded sample of templates."""
    w = tcw_inputs.make_workload("cfg2")
    f0, tau, brk, sky = tcw_inputs.random_bank(200_000, 500.0, 1000.0, 2, sky=w.sky[0])
    stat, inband, _, n_exact = gpu_bank(tcw, w, f0, tau, brk, sky, want_k=False)
    sel = np.random.default_rng(1).choice(len(f0), size=1500, replace=False)
    ref = oracle.evaluate_bank(w, f0[sel], tau[sel], brk[sel], sky)
    assert_bank_parity(w, ref, stat[sel], inband[sel], None)
    assert n_exact < 1e-6 * len(f0) * w.n_sft
    assert np.isfinite(stat).all() and (inband <= w.n_sft).all()
