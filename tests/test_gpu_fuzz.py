"""Randomised GPU parity: seeded random problem shapes (SFT length 4/8/10 s, holes in the timestamps,
random bands, f0 spacings of half / one / two bins, templates above and below the band, 1-300 sky
points on caps or the whole sphere, T0 before / at / inside the data) through every kernel that
accepts them (gather, staged with and without SFT chunks, the three sky-block sizes), the weighted
search and the bank search, each against the oracle with the usual bars."""
import numpy as np
import pytest

import oracle
import tcw_inputs
from tcw_inputs import Workload, detector_velocity, fibonacci_cap, fibonacci_sphere

from test_gpu_parity import KERNELS, tcw  # noqa: F401

pytestmark = pytest.mark.gpu


def _random_workload(rng):
    T = float(rng.choice([8.0, 10.0, 4.0]))
    n_slots = int(rng.integers(40, 700))
    keep = rng.random(n_slots) > rng.choice([0.0, 0.2])
    keep[0] = True
    ts = (T * np.arange(n_slots) + T / 2)[keep]
    n_bins = int(rng.integers(150, 3000))
    f_min = float(rng.integers(200, 1500))
    vel = detector_velocity(ts * rng.choice([1.0, 50.0])) if rng.random() < 0.8 else np.zeros((len(ts), 3))
    fmt = str(rng.choice(["f32", "u8", "bits"]))
    rho = rng.standard_exponential((len(ts), n_bins)).astype(np.float32)
    step = float(rng.choice([1.0, 0.5, 1.0, 2.0])) / T
    n_f0 = int(rng.integers(1, 900))
    f0 = f_min - 20 * step + step * np.arange(n_f0) + float(rng.integers(0, n_bins)) * step * rng.choice([0, 1])
    f0 = f0[f0 > 1.0]
    tau = np.sort(rng.uniform(2000, 60000, size=int(rng.integers(1, 4))))
    brk = np.sort(rng.uniform(1.5, 9.0, size=int(rng.integers(1, 4))))
    nsky = int(rng.choice([1, 3, 20, 70, 300]))
    sky = (fibonacci_sphere(nsky)[rng.permutation(nsky)] if rng.random() < 0.5
           else fibonacci_cap(nsky, 1.0, 0.3, float(rng.choice([2.0, 10.0, 60.0]))))
    T0 = float(rng.choice([ts[0] - 1.0, ts[0], ts[len(ts) // 3] + 0.5]))
    if len(f0) == 0:
        f0 = np.array([f_min + 1.0])
    return Workload("fuzz", "f32", rho, len(ts), n_bins, f_min, T, ts, vel, T0, f0, tau, brk, sky).with_format(fmt)


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_shapes_every_kernel(tcw, seed):
    import torch
    rng = np.random.default_rng(seed)
    runs = 0
    for it in range(25):
        w = _random_workload(rng)
        ref = oracle.evaluate(w)
        clean = ref.n_ambig == 0
        combos = [("auto", 0), ("gather", 0), ("staged", 0)]
        if w.fmt != "f32":
            combos += [("skyblock", 64), ("skyblock", 128)] + ([("skyblock", 256)] if w.fmt == "bits" else [])
        for kernel, sb in combos:
            with tcw.Handle.from_workload(w) as h:
                h.set_option(tcw.TCW_OPT_KERNEL, KERNELS[kernel])
                h.set_option(tcw.TCW_OPT_SKY_BLOCK, sb)
                h.set_option(tcw.TCW_OPT_CHUNK_ROWS, int(rng.choice([0, 64, -1])))
                try:
                    stat, _ = h.search(tcw.Grid.of(w))
                except tcw.TcwError as e:
                    assert e.code == tcw.TCW_EUNSUPPORTED      # f0 spacing too wide for a staged window
                    continue
                torch.cuda.synchronize()
                assert h.info()["status"] == 0
                got = stat.cpu().numpy().reshape(-1)
            runs += 1
            if w.fmt == "f32":
                assert np.all(np.abs(got[clean] - ref.stat[clean]) <= 1e-4 * np.maximum(1.0, np.abs(ref.stat[clean]))), (it, kernel)
            else:
                assert np.array_equal(got[clean].astype(np.int64), ref.stat[clean]), (it, kernel, sb)
        wt = tcw_inputs.synthetic_weights(w.sky, w.timestamps, it)
        rw = oracle.evaluate_weighted(w, wt, 1.0, 1.0)
        nb = min(200, len(w.f0))
        bf0 = rng.uniform(w.f0[0], w.f0[-1] + 1e-9, nb)
        bt, bn = rng.uniform(2000, 60000, nb), rng.uniform(1.5, 9.0, nb)
        rb = oracle.evaluate_bank(w, bf0, bt, bn, w.sky[0])
        with tcw.Handle.from_workload(w) as h:
            _, st, _ = h.search_weighted(tcw.Grid.of(w), wt, 1.0, 1.0)
            _, inb, _ = h.search_bank(bf0, bt, bn, w.sky[0], T0=w.T0)
            torch.cuda.synchronize()
            err = np.abs(st.cpu().numpy().reshape(-1) - rw.s)
            assert np.all(err[clean] <= 1e-4 * np.maximum(1.0, np.abs(rw.s[clean]))), it
            cb = rb.n_ambig == 0
            assert np.array_equal(inb.cpu().numpy()[cb], rb.n_inband[cb]), it
    assert runs > 60
