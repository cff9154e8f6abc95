"""The five synthetic workloads of BASELINE.json:configs, as deterministic functions of a seed.

Stand-ins: the paper measures on LALSuite-generated injections in Advanced-LIGO design noise
(section 3).  Neither LALSuite nor detector data exist here, so each workload
is seeded synthetic data with the paper's shapes: 8-s SFTs, 24 h or 72 h of
data, parameter ranges f0 500-3000 Hz, tau 3500-35000 s, n 3-7,
normalised power rho ~ Exp(1) (mean-1 power under Gaussian noise) or the thresholded number
count nu = (rho > 1.6).  The recipe is restated in DESIGN.md section 4.

Nothing here is search arithmetic shared by the oracle or the CUDA path.  The one place that
evaluates eq. (1)-(2) is `_inject_tracks`, the stand-in for lalpulsar_Makefakedata_v5: it
decides where synthetic signal power is *added to the input*; no expected value is taken
from it.
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass, field

import numpy as np

C_LIGHT = 299792458.0  # m/s
T_SFT = 8.0            # s
SEED_BASE = 250707800  # seed = SEED_BASE + config index
NU_THRESHOLD = 1.6     # BASELINE.json:configs[2]

CONFIG_NAMES = ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5")


# --------------------------------------------------------------------------- geometry
def sky_vector(ra: float, dec: float) -> np.ndarray:
    """Unit vector n-hat pointing to (right ascension, declination), equatorial frame."""
    return np.array([math.cos(dec) * math.cos(ra), math.cos(dec) * math.sin(ra), math.sin(dec)])


def detector_velocity(t: np.ndarray) -> np.ndarray:
    """Detector velocity wrt the SSB, m/s, equatorial frame, shape [len(t), 3].

    BASELINE.json:configs[0]: circular Earth orbit, 29.78 km/s, in the ecliptic (obliquity
    23.44 deg) plus rotation 0.465*cos(46.45 deg) km/s at the sidereal rate.  Phases are 0
    at t = 0.
    """
    t = np.asarray(t, dtype=np.float64)
    v_orb = 29780.0
    eps = np.deg2rad(23.44)
    w_orb = 2.0 * np.pi / (365.25636 * 86400.0)
    v_rot = 465.0 * np.cos(np.deg2rad(46.45))
    w_rot = 2.0 * np.pi / 86164.0905
    lam = w_orb * t
    th = w_rot * t
    vx = -v_orb * np.sin(lam) - v_rot * np.sin(th)
    vy = v_orb * np.cos(lam) * np.cos(eps) + v_rot * np.cos(th)
    vz = v_orb * np.cos(lam) * np.sin(eps) + 0.0 * t
    return np.ascontiguousarray(np.stack([vx, vy, vz], axis=-1))


def fibonacci_sphere(n: int) -> np.ndarray:
    """Fibonacci lattice on the full sphere: z_i = 1 - 2(i + 1/2)/n, phi_i = i*pi*(3 - sqrt 5)."""
    i = np.arange(n, dtype=np.float64)
    z = 1.0 - 2.0 * (i + 0.5) / n
    phi = i * (np.pi * (3.0 - np.sqrt(5.0)))
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    v = np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=-1)
    return _renormalise(v)


def fibonacci_cap(n: int, ra: float, dec: float, radius_deg: float) -> np.ndarray:
    """Fibonacci lattice inside a spherical cap of the given radius centred on (ra, dec).

    Cap-local axes: pole p = n-hat(ra, dec), e1 = local east (-sin ra, cos ra, 0), e2 = p x e1.
    """
    i = np.arange(n, dtype=np.float64)
    z = 1.0 - (1.0 - math.cos(math.radians(radius_deg))) * (i + 0.5) / n
    phi = i * (np.pi * (3.0 - np.sqrt(5.0)))
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    p = sky_vector(ra, dec)
    e1 = np.array([-math.sin(ra), math.cos(ra), 0.0])
    e2 = np.cross(p, e1)
    v = (r * np.cos(phi))[:, None] * e1 + (r * np.sin(phi))[:, None] * e2 + z[:, None] * p
    return _renormalise(v)


def _renormalise(v: np.ndarray) -> np.ndarray:
    v = v / np.linalg.norm(v, axis=-1, keepdims=True)
    return np.ascontiguousarray(v, dtype=np.float64)


def pack_bits(nu: np.ndarray) -> np.ndarray:
    """[n_sft][n_bins] 0/1 -> uint32 [n_sft][ceil(n_bins/32)], bit k of a row is
    (word[k >> 5] >> (k & 31)) & 1 (LSB first; include/tcw.h TCW_BIT_COUNT)."""
    nu = np.asarray(nu, dtype=np.uint8)
    n_sft, n_bins = nu.shape
    n_words = (n_bins + 31) // 32
    padded = np.zeros((n_sft, n_words * 32), dtype=np.uint8)
    padded[:, :n_bins] = nu
    by = np.packbits(padded, axis=1, bitorder="little")          # [n_sft][n_words*4] bytes
    return np.ascontiguousarray(by).view("<u4").reshape(n_sft, n_words)


def random_bank(n: int, f_lo: float, f_hi: float, seed: int, sky=None):
    """Uniform random template bank (PAPER.md:63 (ii)): f0 ~ U[f_lo, f_hi], tau ~ U[3500, 35000] s,
    n ~ U[3, 7] ("the full theoretical ranges").  sky = None draws isotropic
    unit vectors per template; otherwise the given vector is shared by all templates.
    Returns float64 arrays (f0, tau, brk, sky) with sky [n][3] or [1][3]."""
    rng = np.random.Generator(np.random.PCG64(seed + 104729))
    f0 = rng.uniform(f_lo, f_hi, size=n)
    tau = rng.uniform(3500.0, 35000.0, size=n)
    brk = rng.uniform(3.0, 7.0, size=n)
    if sky is None:
        v = rng.standard_normal((n, 3))
        sky = _renormalise(v)
    else:
        sky = np.asarray(sky, dtype=np.float64).reshape(1, 3)
    return (np.ascontiguousarray(f0), np.ascontiguousarray(tau), np.ascontiguousarray(brk),
            np.ascontiguousarray(sky, dtype=np.float64))


def synthetic_strain(n_sft: int, fs: float, T_sft: float, seed: int, lines=()):
    """Stand-in for detector strain (the paper uses coloured Gaussian noise at the aLIGO design
    sensitivity): float32 white Gaussian noise shaped by a gentle per-segment drift of
    the noise level (non-stationary floor, factor U[0.7, 1.3] per 8-s segment) plus optional
    sinusoidal lines (frequency Hz, amplitude) so that some bins stand far above the floor."""
    rng = np.random.Generator(np.random.PCG64(seed + 15485863))
    N = int(round(fs * T_sft))
    x = rng.standard_normal((n_sft, N))
    x *= rng.uniform(0.7, 1.3, size=(n_sft, 1))
    x = x.reshape(-1)
    t = np.arange(x.size, dtype=np.float64) / fs
    for f, a in lines:
        x += a * np.cos(2.0 * np.pi * f * t)
    return np.ascontiguousarray(x, dtype=np.float32)


def synthetic_weights(sky: np.ndarray, timestamps: np.ndarray, seed: int) -> np.ndarray:
    """Stand-in for the weights of the paper's ref. [14] ("antenna patterns and changing noise
    floors"): float32 [n_sky][n_sft], positive, mean 1 along each row.

    w[s][j] = F_s(t_j) / S_j with a smooth sidereal-day antenna-pattern-like modulation
    F_s(t) = 0.55 + 0.35 cos(theta(t) - alpha_s) cos(delta_s) + 0.10 sin(2 (theta(t) - alpha_s)),
    theta(t) = 2 pi t / 86164.0905 s, (alpha_s, delta_s) the sky point's right ascension and
    declination, and a seeded per-SFT noise-floor factor S_j ~ U[0.7, 1.3]^2.  Input synthesis
    only: the search treats the weights as given numbers."""
    sky = np.asarray(sky, dtype=np.float64)
    t = np.asarray(timestamps, dtype=np.float64)
    rng = np.random.Generator(np.random.PCG64(seed + 7919))
    alpha = np.arctan2(sky[:, 1], sky[:, 0])[:, None]
    cdel = np.sqrt(np.maximum(0.0, 1.0 - sky[:, 2] ** 2))[:, None]
    th = (2.0 * np.pi / 86164.0905) * t[None, :] - alpha
    F = 0.55 + 0.35 * np.cos(th) * cdel + 0.10 * np.sin(2.0 * th)
    S = rng.uniform(0.7, 1.3, size=len(t)) ** 2
    w = F / S[None, :]
    w /= w.mean(axis=1, keepdims=True)
    return np.ascontiguousarray(w, dtype=np.float32)


# --------------------------------------------------------------------------- workload
@dataclass
class Workload:
    name: str
    fmt: str                      # "f32" (normalised power) | "u8" | "bits" (number count)
    spectrogram: np.ndarray       # f32/u8 [n_sft][n_bins], or uint32 [n_sft][n_words]
    n_sft: int
    n_bins: int
    f_min: float
    T_sft: float
    timestamps: np.ndarray        # f64 [n_sft], evaluation (mid-SFT) times
    velocities: np.ndarray        # f64 [n_sft][3], m/s
    T0: float
    f0: np.ndarray                # f64 [n_f0], ascending
    tau: np.ndarray               # f64 [n_tau]
    brk: np.ndarray               # f64 [n_brk], braking index n
    sky: np.ndarray               # f64 [n_sky][3]
    injections: list = field(default_factory=list)
    seed: int = 0

    @property
    def n_groups(self) -> int:
        return len(self.sky) * len(self.tau) * len(self.brk)

    @property
    def n_templates(self) -> int:
        return self.n_groups * len(self.f0)

    @property
    def nominal_lookups(self) -> int:
        return self.n_templates * self.n_sft

    def subgrid(self, f0=None, tau=None, brk=None, sky=None) -> "Workload":
        """Same data, a sub-selection of the grid axes (index arrays or slices)."""
        def pick(a, sel):
            return a if sel is None else np.ascontiguousarray(a[sel])
        return dataclasses.replace(self, f0=pick(self.f0, f0), tau=pick(self.tau, tau),
                                   brk=pick(self.brk, brk), sky=pick(self.sky, sky))

    def with_format(self, fmt: str) -> "Workload":
        """Number-count view of a power workload: nu = (rho > 1.6) as u8 or bits; or u8 -> bits."""
        if fmt == self.fmt:
            return self
        if self.fmt == "f32":
            nu = (self.spectrogram > np.float32(NU_THRESHOLD)).astype(np.uint8)
        elif self.fmt == "u8":
            nu = self.spectrogram
        else:
            raise ValueError("cannot widen a bit-packed spectrogram")
        if fmt == "u8":
            return dataclasses.replace(self, fmt="u8", spectrogram=np.ascontiguousarray(nu))
        if fmt == "bits":
            return dataclasses.replace(self, fmt="bits", spectrogram=pack_bits(nu))
        raise ValueError(fmt)


def _timestamps(n_slots: int) -> np.ndarray:
    return 8.0 * np.arange(n_slots, dtype=np.float64) + 4.0      # t_j = 8j + 4, T0 = 0


def _exp1(rng: np.random.Generator, shape) -> np.ndarray:
    return rng.standard_exponential(size=shape, dtype=np.float32)


def _inject_tracks(rho, timestamps, velocities, f_min, T_sft, T0, injections, amp=2.0):
    """Stand-in for lalpulsar_Makefakedata_v5: add `amp` to the bin the signal
    of eq. (1)-(2) falls in at each SFT.  Input synthesis only (see module docstring)."""
    k_min = int(round(f_min * T_sft))
    n_bins = rho.shape[1]
    rows = np.arange(rho.shape[0])
    for inj in injections:
        base = (timestamps - T0) / inj["tau"] + 1.0
        f_src = inj["f0"] * np.power(base, 1.0 / (1.0 - inj["n"]))
        f_det = f_src * (1.0 + velocities @ np.asarray(inj["nhat"]) / C_LIGHT)
        k = np.rint(f_det * T_sft).astype(np.int64) - k_min
        ok = (k >= 0) & (k < n_bins) & (timestamps >= T0)
        rho[rows[ok], k[ok]] += np.float32(amp)


def _geomspace(lo: float, hi: float, n: int) -> np.ndarray:
    return np.ascontiguousarray(np.geomspace(lo, hi, n), dtype=np.float64)


def make_workload(name: str, fmt: str | None = None, seed: int | None = None) -> Workload:
    """Build one of cfg1..cfg5.  `fmt` picks the stored format where the config has several
    (cfg3: "u8" or "bits"); the default is the config's first-named format."""
    if name not in CONFIG_NAMES:
        raise ValueError(f"unknown config {name!r}; expected one of {CONFIG_NAMES}")
    idx = CONFIG_NAMES.index(name)
    if seed is None:
        # cfg3 is cfg2's data thresholded (BASELINE.json:configs[2]) -> same seed as cfg2
        seed = SEED_BASE + (1 if name == "cfg3" else idx)
    rng = np.random.Generator(np.random.PCG64(seed))
    sky1 = sky_vector(1.0, 0.3)

    if name == "cfg1":
        n_sft, n_bins, f_min = 256, 1024, 500.0
        ts = _timestamps(n_sft)
        vel = detector_velocity(ts)
        rho = _exp1(rng, (n_sft, n_bins))
        inj = [dict(f0=550.0, tau=5000.0, n=5.0, nhat=sky1)]
        _inject_tracks(rho, ts, vel, f_min, T_SFT, 0.0, inj)
        w = Workload(name, "f32", rho, n_sft, n_bins, f_min, T_SFT, ts, vel, 0.0,
                     f0=520.0 + 0.125 * np.arange(64, dtype=np.float64),
                     tau=_geomspace(3500.0, 35000.0, 4),
                     brk=np.array([3.0, 5.0, 7.0]),
                     sky=sky1[None, :].copy(), injections=inj, seed=seed)

    elif name in ("cfg2", "cfg3"):
        n_sft, n_bins, f_min = 10800, 4000, 500.0
        ts = _timestamps(n_sft)
        vel = detector_velocity(ts)
        rho = _exp1(rng, (n_sft, n_bins))
        inj = [dict(f0=float(rng.uniform(500.0, 1000.0)), tau=float(rng.uniform(3500.0, 35000.0)),
                    n=float(rng.uniform(3.0, 7.0)), nhat=sky1) for _ in range(20)]
        _inject_tracks(rho, ts, vel, f_min, T_SFT, 0.0, inj)
        f0 = 500.0 + 0.125 * np.arange(4000, dtype=np.float64)
        if name == "cfg2":
            w = Workload(name, "f32", rho, n_sft, n_bins, f_min, T_SFT, ts, vel, 0.0, f0=f0,
                         tau=_geomspace(3500.0, 35000.0, 32),
                         brk=np.array([3.0, 4.0, 5.0, 6.0, 7.0]),
                         sky=sky1[None, :].copy(), injections=inj, seed=seed)
        else:
            w = Workload(name, "f32", rho, n_sft, n_bins, f_min, T_SFT, ts, vel, 0.0, f0=f0,
                         tau=_geomspace(3500.0, 35000.0, 16),
                         brk=np.array([3.0, 4.0, 5.0, 6.0, 7.0]),
                         sky=fibonacci_cap(256, 3.45, -0.41, 10.0), injections=inj, seed=seed)
            w = w.with_format(fmt or "u8")

    elif name == "cfg4":
        n_slots, n_bins, f_min = 32400, 20000, 500.0
        present = np.ones(n_slots, dtype=bool)
        while (~present).mean() < 0.30:                           # random 1-6 h gaps
            length = int(rng.uniform(1.0, 6.0) * 450.0)           # 450 slots per hour
            start = int(rng.integers(0, n_slots - length))
            present[start:start + length] = False
        ts = _timestamps(n_slots)[present]
        n_sft = len(ts)
        vel = detector_velocity(ts)
        rho = _exp1(rng, (n_sft, n_bins))
        w = Workload(name, "f32", rho, n_sft, n_bins, f_min, T_SFT, ts, vel, 0.0,
                     f0=500.0 + 0.125 * np.arange(20000, dtype=np.float64),
                     tau=_geomspace(3500.0, 35000.0, 64),
                     brk=3.0 + 0.5 * np.arange(9, dtype=np.float64),
                     sky=sky1[None, :].copy(), seed=seed)

    else:  # cfg5
        n_sft, n_bins, f_min = 10800, 4000, 1000.0
        ts = _timestamps(n_sft)
        vel = detector_velocity(ts)
        rho = _exp1(rng, (n_sft, n_bins))
        floor = rng.uniform(0.7, 1.3, size=n_sft).astype(np.float32)   # non-stationary noise floor
        nu = (rho * floor[:, None] > np.float32(NU_THRESHOLD)).astype(np.uint8)
        del rho
        w = Workload(name, "u8", nu, n_sft, n_bins, f_min, T_SFT, ts, vel, 0.0,
                     f0=1000.0 + 0.125 * np.arange(4000, dtype=np.float64),
                     tau=_geomspace(3500.0, 35000.0, 8),
                     brk=np.array([3.0, 5.0, 7.0]),
                     sky=fibonacci_sphere(4096), seed=seed)
        w = w.with_format(fmt or "bits")

    if fmt is not None and w.fmt != fmt:
        w = w.with_format(fmt)
    return w
