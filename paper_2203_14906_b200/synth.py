"""Seeded synthetic RF generator (input data only; none of the method's arithmetic).

Stands in for the paper's k-Wave simulations and ex-vivo acquisition
(Sec. III, Sec. IV), which are
not available here.  It produces linear-array photoacoustic channel data with
the shapes and sizes of BASELINE.json configs C1..C5 (+ the headline C2b) from
an analytic pulse model, as SURVEY.md §8(d) states it:

  element i, absorber a at distance r_ia:   A_a * g(t - r_ia / c)
  point absorber:  g(tau) = -(tau/sigma) * exp(0.5 - tau^2 / (2 sigma^2)),  sigma = 1/(2 pi f0)
                   (derivative of a Gaussian, bipolar "N-shaped", peak |g| = 1)
  disc absorber of radius R: ideal N-wave -tau/T on |tau| <= T = R/c convolved with a unit-area
                   Gaussian of width sigma (closed form), normalised to peak 1
  no geometric spreading; sample n is at t = n / fs; additive noise per frame with
  sigma_noise = max|clean| * 10^(-SNR/20)  (peak-based reading, A16).

Both the fp64 oracle (oracle/) and the CUDA library are fed the arrays made
here, so no RNG has to match across languages.  This module imports neither.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

try:  # closed-form disc pulse needs erf; scipy is in the image, math.erf is the fallback
    from scipy.special import erf as _erf
except Exception:  # pragma: no cover
    _erf = np.vectorize(math.erf)


@dataclass
class Geometry:
    """Array + grid parameters exactly as they cross the C ABI (all float32-representable)."""
    n_elem: int
    n_samp: int
    fs: float          # Hz
    c: float           # m/s
    pitch: float       # m
    nx: int
    nz: int
    x0: float          # m, centre of pixel column 0
    dx: float
    z0: float          # m, centre of pixel row 0
    dz: float

    def f32(self) -> "Geometry":
        """Round every float parameter to float32 (what the ABI carries); oracle gets the same values."""
        r = lambda v: float(np.float32(v))
        return Geometry(self.n_elem, self.n_samp, r(self.fs), r(self.c), r(self.pitch),
                        self.nx, self.nz, r(self.x0), r(self.dx), r(self.z0), r(self.dz))

    def elem_x(self) -> np.ndarray:
        return (np.arange(self.n_elem) - (self.n_elem - 1) / 2.0) * self.pitch

    def pix_x(self) -> np.ndarray:
        return self.x0 + np.arange(self.nx) * self.dx

    def pix_z(self) -> np.ndarray:
        return self.z0 + np.arange(self.nz) * self.dz


@dataclass
class Workload:
    name: str
    geom: Geometry
    rf: np.ndarray                  # [F][N][S], float32 or int16
    orders: tuple
    f0: float                       # pulse centre frequency, Hz
    post: dict | None = None        # band-pass / envelope / log parameters, if the config asks for them
    truth: list = field(default_factory=list)   # per frame: list of (x, z, amplitude, radius)
    seed: int = 0


# ----------------------------------------------------------------------------------------------
# pulse shapes
# ----------------------------------------------------------------------------------------------
def pulse_point(tau: np.ndarray, f0: float) -> np.ndarray:
    """Derivative-of-Gaussian pulse, peak magnitude 1 at tau = -/+ sigma."""
    sigma = 1.0 / (2.0 * math.pi * f0)
    u = tau / sigma
    return -u * np.exp(0.5 - 0.5 * u * u)


def _disc_raw(tau: np.ndarray, T: float, sigma: float) -> np.ndarray:
    Phi = lambda v: 0.5 * (1.0 + _erf(v / math.sqrt(2.0)))
    phi = lambda v: np.exp(-0.5 * (v / sigma) ** 2) / (sigma * math.sqrt(2.0 * math.pi))
    a = tau + T
    b = tau - T
    return -(1.0 / T) * (tau * (Phi(a / sigma) - Phi(b / sigma)) + sigma * sigma * (phi(a) - phi(b)))


def pulse_disc(tau: np.ndarray, f0: float, radius: float, c: float) -> np.ndarray:
    """N-wave of a disc of given radius, Gaussian-smoothed, normalised to peak 1."""
    sigma = 1.0 / (2.0 * math.pi * f0)
    T = radius / c
    fine = np.linspace(-T - 5 * sigma, T + 5 * sigma, 4001)
    peak = np.max(np.abs(_disc_raw(fine, T, sigma)))
    return _disc_raw(tau, T, sigma) / peak


# ----------------------------------------------------------------------------------------------
# frame synthesis
# ----------------------------------------------------------------------------------------------
def pulse_gauss(tau: np.ndarray, f0: float) -> np.ndarray:
    """Unipolar Gaussian pulse, peak 1 at tau = 0 (used by the point-target pin only)."""
    sigma = 1.0 / (2.0 * math.pi * f0)
    return np.exp(-0.5 * (tau / sigma) ** 2)


def _add_absorbers(rf: np.ndarray, geom: Geometry, absorbers, f0: float, shape: str = "n") -> None:
    """rf [N][S] float64 += pulses of every (x, z, A, R) in absorbers, evaluated in a local window."""
    N, S = rf.shape
    xe = geom.elem_x()
    sigma = 1.0 / (2.0 * math.pi * f0)
    n_all = np.arange(S)
    for (xa, za, amp, rad) in absorbers:
        r = np.sqrt((xe - xa) ** 2 + za * za)            # [N]
        t_arr = r / geom.c
        half = (6.0 * sigma + (rad / geom.c if rad > 0 else 0.0)) * geom.fs
        half_n = int(math.ceil(half)) + 2
        centre = np.rint(t_arr * geom.fs).astype(np.int64)   # [N]
        offs = np.arange(-half_n, half_n + 1)
        idx = centre[:, None] + offs[None, :]              # [N][w]
        ok = (idx >= 0) & (idx < S)
        tau = idx / geom.fs - t_arr[:, None]
        if shape == "gauss":
            val = pulse_gauss(tau, f0)
        elif rad > 0:
            val = pulse_disc(tau, f0, rad, geom.c)
        else:
            val = pulse_point(tau, f0)
        rows = np.broadcast_to(np.arange(N)[:, None], idx.shape)
        np.add.at(rf, (rows[ok], idx[ok]), amp * val[ok])
    del n_all


def _white_noise(rng, shape, clean_peak: float, snr_db: float) -> np.ndarray:
    return rng.standard_normal(shape) * (clean_peak * 10.0 ** (-snr_db / 20.0))


def _draw_absorbers(rng, n, x_rng, z_rng, amp=("const", 1.0), n_disc=0, r_rng=(0.1e-3, 0.5e-3)):
    out = []
    for a in range(n):
        x = rng.uniform(*x_rng)
        z = rng.uniform(*z_rng)
        if amp[0] == "const":
            A = amp[1]
        elif amp[0] == "uniform":
            A = rng.uniform(amp[1], amp[2])
        elif amp[0] == "log40":
            A = 10.0 ** (-rng.uniform(0.0, 2.0))
        elif amp[0] == "counts":
            A = rng.uniform(amp[1], amp[2]) * rng.choice([-1.0, 1.0])
        else:
            raise ValueError(amp)
        R = rng.uniform(*r_rng) if a >= n - n_disc else 0.0
        out.append((x, z, A, R))
    return out


def _jitter(rng, absorbers, sd=0.1e-3):
    return [(x + rng.normal(0, sd), z + rng.normal(0, sd), A, R) for (x, z, A, R) in absorbers]


def _frames(rng, geom, base, f0, n_frames, snr_db, jitter, dtype=np.float32, noise_counts=None):
    N, S = geom.n_elem, geom.n_samp
    rf = np.empty((n_frames, N, S), dtype=dtype)
    truth = []
    for f in range(n_frames):
        ab = _jitter(rng, base) if jitter else list(base)
        fr = np.zeros((N, S))
        _add_absorbers(fr, geom, ab, f0)
        if noise_counts is not None:
            fr += rng.standard_normal(fr.shape) * noise_counts
            fr = np.clip(np.rint(fr), -32767, 32767)
        elif snr_db is not None:
            fr += _white_noise(rng, fr.shape, np.max(np.abs(fr)), snr_db)
        rf[f] = fr.astype(dtype)
        truth.append(ab)
    return rf, truth


# ----------------------------------------------------------------------------------------------
# the configs of BASELINE.json (SURVEY.md §8(d) recipes)
# ----------------------------------------------------------------------------------------------
_MM = 1e-3


def geometry(cfg: str) -> Geometry:
    """Geometry of a named config; float32-rounded (the ABI's view)."""
    c = 1540.0
    if cfg == "C1":
        g = Geometry(16, 1024, 40e6, c, 0.3 * _MM, 16, 128, -2.25 * _MM, 0.3 * _MM, 0.0, 30 * _MM / 128)
    elif cfg in ("C2", "C2b"):
        dx = 0.15 * _MM
        g = Geometry(128, 2048, 40e6, c, 0.3 * _MM, 256, 1024, -127.5 * dx, dx, 5 * _MM, 45 * _MM / 1024)
    elif cfg == "C3":
        dx = 0.3 * _MM
        g = Geometry(128, 2048, 40e6, c, 0.3 * _MM, 128, 512, -63.5 * dx, dx, 10 * _MM, c / 40e6)
    elif cfg == "C4":
        dx = 0.1 * _MM
        g = Geometry(256, 4096, 62.5e6, c, 0.2 * _MM, 512, 2048, -255.5 * dx, dx, 5 * _MM, 75 * _MM / 2048)
    elif cfg == "C5":
        dx = 0.3 * _MM
        g = Geometry(192, 3072, 40e6, c, 0.3 * _MM, 192, 768, -95.5 * dx, dx, 10 * _MM, c / 40e6)
    else:
        raise ValueError(f"unknown config {cfg}")
    return g.f32()


_SEEDS = {"C1": 1001, "C2": 1002, "C2b": 1012, "C3": 1003, "C4": 1004, "C5": 1005}
_POST_LOG = dict(mode="log", f_center=10e6, f_halfwidth=2.5e6, n_taps_bp=64, n_taps_hilbert=63, dyn_range_db=60.0)


def make_config(cfg: str, seed: int | None = None, n_frames: int | None = None) -> Workload:
    """Build the seeded synthetic workload for config `cfg` (C1, C2, C2b, C3, C4, C5).

    n_frames overrides the frame count (tests use a few frames of the streaming configs).
    """
    seed = _SEEDS[cfg] if seed is None else seed
    rng = np.random.default_rng(seed)
    g = geometry(cfg)
    f0 = 5e6
    if cfg == "C1":
        base = _draw_absorbers(rng, 3, (-2 * _MM, 2 * _MM), (8 * _MM, 26 * _MM))
        rf, truth = _frames(rng, g, base, f0, n_frames or 1, 20.0, False)
        return Workload(cfg, g, rf, (1, 2, 3, 4, 5), f0, None, truth, seed)
    if cfg in ("C2", "C2b"):
        base = _draw_absorbers(rng, 10, (-17 * _MM, 17 * _MM), (8 * _MM, 47 * _MM), ("uniform", 0.5, 1.0), n_disc=4)
        F = n_frames or (1 if cfg == "C2" else 64)
        rf, truth = _frames(rng, g, base, f0, F, 10.0, cfg == "C2b")
        return Workload(cfg, g, rf, (1, 2, 3) if cfg == "C2" else (3,), f0, None, truth, seed)
    if cfg == "C3":
        base = _draw_absorbers(rng, 10, (-17 * _MM, 17 * _MM), (12 * _MM, 28 * _MM), ("uniform", 0.5, 1.0))
        rf, truth = _frames(rng, g, base, f0, n_frames or 256, 10.0, True)
        return Workload(cfg, g, rf, (3,), f0, dict(_POST_LOG), truth, seed)
    if cfg == "C4":
        base = _draw_absorbers(rng, 50, (-24 * _MM, 24 * _MM), (8 * _MM, 76 * _MM), ("log40",))
        F = n_frames or 1
        rf, truth = _frames(rng, g, base, f0, F, None, False, dtype=np.float64)
        # correlated clutter: white noise convolved in time with the pulse and across channels with [1/4,1/2,1/4],
        # scaled to 20 dB below the strongest pulse (level is a DESIGN.md choice; the config gives none)
        sigma = 1.0 / (2.0 * math.pi * f0)
        k_t = pulse_point(np.arange(-24, 25) / g.fs, f0)
        for f in range(F):
            w = rng.standard_normal((g.n_elem, g.n_samp))
            w = np.apply_along_axis(lambda r: np.convolve(r, k_t, mode="same"), 1, w)
            w = 0.25 * np.roll(w, 1, 0) + 0.5 * w + 0.25 * np.roll(w, -1, 0)
            w *= 0.1 * np.max(np.abs(rf[f])) / np.max(np.abs(w))
            rf[f] += w
        del sigma
        return Workload(cfg, g, rf.astype(np.float32), (4, 5), f0, None, truth, seed)
    if cfg == "C5":
        base = _draw_absorbers(rng, 10, (-25 * _MM, 25 * _MM), (12 * _MM, 38 * _MM), ("counts", 200.0, 2000.0))
        rf, truth = _frames(rng, g, base, f0, n_frames or 1024, None, True, dtype=np.int16, noise_counts=8.0)
        return Workload(cfg, g, rf, (3,), f0, dict(_POST_LOG), truth, seed)
    raise ValueError(cfg)


def simulation1_phantom(seed: int = 1101, n_frames: int = 1) -> Workload:
    """A phantom laid out like the paper's Simulation 1: 128 elements, pitch 0.1 mm, 7.5 MHz,
    fs 100 MHz, c 1500 m/s, ten point targets as five pairs 3 mm apart at depths 17, 20, 23, 26, 29 mm, white noise
    at 30 dB (A16).  Stands in for the k-Wave data, which is not available; pulses are this module's analytic model."""
    rng = np.random.default_rng(seed)
    nx, nz = 128, 512
    g = Geometry(128, 2560, 100e6, 1500.0, 0.1 * _MM, nx, nz, -5.0 * _MM, 10.0 * _MM / nx, 15.0 * _MM,
                 16.0 * _MM / nz).f32()
    base = [(sx * 1.5 * _MM, z * _MM, 1.0, 0.0) for z in (17, 20, 23, 26, 29) for sx in (-1.0, 1.0)]
    rf, truth = _frames(rng, g, base, 7.5e6, n_frames, 30.0, False)
    post = dict(mode="envelope", f_center=7.5e6, f_halfwidth=4.0e6, n_taps_bp=64, n_taps_hilbert=63, dyn_range_db=60.0)
    return Workload("SIM1", g, rf, (1, 2, 3, 4, 5), 7.5e6, post, truth, seed)


def point_target_frame(g: Geometry, ix: int, iz: int, f0: float = 5e6, shape: str = "n") -> np.ndarray:
    """Noiseless single point absorber on the centre of pixel (iz, ix); [1][N][S] float32 (pin P8).

    shape "n": the bipolar N-shaped pulse of the workloads (zero crossing AT the absorber);
    shape "gauss": a unipolar Gaussian, whose beamformed peak sits on the absorber's pixel."""
    fr = np.zeros((g.n_elem, g.n_samp))
    _add_absorbers(fr, g, [(g.x0 + ix * g.dx, g.z0 + iz * g.dz, 1.0, 0.0)], f0, shape)
    return fr.astype(np.float32)[None]


def random_geometry(rng, n_elem, n_samp, nx, nz, in_range=True) -> Geometry:
    """A random small geometry for property tests (ragged tiles, odd sizes)."""
    fs, c = 40e6, 1540.0
    pitch = rng.uniform(0.2, 0.4) * _MM
    dx = rng.uniform(0.1, 0.4) * _MM
    rec = (n_samp - 3) * c / fs
    half = max((n_elem - 1) * pitch / 2, (nx - 1) * dx / 2)
    zmax = math.sqrt(max(rec * rec - (2 * half) ** 2, (0.3 * rec) ** 2)) if in_range else 1.3 * rec
    z0 = rng.uniform(0.0, 0.2) * zmax
    dz = (zmax * rng.uniform(0.7, 0.98) - z0) / max(nz - 1, 1)
    return Geometry(n_elem, n_samp, fs, c, pitch, nx, nz, -(nx - 1) * dx / 2 + rng.uniform(-1, 1) * dx, dx, z0, dz).f32()
