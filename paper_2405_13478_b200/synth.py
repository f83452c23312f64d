"""Seeded synthetic workloads shaped like the paper's EDA2 / MWA data.

This module is INPUT GENERATION ONLY: array layouts, frequencies, and visibilities synthesised from
a model sky with the measurement equation (Eq. 5, A = 1, w = 0, TRUE un-snapped u,v)
plus Gaussian noise.  It holds none of the method's arithmetic (no cell indices, no gridding, no
transforms) and is the one module both the oracle-side tests and the CUDA-side tests take inputs
from; the same numpy arrays are handed to both, so no RNG is shared across languages.

These inputs stand in for the paper's real recordings (EDA2 2021-11-16 / 2023-02-05 / 2023-06-01,
MWA simulations), which are not available here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

C_M_PER_S = 299792458.0
ARCSEC = math.pi / 648000.0
NATURAL, UNIFORM = 0, 1


def n_baselines(n_ant: int) -> int:
    return n_ant * (n_ant - 1) // 2


def baseline_pairs(n_ant: int):
    """(i, j) with 0 <= i < j < n_ant in boundary order bl = i(2n-i-1)/2 + (j-i-1)."""
    return np.triu_indices(n_ant, 1)


# ----------------------------------------------------------------------------- array layouts
def disc_layout(n_ant: int, diameter_m: float, seed: int, min_spacing_m: float = 0.0):
    """n_ant antennas uniform-random in a disc, optional minimum spacing by rejection."""
    rng = np.random.Generator(np.random.PCG64(seed))
    pts = []
    r_max = diameter_m / 2.0
    while len(pts) < n_ant:
        x, y = rng.uniform(-r_max, r_max, 2)
        if x * x + y * y > r_max * r_max:
            continue
        if min_spacing_m > 0 and pts:
            d = np.hypot(np.array(pts)[:, 0] - x, np.array(pts)[:, 1] - y)
            if d.min() < min_spacing_m:
                continue
        pts.append((x, y))
    enu = np.zeros((n_ant, 3), np.float64)
    enu[:, :2] = np.array(pts)
    return enu


def mwa_phase1_layout(seed: int):
    """112 tiles, exponential radial density (scale 300 m) truncated at 1.5 km, + 16 outliers
    uniform in radius 1.5-3 km; uniform azimuth (BASELINE.json config 3, read literally)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    r_core = []
    while len(r_core) < 112:
        r = rng.exponential(300.0)
        if r <= 1500.0:
            r_core.append(r)
    r = np.concatenate([np.array(r_core), rng.uniform(1500.0, 3000.0, 16)])
    az = rng.uniform(0.0, 2.0 * math.pi, 128)
    enu = np.zeros((128, 3), np.float64)
    enu[:, 0] = r * np.sin(az)
    enu[:, 1] = r * np.cos(az)
    return enu


def mwa_phase2_layout(seed: int):
    """128 tiles, radius log-uniform in [20 m, 2.5 km] (max baseline 5 km), uniform azimuth."""
    rng = np.random.Generator(np.random.PCG64(seed))
    r = np.exp(rng.uniform(math.log(20.0), math.log(2500.0), 128))
    az = rng.uniform(0.0, 2.0 * math.pi, 128)
    enu = np.zeros((128, 3), np.float64)
    enu[:, 0] = r * np.sin(az)
    enu[:, 1] = r * np.cos(az)
    return enu


def lattice_layout(nx: int, ny: int, pitch_m: float):
    """Antennas on a regular lattice (used by the oracle pins: snapping is exact)."""
    enu = np.zeros((nx * ny, 3), np.float64)
    gx, gy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="xy")
    enu[:, 0] = gx.ravel() * pitch_m
    enu[:, 1] = gy.ravel() * pitch_m
    return enu


# ----------------------------------------------------------------------------- workloads
@dataclass
class Workload:
    name: str
    ant_enu_m: np.ndarray          # [n_ant, 3] fp64
    freq_hz: np.ndarray            # [n_ch] fp64
    n_pix: int
    pixscale: float                # direction-cosine units per pixel (dx)
    weighting: int
    n_t: int
    seed: int
    src_l: np.ndarray = field(default_factory=lambda: np.zeros(0))
    src_m: np.ndarray = field(default_factory=lambda: np.zeros(0))
    src_flux: np.ndarray = field(default_factory=lambda: np.zeros(0))
    noise_sigma: float = 0.0
    diffuse_sigma: float = 0.0     # station config: CN(0, sigma_d^2 / (1+|uv|)^2), fixed in time
    pulse: dict | None = None      # sweep config: dispersed pulse description
    _sky: np.ndarray | None = None

    @property
    def n_ant(self) -> int:
        return self.ant_enu_m.shape[0]

    @property
    def n_ch(self) -> int:
        return self.freq_hz.shape[0]

    @property
    def n_bl(self) -> int:
        return n_baselines(self.n_ant)

    @property
    def n_snapshots(self) -> int:
        return self.n_t * self.n_ch

    def uv_true(self):
        """True (un-snapped) u, v in wavelengths, [n_ch, n_bl] fp64; b_ij = r_j - r_i."""
        i, j = baseline_pairs(self.n_ant)
        de = self.ant_enu_m[j, 0] - self.ant_enu_m[i, 0]
        dn = self.ant_enu_m[j, 1] - self.ant_enu_m[i, 1]
        sc = (self.freq_hz / C_M_PER_S)[:, None]
        return de[None, :] * sc, dn[None, :] * sc

    def sky_vis(self):
        """Static sky part V_sky[ch, bl] = sum_s S_s exp(-2 pi i (u l_s + v m_s)) (+ diffuse)."""
        if self._sky is None:
            u, v = self.uv_true()
            acc = np.zeros(u.shape, np.complex128)
            for l, m, s in zip(self.src_l, self.src_m, self.src_flux):
                acc += s * np.exp(-2j * math.pi * (u * l + v * m))
            if self.diffuse_sigma > 0:
                rng = np.random.Generator(np.random.PCG64([self.seed, 7777]))
                d = rng.standard_normal(u.shape) + 1j * rng.standard_normal(u.shape)
                acc += d * (self.diffuse_sigma / math.sqrt(2.0)) / (1.0 + np.hypot(u, v))
            self._sky = acc
        return self._sky

    def vis(self, t0: int = 0, t1: int | None = None) -> np.ndarray:
        """complex64 [t1-t0, n_ch, n_bl]; noise is seeded per time step so chunks reproduce."""
        t1 = self.n_t if t1 is None else t1
        sky = self.sky_vis()
        out = np.empty((t1 - t0, self.n_ch, self.n_bl), np.complex64)
        for k, t in enumerate(range(t0, t1)):
            frame = sky
            if self.pulse is not None:
                frame = sky + self._pulse_vis(t)
            if self.noise_sigma > 0:
                rng = np.random.Generator(np.random.PCG64([self.seed, 1000 + t]))
                nz = rng.standard_normal((self.n_ch, self.n_bl, 2), dtype=np.float32)
                nz *= np.float32(self.noise_sigma)
                out[k] = frame.astype(np.complex64) + nz.view(np.complex64)[..., 0]
            else:
                out[k] = frame.astype(np.complex64)
        return out

    def _pulse_vis(self, t: int):
        """Dispersed pulse: flux non-zero only at t = t0 + round(4.149 ms DM (nu^-2 - nu_ref^-2)/dt)."""
        p = self.pulse
        nu_ghz = self.freq_hz / 1e9
        delay_ms = 4.149 * p["dm"] * (nu_ghz ** -2 - p["nu_ref_ghz"] ** -2)
        t_arr = p["t0"] + np.rint(delay_ms / p["dt_ms"]).astype(np.int64)
        on = (t_arr == t)
        if not on.any():
            return 0.0
        u, v = self.uv_true()
        ph = np.exp(-2j * math.pi * (u * p["l"] + v * p["m"]))
        return ph * (p["flux"] * on[:, None])


def _random_sources(rng, n, flux_lo, flux_hi, r2_max):
    l, m = [], []
    while len(l) < n:
        a, b = rng.uniform(-1.0, 1.0, 2) * math.sqrt(r2_max)
        if a * a + b * b < r2_max:
            l.append(a)
            m.append(b)
    return np.array(l), np.array(m), rng.uniform(flux_lo, flux_hi, n)


def config_tiny(seed: int = 1) -> Workload:
    """BASELINE.json configs[0]: 32 antennas in a 35 m disc, 1 ch @160 MHz, 1 t, 128^2 all-sky."""
    rng = np.random.Generator(np.random.PCG64([seed, 1]))
    l, m, s = _random_sources(rng, 3, 1.0, 10.0, 0.8)
    return Workload("tiny", disc_layout(32, 35.0, seed), np.array([160e6]), 128, 2.0 / 128,
                    NATURAL, 1, seed, l, m, s, noise_sigma=0.1)


def config_station(seed: int = 2, n_t: int = 100, n_ch: int = 32, n_pix: int = 256) -> Workload:
    """configs[1]: SKA-Low station (EDA2-like), 256 ant in a 38 m disc, 32 fine channels of one
    0.94 MHz coarse channel around 160 MHz, natural, all-sky."""
    rng = np.random.Generator(np.random.PCG64([seed, 1]))
    l, m, s = _random_sources(rng, 50, 1.0, 10.0, 0.9)
    freq = 160e6 + np.arange(n_ch, dtype=np.float64) * (0.94e6 / 32.0)
    return Workload("station", disc_layout(256, 38.0, seed, 0.5), freq, n_pix, 2.0 / n_pix,
                    NATURAL, n_t, seed, l, m, s, noise_sigma=1.0, diffuse_sigma=50.0)


def config_mwa1(seed: int = 3, n_t: int = 100, n_ch: int = 24) -> Workload:
    """configs[2]: MWA Phase I-like, 128 tiles, 24 x 10 kHz at 154 MHz, uniform, 1024^2 at 1'."""
    rng = np.random.Generator(np.random.PCG64([seed, 1]))
    half_fov = 0.5 * 1024 * 60.0 * ARCSEC
    l, m, s = _random_sources(rng, 20, 1.0, 10.0, (0.9 * half_fov) ** 2)
    freq = 154e6 + np.arange(n_ch, dtype=np.float64) * 10e3
    return Workload("mwa1", mwa_phase1_layout(seed), freq, 1024, 60.0 * ARCSEC, UNIFORM, n_t, seed,
                    l, m, s, noise_sigma=0.5)


def config_mwa2(seed: int = 4, n_t: int = 20, n_ch: int = 24) -> Workload:
    """configs[3]: MWA Phase II extended-like, 128 tiles to 5 km, 4096^2 at 15", natural."""
    rng = np.random.Generator(np.random.PCG64([seed, 1]))
    half_fov = 0.5 * 4096 * 15.0 * ARCSEC
    l, m, s = _random_sources(rng, 100, 1.0, 10.0, (0.9 * half_fov) ** 2)
    freq = 200e6 + np.arange(n_ch, dtype=np.float64) * 10e3
    return Workload("mwa2", mwa_phase2_layout(seed), freq, 4096, 15.0 * ARCSEC, NATURAL, n_t, seed,
                    l, m, s, noise_sigma=0.5)


def config_sweep(n_pix: int, seed: int = 2, n_t: int = 1000, n_ch: int = 4) -> Workload:
    """configs[4]: station layout of config 2, 1000 t x 4 coarse channels, all-sky n_pix^2,
    noise + one dispersed pulse (quadratic nu^-2 delay across channels)."""
    freq = 160e6 + np.arange(n_ch, dtype=np.float64) * 0.94e6
    nu_ref = (freq[-1] + 0.94e6) / 1e9
    # DM chosen so the sweep spans ~200 time steps of 1 ms across the band
    span = (freq[0] / 1e9) ** -2 - nu_ref ** -2
    dm = 200.0 * 1.0 / (4.149 * span)
    pulse = dict(l=0.3, m=-0.2, flux=20.0, dm=dm, nu_ref_ghz=nu_ref, dt_ms=1.0, t0=100)
    return Workload(f"sweep{n_pix}", disc_layout(256, 38.0, seed, 0.5), freq, n_pix, 2.0 / n_pix,
                    NATURAL, n_t, seed, noise_sigma=1.0, pulse=pulse)


CONFIGS = {
    "tiny": config_tiny,
    "station": config_station,
    "mwa1": config_mwa1,
    "mwa2": config_mwa2,
}
