"""Seeded configs C0..C4 (BASELINE.json:configs[0..4]) and the paper's conv sweep shapes.

Draw recipe: SURVEY.md §8(d) D1 (numpy PCG64, float64 draws, fixed order),
D2 (values BASELINE.json leaves open), D4 (concrete inputs).  Every generator
takes optional size overrides so the same recipe yields the small parity cases
the CPU oracle finishes in seconds.  No lensing arithmetic lives here.
"""
from dataclasses import dataclass, field, replace
import math

import numpy as np

from .psf import gaussian_psf, mixture3_psf, mixture3_psf_batch, airymix_psf

SEEDS = {"C1": 154701, "C2": 154702, "C3": 154703, "C4": 154704, "sweep": 154710}

# C0's fixed macro-lens and source (BASELINE.json:configs[0]); C2 and C4 reuse them (D2).
C0_SIE = (1.0, 0.1, -0.05, 0.0, 0.0)        # theta_E, e1, e2, cx, cy
C0_SHEAR = (0.03, 0.01)                     # gamma1, gamma2
C0_SOURCE = (10.0, 0.2, 1.5, 0.05, 0.02, 0.05, 0.0)  # amp, R_sersic, n_sersic, e1, e2, cx, cy


def _f32_round(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)


@dataclass
class Workload:
    """One lens system.  All parameter arrays are float64 (possibly f32-rounded values)."""
    name: str
    dtype: str                       # "f64" or "f32": arithmetic type of the call
    nx: int
    ny: int
    pixel_scale: float
    supersample: int
    sie: tuple                       # (theta_E, e1, e2, cx, cy) or None
    shear: tuple                     # (gamma1, gamma2) or None
    tnfw: np.ndarray                 # [5][M] rows cx, cy, Rs, alpha_Rs, r_trunc
    sources: np.ndarray              # [n_src][7] amp, R_sersic, n_sersic, e1, e2, cx, cy
    psf: np.ndarray                  # [ky][kx], odd sizes
    cx: float = 0.0
    cy: float = 0.0
    notes: dict = field(default_factory=dict)

    @property
    def n_rays(self):
        return self.nx * self.supersample * self.ny * self.supersample

    @property
    def n_tnfw(self):
        return int(self.tnfw.shape[1])

    @property
    def n_deflectors(self):
        return self.n_tnfw + (1 if self.sie is not None else 0) + (1 if self.shear is not None else 0)

    @property
    def evals(self):
        """ray x deflector evaluations."""
        return self.n_rays * self.n_deflectors

    def as_dtype(self, dtype):
        """Q19: for f32 the draws are rounded ONCE to float32; both sides consume those values."""
        if dtype == "f64":
            return replace(self, dtype="f64")
        if dtype != "f32":
            raise ValueError(dtype)
        return replace(
            self, dtype="f32",
            sie=None if self.sie is None else tuple(_f32_round(self.sie).tolist()),
            shear=None if self.shear is None else tuple(_f32_round(self.shear).tolist()),
            tnfw=_f32_round(self.tnfw), sources=_f32_round(self.sources), psf=_f32_round(self.psf))


@dataclass
class BatchWorkload:
    """B independent lens systems sharing one grid (BASELINE.json:configs[3])."""
    name: str
    dtype: str
    B: int
    nx: int
    ny: int
    pixel_scale: float
    supersample: int
    sie: np.ndarray                  # [B][5]
    shear: np.ndarray                # [B][2]
    tnfw: np.ndarray                 # [B][5][M]
    sources: np.ndarray              # [B][n_src][7]
    psf: np.ndarray                  # [B][ky][kx]
    cx: float = 0.0
    cy: float = 0.0

    @property
    def n_rays(self):
        return self.nx * self.supersample * self.ny * self.supersample

    @property
    def n_tnfw(self):
        return int(self.tnfw.shape[2])

    @property
    def evals(self):
        return self.B * self.n_rays * (self.n_tnfw + 2)

    def as_dtype(self, dtype):
        if dtype == "f64":
            return replace(self, dtype="f64")
        return replace(self, dtype="f32", sie=_f32_round(self.sie), shear=_f32_round(self.shear),
                       tnfw=_f32_round(self.tnfw), sources=_f32_round(self.sources),
                       psf=_f32_round(self.psf))

    def system(self, b):
        """System b as a single-image Workload (for per-system oracle calls)."""
        return Workload(
            name=f"{self.name}[{b}]", dtype=self.dtype, nx=self.nx, ny=self.ny,
            pixel_scale=self.pixel_scale, supersample=self.supersample,
            sie=tuple(self.sie[b].tolist()), shear=tuple(self.shear[b].tolist()),
            tnfw=np.ascontiguousarray(self.tnfw[b]), sources=np.ascontiguousarray(self.sources[b]),
            psf=np.ascontiguousarray(self.psf[b]), cx=self.cx, cy=self.cy)


def _log_uniform(rng, lo, hi, size):
    return np.exp(rng.uniform(math.log(lo), math.log(hi), size=size))


def _draw_sources(rng, n):
    """Per source: amp, R_sersic, n_sersic, e1, e2, cx, cy (C1 priors + D2)."""
    out = np.zeros((n, 7), dtype=np.float64)
    for k in range(n):
        out[k, 0] = rng.uniform(5.0, 20.0)
        out[k, 1] = rng.uniform(0.1, 0.5)
        out[k, 2] = rng.uniform(0.5, 4.0)
        out[k, 3] = rng.uniform(-0.2, 0.2)
        out[k, 4] = rng.uniform(-0.2, 0.2)
        out[k, 5] = rng.uniform(-0.2, 0.2)
        out[k, 6] = rng.uniform(-0.2, 0.2)
    return out


def _draw_subhalos(rng, M, half_width):
    """cx[M], cy[M], Rs[M], alpha_Rs[M]; r_trunc = 5 Rs (C2 priors)."""
    t = np.zeros((5, M), dtype=np.float64)
    t[0] = rng.uniform(-half_width, half_width, size=M)
    t[1] = rng.uniform(-half_width, half_width, size=M)
    t[2] = _log_uniform(rng, 0.005, 0.05, M)
    t[3] = _log_uniform(rng, 1e-4, 1e-2, M)
    t[4] = 5.0 * t[2]
    return t


def config_c0(nx=60, dtype="f64", seed_offset=0):
    """C0: single lens image, 60x60, no supersampling, SIE + shear, one Sersic, 11x11 Gaussian PSF."""
    w = Workload(
        name="C0", dtype="f64", nx=nx, ny=nx, pixel_scale=0.05, supersample=1,
        sie=C0_SIE, shear=C0_SHEAR, tnfw=np.zeros((5, 0)), sources=np.array([C0_SOURCE]),
        psf=gaussian_psf(0.1, 0.05, K=None, truncate_sigma=5.0))
    return w.as_dtype(dtype)


def config_c1(nx=100, supersample=3, K=31, dtype="f64", seed_offset=0):
    """C1: 100x100, supersampling 3, SIE + shear + one TNFW, two Sersics, Mixture3(31) PSF."""
    rng = np.random.default_rng(SEEDS["C1"] + seed_offset)
    theta_E = rng.uniform(0.8, 1.5)
    e1 = rng.uniform(-0.2, 0.2)
    e2 = rng.uniform(-0.2, 0.2)
    g1 = rng.uniform(-0.05, 0.05)
    g2 = rng.uniform(-0.05, 0.05)
    sources = _draw_sources(rng, 2)
    psf = mixture3_psf(rng, K, sigma_max=4.0 if K >= 31 else 3.0)
    tnfw = np.array([[0.8], [0.3], [0.2], [0.1], [1.0]])
    w = Workload(
        name="C1", dtype="f64", nx=nx, ny=nx, pixel_scale=0.05, supersample=supersample,
        sie=(theta_E, e1, e2, 0.0, 0.0), shear=(g1, g2), tnfw=tnfw, sources=sources, psf=psf)
    return w.as_dtype(dtype)


def config_c2(nx=200, supersample=2, n_tnfw=10000, K=21, dtype="f64", seed_offset=0):
    """C2: 200x200 @0.04, supersampling 2, C0 macro-lens + 10,000 TNFW in a 4x4 square."""
    rng = np.random.default_rng(SEEDS["C2"] + seed_offset)
    tnfw = _draw_subhalos(rng, n_tnfw, 2.0)
    w = Workload(
        name="C2", dtype="f64", nx=nx, ny=nx, pixel_scale=0.04, supersample=supersample,
        sie=C0_SIE, shear=C0_SHEAR, tnfw=tnfw, sources=np.array([C0_SOURCE]),
        psf=gaussian_psf(0.1, 0.04, K=K))
    return w.as_dtype(dtype)


def config_c3(B=4096, nx=64, supersample=2, n_tnfw=100, K=21, dtype="f32", seed_offset=0):
    """C3: B independent systems, 64x64 @0.08, supersampling 2, 100 TNFW each, own Mixture3(21) PSF."""
    rng = np.random.default_rng(SEEDS["C3"] + seed_offset)
    sie = np.zeros((B, 5), dtype=np.float64)
    sie[:, 0] = rng.uniform(0.8, 1.5, size=B)
    sie[:, 1] = rng.uniform(-0.2, 0.2, size=B)
    sie[:, 2] = rng.uniform(-0.2, 0.2, size=B)
    shear = np.zeros((B, 2), dtype=np.float64)
    shear[:, 0] = rng.uniform(-0.05, 0.05, size=B)
    shear[:, 1] = rng.uniform(-0.05, 0.05, size=B)
    tnfw = np.zeros((B, 5, n_tnfw), dtype=np.float64)
    tnfw[:, 0] = rng.uniform(-2.0, 2.0, size=(B, n_tnfw))
    tnfw[:, 1] = rng.uniform(-2.0, 2.0, size=(B, n_tnfw))
    tnfw[:, 2] = _log_uniform(rng, 0.005, 0.05, (B, n_tnfw))
    tnfw[:, 3] = _log_uniform(rng, 1e-4, 1e-2, (B, n_tnfw))
    tnfw[:, 4] = 5.0 * tnfw[:, 2]
    src = np.zeros((B, 1, 7), dtype=np.float64)
    src[:, 0, 0] = rng.uniform(5.0, 20.0, size=B)
    src[:, 0, 1] = rng.uniform(0.1, 0.5, size=B)
    src[:, 0, 2] = rng.uniform(0.5, 4.0, size=B)
    src[:, 0, 3] = rng.uniform(-0.2, 0.2, size=B)
    src[:, 0, 4] = rng.uniform(-0.2, 0.2, size=B)
    src[:, 0, 5] = rng.uniform(-0.2, 0.2, size=B)
    src[:, 0, 6] = rng.uniform(-0.2, 0.2, size=B)
    psf = mixture3_psf_batch(rng, B, K, sigma_max=3.0)
    w = BatchWorkload(
        name="C3", dtype="f64", B=B, nx=nx, ny=nx, pixel_scale=0.08, supersample=supersample,
        sie=sie, shear=shear, tnfw=tnfw, sources=src, psf=psf)
    return w.as_dtype(dtype)


@dataclass
class SwarmWorkload(BatchWorkload):
    """A particle swarm's inner loop: B parameter vectors, one data image and noise map."""
    data: np.ndarray = None          # [ny][nx]
    sigma: np.ndarray = None         # [ny][nx]

    def as_dtype(self, dtype):
        w = super().as_dtype(dtype)
        if dtype == "f32":
            w = replace(w, data=_f32_round(self.data), sigma=_f32_round(self.sigma))
        return w


def config_swarm(B=256, nx=100, K=13, supersample=1, dtype="f64", seed_offset=0):
    """NEXT-3: the shape of the paper's particle-swarm benchmark, PAPER.md:122 -- a 100x100 grid
    (0.05 arcsec pixels as in C1), a 13-pixel PSF (Gaussian FWHM 0.1 arcsec, the same for every particle), SIE + shear
    mass model and one elliptical Sersic source per particle, no subhalos.  The particles are a seeded truth (C1 priors)
    perturbed by 5 % Gaussian scatter; the data image is the pre-computed noise-free truth plus noise of rms sigma.
    The paper's lens light and point source are outside the hot path.
    `data` is filled by the caller (tests and bench.py form it with the oracle or with jt_simulate_batch on the truth,
    which this module -- free of lensing arithmetic -- cannot do); `sigma` is a constant background rms."""
    rng = np.random.default_rng(SEEDS["sweep"] + 77 + seed_offset)
    truth_sie = np.array([rng.uniform(0.8, 1.5), rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), 0.0, 0.0])
    truth_shear = rng.uniform(-0.05, 0.05, size=2)
    truth_src = np.array([rng.uniform(5.0, 20.0), rng.uniform(0.1, 0.5), rng.uniform(0.5, 4.0), rng.uniform(-0.2, 0.2),
                          rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2)])
    jitter = lambda v, n: v[None, :] * (1.0 + 0.05 * rng.standard_normal((n, v.size))) + 0.01 * rng.standard_normal((n, v.size))
    sie = jitter(truth_sie, B)
    sie[0] = truth_sie                                   # particle 0 is the truth itself
    shear = jitter(truth_shear, B)
    shear[0] = truth_shear
    src = jitter(truth_src, B)
    src[0] = truth_src
    src[:, 2] = np.clip(src[:, 2], 0.5, 4.0)
    psf = np.broadcast_to(gaussian_psf(0.1, 0.05, K=K), (B, K, K)).copy()
    sigma = np.full((nx, nx), 0.02)
    noise = sigma * rng.standard_normal((nx, nx))
    w = SwarmWorkload(name="swarm", dtype="f64", B=B, nx=nx, ny=nx, pixel_scale=0.05, supersample=supersample,
                      sie=sie, shear=shear, tnfw=np.zeros((B, 5, 0)), sources=src[:, None, :], psf=psf,
                      data=noise, sigma=sigma)           # data = truth image + this noise: the caller adds the truth
    return w.as_dtype(dtype)


def config_c4(nx=500, supersample=5, n_tnfw=50000, K=101, half_width=5.0, dtype="f64", seed_offset=0):
    """C4: 500x500 @0.02, supersampling 5, C0 macro-lens + 50,000 TNFW over 10x10, 3 Sersics, AiryMix(101)."""
    rng = np.random.default_rng(SEEDS["C4"] + seed_offset)
    tnfw = _draw_subhalos(rng, n_tnfw, half_width)
    sources = _draw_sources(rng, 3)
    psf = airymix_psf(rng, K)
    w = Workload(
        name="C4", dtype="f64", nx=nx, ny=nx, pixel_scale=0.02, supersample=supersample,
        sie=C0_SIE, shear=C0_SHEAR, tnfw=tnfw, sources=sources, psf=psf)
    return w.as_dtype(dtype)


def conv_sweep_case(N, K, dtype="f64"):
    """Convolution-only case at the paper's shapes: U[0,1] image, Gaussian sigma=K/8 px."""
    rng = np.random.default_rng(SEEDS["sweep"] + 1000 * N + K)
    img = rng.uniform(0.0, 1.0, size=(N, N))
    h = K // 2
    u = np.arange(-h, h + 1, dtype=np.float64)[:, None]
    v = np.arange(-h, h + 1, dtype=np.float64)[None, :]
    sig = K / 8.0
    ker = np.exp(-(u * u + v * v) / (2.0 * sig * sig))
    ker /= ker.sum()
    if dtype == "f32":
        img, ker = _f32_round(img), _f32_round(ker)
    return img, ker
