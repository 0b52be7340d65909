"""PSF kernel constructions (harness side; the library only receives K[ky][kx]).

SURVEY.md §8(d) D3.  Offsets u (row) and v (column) run over {-h..h} pixels.
All kernels are float64, strictly positive and normalised to sum 1.
"""
import math

import numpy as np


def _offsets(K):
    if K < 1 or K % 2 == 0:
        raise ValueError("PSF size must be odd and >= 1")
    h = K // 2
    u = np.arange(-h, h + 1, dtype=np.float64)[:, None]
    v = np.arange(-h, h + 1, dtype=np.float64)[None, :]
    return u, v


def fwhm_to_sigma(fwhm):
    return fwhm / (2.0 * math.sqrt(2.0 * math.log(2.0)))


def gaussian_psf(fwhm, pixel_scale, K=None, truncate_sigma=5.0):
    """Point-sampled circular Gaussian on a KxK square, normalised to 1.

    K=None derives the size from the truncation radius: h = ceil(t*sigma_px)
    (BASELINE.json:configs[0] "truncated at 5 sigma" -> 11x11 for C0).
    """
    sigma_px = fwhm_to_sigma(fwhm) / pixel_scale
    if K is None:
        K = 2 * int(math.ceil(truncate_sigma * sigma_px)) + 1
    u, v = _offsets(K)
    g = np.exp(-(u * u + v * v) / (2.0 * sigma_px * sigma_px))
    return g / g.sum()


def mixture3_psf(rng, K, sigma_max, n_comp=3):
    """Seeded sum of n_comp Gaussians with sub-pixel offsets (asymmetric on purpose).

    Draw order per component: w, sigma, du, dv.
    """
    u, v = _offsets(K)
    out = np.zeros((K, K), dtype=np.float64)
    for _ in range(n_comp):
        w = rng.uniform(0.2, 1.0)
        sig = rng.uniform(0.8, sigma_max)
        du = rng.uniform(-0.5, 0.5)
        dv = rng.uniform(-0.5, 0.5)
        out += w * np.exp(-((u - du) ** 2 + (v - dv) ** 2) / (2.0 * sig * sig))
    return out / out.sum()


def mixture3_psf_batch(rng, B, K, sigma_max, n_comp=3):
    """Batched Mixture3: draws w[B,3], sigma[B,3], du[B,3], dv[B,3] in that order."""
    w = rng.uniform(0.2, 1.0, size=(B, n_comp))
    sig = rng.uniform(0.8, sigma_max, size=(B, n_comp))
    du = rng.uniform(-0.5, 0.5, size=(B, n_comp))
    dv = rng.uniform(-0.5, 0.5, size=(B, n_comp))
    u, v = _offsets(K)
    out = np.zeros((B, K, K), dtype=np.float64)
    for k in range(n_comp):
        wk = w[:, k, None, None]
        sk = sig[:, k, None, None]
        out += wk * np.exp(-((u[None] - du[:, k, None, None]) ** 2 +
                             (v[None] - dv[:, k, None, None]) ** 2) / (2.0 * sk * sk))
    return out / out.sum(axis=(1, 2), keepdims=True)


def airymix_psf(rng, K=101):
    """Two Gaussians plus an r^-3 wing with ring modulation (C4), normalised to 1."""
    u, v = _offsets(K)
    out = np.zeros((K, K), dtype=np.float64)
    for _ in range(2):
        w = rng.uniform(0.5, 1.0)
        sig = rng.uniform(1.5, 3.0)
        du = rng.uniform(-0.5, 0.5)
        dv = rng.uniform(-0.5, 0.5)
        out += w * np.exp(-((u - du) ** 2 + (v - dv) ** 2) / (2.0 * sig * sig))
    w_w = rng.uniform(0.02, 0.05)
    r0 = rng.uniform(3.0, 6.0)
    p = rng.uniform(6.0, 10.0)
    a = 0.3
    r = np.sqrt(u * u + v * v)
    out += w_w * (1.0 + (r / r0) ** 2) ** (-1.5) * (1.0 + a * np.cos(2.0 * math.pi * r / p))
    return out / out.sum()
