"""Pins for the oracle's grid, Sersic, binning, convolution and composition
(definitions G, R, B, P; SURVEY.md §8(c) pins table)."""
import math

import numpy as np
import pytest
from scipy import integrate, signal, special

import workloads
from conftest import rel_err


# ---------------------------------------------------------------- G
def test_grid_geometry(orc):
    nx, ny, ps, s = 6, 4, 0.05, 3
    tx, ty = orc.grid(nx, ny, ps, 0.1, -0.2, s)
    tx = tx.reshape(ny * s, nx * s)
    ty = ty.reshape(ny * s, nx * s)
    h = ps / s
    assert np.allclose(np.diff(tx, axis=1), h, atol=1e-15) and np.allclose(np.diff(ty, axis=0), h, atol=1e-15)
    assert np.all(tx[0] == tx[-1]) and np.all(ty[:, 0] == ty[:, -1])        # x fastest, row-major
    assert abs(tx.mean() - 0.1) < 1e-15 and abs(ty.mean() + 0.2) < 1e-15     # centred on (cx, cy)
    # the s x s sub-rays of pixel (j,i) are symmetric about the pixel centre of the s=1 grid
    px, py = orc.grid(nx, ny, ps, 0.1, -0.2, 1)
    px = px.reshape(ny, nx)
    py = py.reshape(ny, nx)
    for j in range(ny):
        for i in range(nx):
            assert abs(tx[j * s:(j + 1) * s, i * s:(i + 1) * s].mean() - px[j, i]) < 1e-15
            assert abs(ty[j * s:(j + 1) * s, i * s:(i + 1) * s].mean() - py[j, i]) < 1e-15
    # C0: 60 px of 0.05": outermost pixel centres at +-1.475
    tx, ty = orc.grid(60, 60, 0.05)
    assert abs(tx[0] + 1.475) < 1e-15 and abs(tx[59] - 1.475) < 1e-15 and abs(ty[-1] - 1.475) < 1e-15


# ---------------------------------------------------------------- R
@pytest.mark.parametrize("n", [0.5, 1.0, 1.5, 4.0])
def test_sersic_isophote_equals_amp(orc, n):
    """I = amp on the R = R_sersic isophote for any n, e (closed form)."""
    amp, Rs, e1, e2, cx, cy = 7.0, 0.3, 0.15, -0.1, 0.05, -0.02
    phi, q = orc.ellipticity(e1, e2)
    for t in np.linspace(0, 2 * math.pi, 9):
        xr = Rs / math.sqrt(q) * math.cos(t)          # q x'^2 + y'^2/q = Rs^2
        yr = Rs * math.sqrt(q) * math.sin(t)
        x = cx + math.cos(phi) * xr - math.sin(phi) * yr
        y = cy + math.sin(phi) * xr + math.cos(phi) * yr
        assert abs(orc.sersic(x, y, amp, Rs, n, e1, e2, cx, cy) - amp) < 1e-13 * amp


@pytest.mark.parametrize("n,e1,e2", [(1.5, 0.0, 0.0), (1.0, 0.3, -0.2), (2.5, -0.1, 0.25)])
def test_sersic_total_flux_closed_form(orc, n, e1, e2):
    """Total flux = amp Rs^2 2 pi n e^b b^(-2n) Gamma(2n), independent of (e1,e2,centre): pins the
    product-averaged elliptical radius (Q11) and b_n's use."""
    amp, Rs = 1.0, 0.7
    b = 1.9992 * n - 0.3271
    want = amp * Rs ** 2 * 2 * math.pi * n * math.exp(b) * b ** (-2 * n) * special.gamma(2 * n)
    f = lambda r, t: orc.sersic(0.2 + r * math.cos(t), -0.1 + r * math.sin(t), amp, Rs, n, e1, e2, 0.2, -0.1) * r
    got, _ = integrate.dblquad(f, 0, 2 * math.pi, 0, 200.0, epsabs=1e-11, epsrel=1e-11)
    assert abs(got - want) < 2e-8 * want


def _golden(name):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    return np.loadtxt(path, comments="#", ndmin=2)


@pytest.mark.parametrize("row", range(4))
def test_sersic_half_light_fraction_pins_bn(orc, row):
    """Pins the constants of b_n (reading Q10) without retyping them: the flux of orc.sersic inside the R_sersic isophote
    over its total flux, both by quadrature of the oracle's own function, against (i) the four values SURVEY.md section
    8(c) Q10 prints for this reading (tests/golden/sersic_half_light.txt), (ii) scipy's regularised incomplete gamma
    function at the b recovered from the oracle's centre value I(0)/amp = e^b, and (iii) the definition of a half-light
    radius (fraction near 1/2 for n in [0.5, 4]).  A wrong digit in either constant moves the fraction by > 1e-3."""
    n, want = _golden("sersic_half_light.txt")[row]
    amp, Rs = 2.0, 0.35
    prof = lambda r: orc.sersic(r, 0.0, amp, Rs, n, 0.0, 0.0, 0.0, 0.0) * r
    inner, _ = integrate.quad(prof, 0.0, Rs, epsabs=1e-13, epsrel=1e-12, limit=400)
    outer = sum(integrate.quad(prof, a, b, epsabs=1e-13, epsrel=1e-12, limit=400)[0]
                for a, b in ((Rs, 10 * Rs), (10 * Rs, 1e3 * Rs), (1e3 * Rs, 1e6 * Rs)))
    frac = inner / (inner + outer)
    assert abs(frac - want) < 2e-4                                         # the survey's printed value (4 digits)
    b = math.log(orc.sersic(0.0, 0.0, amp, Rs, n, 0.0, 0.0, 0.0, 0.0) / amp)
    assert abs(frac - special.gammainc(2 * n, b)) < 1e-9                   # textbook closed form P(2n, b)
    assert abs(frac - 0.5) < 0.011                                         # R_sersic is (nearly) the half-light radius
    # the same fraction for an elliptical source: the isophote region q x'^2 + y'^2/q <= Rs^2 (2-D quadrature)
    if n == 1.5:
        e1, e2 = 0.2, -0.15
        phi, q = orc.ellipticity(e1, e2)

        def f(u, t):        # u in [0,1]: elliptical radius u Rs; area element Rs^2 u du dt (unit Jacobian of the q-stretch)
            xr, yr = u * Rs / math.sqrt(q) * math.cos(t), u * Rs * math.sqrt(q) * math.sin(t)
            x = math.cos(phi) * xr - math.sin(phi) * yr
            y = math.sin(phi) * xr + math.cos(phi) * yr
            return orc.sersic(x, y, amp, Rs, n, e1, e2, 0.0, 0.0) * Rs * Rs * u
        inner2, _ = integrate.dblquad(f, 0, 2 * math.pi, 0, 1.0, epsabs=1e-11, epsrel=1e-11)
        assert abs(inner2 / (2 * math.pi * (inner + outer)) - want) < 2e-4


def test_sersic_centre_and_profile(orc):
    n, Rs = 2.0, 0.4
    b = 1.9992 * n - 0.3271
    assert abs(orc.sersic(0.1, 0.2, 3.0, Rs, n, 0.1, 0.1, 0.1, 0.2) - 3.0 * math.exp(b)) < 1e-12   # R = 0: amp e^b
    # circular: I(r) = amp exp(-b((r/Rs)^(1/n) - 1))
    r = 0.9
    want = 3.0 * math.exp(-b * ((r / Rs) ** (1 / n) - 1))
    assert abs(orc.sersic(r, 0.0, 3.0, Rs, n, 0.0, 0.0, 0.0, 0.0) - want) < 1e-14 * want
    # e1 > 0 stretches along x: brighter on the x axis than on the y axis at equal distance
    assert orc.sersic(r, 0, 3.0, Rs, n, 0.3, 0.0, 0, 0) > orc.sersic(0, r, 3.0, Rs, n, 0.3, 0.0, 0, 0)


def test_source_brightness_sums_components(orc):
    rng = np.random.default_rng(7)
    src = np.array([[5.0, 0.2, 1.0, 0.1, 0.0, 0.0, 0.0], [9.0, 0.4, 3.0, -0.1, 0.2, 0.1, -0.1]])
    bx, by = rng.uniform(-1, 1, 50), rng.uniform(-1, 1, 50)
    got = orc.source_brightness(bx, by, src)
    for i in range(50):
        want = orc.sersic(bx[i], by[i], *src[0]) + orc.sersic(bx[i], by[i], *src[1])
        assert abs(got[i] - want) < 1e-13 * want


# ---------------------------------------------------------------- B
@pytest.mark.parametrize("s", [1, 2, 3, 5])
def test_bin_constant_and_linear(orc, s):
    nx, ny, ps = 7, 5, 0.08
    tx, ty = orc.grid(nx, ny, ps, 0.0, 0.0, s)
    img = orc.bin_rays(nx, ny, s, ps, np.full(tx.size, 2.5))
    assert np.allclose(img, 2.5 * ps * ps, rtol=1e-15)                     # mean x pixel area (Q14)
    # a linear "source": the binned value is the value at the pixel centre for any s (Q13)
    f = 1.0 + 0.3 * tx - 0.7 * ty
    img = orc.bin_rays(nx, ny, s, ps, f)
    px, py = orc.grid(nx, ny, ps)
    want = (1.0 + 0.3 * px - 0.7 * py).reshape(ny, nx) * ps * ps
    assert np.max(np.abs(img - want)) < 1e-15
    # row/column orientation: a ramp in x only varies along the last axis
    img = orc.bin_rays(nx, ny, s, ps, tx)
    assert np.allclose(img[0], img[-1]) and img[0, -1] > img[0, 0]


# ---------------------------------------------------------------- P
def test_convolve_delta_and_shift(orc):
    rng = np.random.default_rng(8)
    img = rng.uniform(size=(9, 12))
    k = np.zeros((5, 7))
    k[2, 3] = 1.0
    assert np.array_equal(orc.convolve(img, k), img)                       # delta -> identity
    k = np.zeros((5, 7))
    k[2 + 1, 3 + 2] = 1.0                                                  # tap at centre + (1, 2)
    out = orc.convolve(img, k)
    want = np.zeros_like(img)
    want[1:, 2:] = img[:-1, :-2]                                           # out[j][i] = img[j-1][i-2]
    assert np.array_equal(out, want)


def test_convolve_equals_scipy_convolve2d(orc):
    rng = np.random.default_rng(9)
    for (ny, nx, ky, kx) in [(8, 8, 5, 3), (13, 7, 3, 9), (6, 10, 11, 11), (20, 17, 7, 5)]:
        img = rng.normal(size=(ny, nx))
        k = rng.normal(size=(ky, kx))
        want = signal.convolve2d(img, k, mode="same", boundary="fill")
        assert np.max(np.abs(orc.convolve(img, k) - want)) < 1e-13
        assert np.max(np.abs(orc.convolve(img, k) - signal.fftconvolve(img, k, mode="same"))) < 1e-12


def test_convolve_brute_force_8x8(orc):
    """O(N^2 K^2) definition with explicit zero padding, written independently as a full 'scatter'."""
    rng = np.random.default_rng(10)
    img = rng.uniform(size=(8, 8))
    k = rng.uniform(size=(5, 5))
    full = np.zeros((8 + 4, 8 + 4))
    for j in range(8):
        for i in range(8):
            for u in range(5):
                for v in range(5):
                    full[j + u, i + v] += img[j, i] * k[u, v]          # each source pixel spreads the kernel
    want = full[2:10, 2:10]
    assert np.max(np.abs(orc.convolve(img, k) - want)) < 1e-14


def test_convolve_flux_conservation(orc):
    rng = np.random.default_rng(11)
    k = workloads.mixture3_psf(rng, 7, 2.0)
    assert abs(k.sum() - 1.0) < 1e-15
    img = np.zeros((20, 20))
    img[3:-3, 3:-3] = rng.uniform(size=(14, 14))                           # zero within K//2 of the border
    assert abs(orc.convolve(img, k).sum() - img.sum()) < 1e-12


def test_convolve_kernel_larger_than_image(orc):
    rng = np.random.default_rng(12)
    img = rng.uniform(size=(4, 5))
    k = rng.uniform(size=(9, 11))
    want = signal.convolve2d(img, k, mode="full")[4:8, 5:10]
    assert np.max(np.abs(orc.convolve(img, k) - want)) < 1e-13


# ---------------------------------------------------------------- composition
def test_no_lens_constant_source_image(orc):
    """No deflectors + (nearly) flat source => pre-PSF image == c pixel_scale^2 (G, B pin)."""
    w = workloads.config_c0(nx=12)
    w.sie = None
    w.shear = None
    w.sources = np.array([[3.0, 1e6, 1.0, 0.0, 0.0, 0.0, 0.0]])           # R_sersic huge -> I = amp e^b, flat
    pre, out = orc.simulate_image(w)
    b = 1.9992 - 0.3271
    assert np.allclose(pre, 3.0 * math.exp(b) * 0.05 ** 2, rtol=1e-5)


@pytest.mark.parametrize("cfg", ["c0", "c1", "c2"])
def test_simulate_image_is_composition_of_steps(orc, cfg):
    w = {"c0": lambda: workloads.config_c0(nx=20),
         "c1": lambda: workloads.config_c1(nx=16, K=9),
         "c2": lambda: workloads.config_c2(nx=12, n_tnfw=40, K=7)}[cfg]()
    pre, out = orc.simulate_image(w)
    tx, ty = orc.grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
    bx, by = orc.ray_shoot(tx, ty, w.sie, w.shear, w.tnfw)
    f = orc.source_brightness(bx, by, w.sources)
    pre2 = orc.bin_rays(w.nx, w.ny, w.supersample, w.pixel_scale, f)
    assert rel_err(pre, pre2) < 1e-15
    assert rel_err(out, orc.convolve(pre2, w.psf)) < 1e-15
    assert np.array_equal(orc.prepsf_rows(w, 3, 7), pre[3:7])
    assert out.max() > 0


def test_simulate_batch_matches_single(orc):
    bw = workloads.config_c3(B=3, nx=10, n_tnfw=5, K=5, dtype="f64")
    out = orc.simulate_batch(bw)
    for b in range(3):
        _, single = orc.simulate_image(bw.system(b))
        assert np.array_equal(out[b], single)
    sub = orc.simulate_batch(bw, systems=[2])
    assert np.array_equal(sub[0], out[2])


# ---------------------------------------------------------------- workloads (host logic)
def test_workload_shapes_and_seeding():
    c0 = workloads.config_c0()
    assert c0.psf.shape == (11, 11) and abs(c0.psf.sum() - 1) < 1e-15 and c0.evals == 7200
    assert c0.psf[0, 0] / c0.psf[5, 5] < 1e-14                           # corner/peak ~ 9e-16 (D3)
    c1 = workloads.config_c1()
    assert c1.n_rays == 90000 and c1.psf.shape == (31, 31) and c1.sources.shape == (2, 7)
    assert 0.8 <= c1.sie[0] <= 1.5
    assert not np.allclose(c1.psf, c1.psf[::-1, ::-1])                     # asymmetric on purpose
    c2 = workloads.config_c2(n_tnfw=100)
    assert c2.tnfw.shape == (5, 100) and np.all(c2.tnfw[4] == 5 * c2.tnfw[2])
    assert np.all((c2.tnfw[2] >= 0.005) & (c2.tnfw[2] <= 0.05))
    a = workloads.config_c2(n_tnfw=100)
    assert np.array_equal(a.tnfw, c2.tnfw)                                 # same seed, same draws
    c2f = c2.as_dtype("f32")
    assert np.array_equal(c2f.tnfw, c2f.tnfw.astype(np.float32).astype(np.float64))
    c3 = workloads.config_c3(B=4)
    assert c3.tnfw.shape == (4, 5, 100) and c3.psf.shape == (4, 21, 21) and c3.dtype == "f32"
    assert np.allclose(c3.psf.sum(axis=(1, 2)), 1.0, atol=1e-6)
    c4 = workloads.config_c4(nx=10, n_tnfw=20)
    assert c4.psf.shape == (101, 101) and np.all(c4.psf > 0) and c4.sources.shape == (3, 7)
    full = workloads.config_c2()
    assert full.evals == 1_600_320_000


def test_prepsf_pixels_matches_rows(orc):
    """The pixel sampler used for full-size C4 parity equals the row routine on a small C4-shaped case."""
    import workloads
    w = workloads.config_c4(nx=12, n_tnfw=40, K=5, half_width=0.3)
    rows = orc.prepsf_rows(w, 0, w.ny)
    cols = np.array([0, 3, 7, 11])
    for j in (0, 5, 11):
        np.testing.assert_allclose(orc.prepsf_pixels(w, j, cols), rows[j, cols], rtol=1e-13, atol=0)
