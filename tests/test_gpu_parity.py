"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json:north_star): max|diff|/max|img| <= 1e-10 in float64 and <= 2e-4 in float32 for images;
per-step tolerances are derived in DESIGN.md "Tolerances".  float32 cases feed both sides the SAME
float32-rounded inputs (reading Q19), so the comparison measures arithmetic error only.
"""
import numpy as np
import pytest

import workloads
from conftest import gpu_simulate, rel_err, to_dev

pytestmark = pytest.mark.gpu

TOL_IMG = {"f64": 1e-10, "f32": 2e-4}


def _rand_lens(rng, M, half=1.5):
    t = np.zeros((5, M))
    t[0] = rng.uniform(-half, half, M)
    t[1] = rng.uniform(-half, half, M)
    t[2] = np.exp(rng.uniform(np.log(0.005), np.log(0.05), M))
    t[3] = np.exp(rng.uniform(np.log(1e-4), np.log(1e-2), M))
    t[4] = 5.0 * t[2]
    return t


def _f32r(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)


def _trace_plan(jt, w):
    """Launch shape of the ray-tracing kernel for a workloads.Workload (jt_trace_plan_query)."""
    return jt.trace_plan(w.dtype, jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample), n_tnfw=w.n_tnfw)


# ------------------------------------------------------------------ step 1: jt_ray_shoot
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n,M", [(1, 0), (5000, 0), (4097, 1), (3001, 700), (20000, 513), (20000, 10000)])
def test_ray_shoot_random(jt, orc, dtype, n, M):
    """Arbitrary ray positions (RAYS mode of k_trace); the last case is C2's subhalo count on 20,000 random rays."""
    plan = jt.trace_plan(dtype, None, n_rays=n, n_tnfw=M)
    assert plan["rays_per_thread"] == 8 and plan["wide"] == 0
    assert (plan["n_chunks"] > 1) == (M >= 513), plan          # few ray tiles + many subhalos: the list is split over CTAs
    if M == 10000:
        assert plan["tile_recs"] >= 160 and plan["chunk_len"] > plan["tile_recs"]         # the record ring is refilled within a CTA
    rng = np.random.default_rng(100 + n + M)
    tx, ty = rng.uniform(-1.5, 1.5, n), rng.uniform(-1.5, 1.5, n)
    tn = _rand_lens(rng, M)
    sie, shear = (1.1, 0.12, -0.07, 0.02, -0.01), (0.03, -0.02)
    if dtype == "f32":
        tx, ty, tn, sie, shear = _f32r(tx), _f32r(ty), _f32r(tn), tuple(_f32r(sie)), tuple(_f32r(shear))
    bx, by = jt.ray_shoot(to_dev(tx, dtype), to_dev(ty, dtype), sie, shear, to_dev(tn, dtype) if M else None)
    wx, wy = orc.ray_shoot(tx, ty, sie, shear, tn)
    tol = 2e-12 if dtype == "f64" else 4e-7          # f32: output storage alone is 1.2e-7 at |beta| ~ 1.5
    assert np.max(np.abs(bx.double().cpu().numpy() - wx)) < tol
    assert np.max(np.abs(by.double().cpu().numpy() - wy)) < tol


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ray_shoot_through_subhalo_cores(jt, orc, dtype):
    """Rays placed at X = R/Rs from 1e-5 to 30 around subhalos: series, core, X~1 and far branches (definition T)."""
    rng = np.random.default_rng(7)
    M = 64
    tn = _rand_lens(rng, M, half=1.0)
    tn[4] = tn[2] * rng.uniform(0.5, 20.0, M)              # tau from 0.5 to 20, both sides of tau = 1
    X = np.concatenate([np.logspace(-5, 1.5, 40), [0.999, 1.0, 1.001, 0.5, 2.0 ** 0.5, 10 ** 0.5]])
    tx, ty = [], []
    for j in range(M):
        ang = rng.uniform(0, 2 * np.pi, X.size)
        tx.append(tn[0, j] + X * tn[2, j] * np.cos(ang))
        ty.append(tn[1, j] + X * tn[2, j] * np.sin(ang))
    tx, ty = np.concatenate(tx), np.concatenate(ty)
    tx = np.append(tx, tn[0, 0])                            # a ray exactly on a centre: alpha = 0 there
    ty = np.append(ty, tn[1, 0])
    if dtype == "f32":
        tx, ty, tn = _f32r(tx), _f32r(ty), _f32r(tn)
    bx, by = jt.ray_shoot(to_dev(tx, dtype), to_dev(ty, dtype), None, None, to_dev(tn, dtype))
    wx, wy = orc.ray_shoot(tx, ty, None, None, tn)
    tol = 2e-13 if dtype == "f64" else 4e-7
    assert np.max(np.abs(bx.double().cpu().numpy() - wx)) < tol
    assert np.max(np.abs(by.double().cpu().numpy() - wy)) < tol
    if dtype == "f64":                                      # deflection itself, relative
        ax, wax = tx - bx.double().cpu().numpy(), tx - wx
        assert np.max(np.abs(ax - wax)) < 1e-10 * np.max(np.abs(wax))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ray_shoot_far_far_series(jt, orc, dtype):
    """One subhalo at a time, rays at X = R/Rs from 4 to 1e4 times max(1, tau), tau from 0.3 to 1000: both sides of
    the far-far radius (9 / 8 max(1, tau)) where the kernel switches from the far form to the 1/X series of the brace.
    The deflection itself is compared, relative to its own size (reading Q9b: series error <= 1e-13 / 2e-8 at
    the radius, falling like (max(1, tau) / X)^14 beyond it, for EVERY tau -- the radius scales with tau; records whose
    coefficients leave the dtype's range, float beyond tau ~ 1e3, keep the far form)."""
    rng = np.random.default_rng(17)
    worst = 0.0
    for tau in (0.3, 0.7, 1.0, 2.0, 5.0, 12.0, 30.0, 60.0, 200.0, 1000.0):
        Rs, aRs = 0.01, 5e-3
        tn = np.array([[0.013], [-0.007], [Rs], [aRs], [tau * Rs]])
        X = np.concatenate([np.logspace(np.log10(4.0), 4.0, 600), np.linspace(7.5, 10.5, 200)]) * max(1.0, tau)
        ang = rng.uniform(0, 2 * np.pi, X.size)
        tx = tn[0, 0] + X * Rs * np.cos(ang)
        ty = tn[1, 0] + X * Rs * np.sin(ang)
        if dtype == "f32":
            tx, ty, tn = _f32r(tx), _f32r(ty), _f32r(tn)
        bx, by = jt.ray_shoot(to_dev(tx, dtype), to_dev(ty, dtype), None, None, to_dev(tn, dtype))
        wx, wy = orc.ray_shoot(tx, ty, None, None, tn)
        ax, ay = tx - bx.double().cpu().numpy(), ty - by.double().cpu().numpy()
        wax, way = tx - wx, ty - wy
        mag = np.hypot(wax, way)
        if dtype == "f64":
            # beta = theta - alpha is stored in double: alpha is recovered to ~1e-16 |theta|
            err = np.hypot(ax - wax, ay - way) / (mag + 1e-16 * np.hypot(tx, ty) / 1e-12)
            worst = max(worst, float(err.max()))
        else:
            # float: beta is stored in float (half an ulp of |theta| = 6e-8 |theta|) and the float arithmetic of one
            # evaluation is good to a few 1e-7 of alpha; the series adds 2e-8
            err = np.hypot(ax - wax, ay - way) / (3e-6 * mag + 2e-7 * np.hypot(tx, ty))
            worst = max(worst, float(err.max()))
    assert worst < (1e-11 if dtype == "f64" else 1.0), worst


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ray_shoot_extreme_truncation(jt, orc, dtype):
    """tau = r_trunc/Rs far outside the priors (100 ... 1e5): the far-far coefficients grow like tau^12; records whose
    coefficients leave the dtype's range must fall back to the far form -- finite results that still match."""
    rng = np.random.default_rng(23)
    for tau in (100.0, 3.0e3, 1.0e5):
        Rs = 0.01
        tn = np.array([[0.0], [0.0], [Rs], [1e-3], [tau * Rs]])
        X = np.logspace(0.5, 7.0, 400)
        ang = rng.uniform(0, 2 * np.pi, X.size)
        tx, ty = X * Rs * np.cos(ang), X * Rs * np.sin(ang)
        if dtype == "f32":
            tx, ty, tn = _f32r(tx), _f32r(ty), _f32r(tn)
        bx, by = jt.ray_shoot(to_dev(tx, dtype), to_dev(ty, dtype), None, None, to_dev(tn, dtype))
        bx, by = bx.double().cpu().numpy(), by.double().cpu().numpy()
        assert np.isfinite(bx).all() and np.isfinite(by).all(), tau
        wx, wy = orc.ray_shoot(tx, ty, None, None, tn)
        scale = np.hypot(tx - wx, ty - wy) * (1e-9 if dtype == "f64" else 1e-5) + np.hypot(tx, ty) * (1e-15 if dtype == "f64" else 2e-7)
        assert (np.hypot(bx - wx, by - wy) <= scale).all(), tau


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("e1,e2", [(-0.3, 0.35), (0.0, 0.0), (1e-9, 0.0), (0.6, -0.5), (0.9, 0.9), (-0.19, -0.12)])
def test_ray_shoot_sie_ellipticities(jt, orc, dtype, e1, e2):
    """SIE alone over the full range of definition E: q below 0.707 (f x'/psi above 1), circular, |e| clamped."""
    rng = np.random.default_rng(21)
    n = 6000
    tx, ty = rng.uniform(-2, 2, n), rng.uniform(-2, 2, n)
    tx[:4], ty[:4] = [0.3, 0.3, 1e-7, -1.5], [0.0, 1e-9, 0.4, 1e-12]        # on and next to the principal axes
    sie = (1.2, e1, e2, 0.05, -0.02)
    if dtype == "f32":
        tx, ty, sie = _f32r(tx), _f32r(ty), tuple(_f32r(sie))
    bx, by = jt.ray_shoot(to_dev(tx, dtype), to_dev(ty, dtype), sie, None, None)
    wx, wy = orc.ray_shoot(tx, ty, sie, None, None)
    tol = 2e-13 if dtype == "f64" else 4e-7
    if e1 * e1 + e2 * e2 > 0.98:
        # clamped |e| = 0.9999: q = 5e-5, atanh(z) is evaluated at 1 - z^2 down to q^2 = 2.5e-9, where a 1e-16 relative
        # error in z moves the result by 1e-16 / 2.5e-9 = 4e-8: both sides are conditioning-limited, not wrong
        tol = 2e-7
    assert np.max(np.abs(bx.double().cpu().numpy() - wx)) < tol
    assert np.max(np.abs(by.double().cpu().numpy() - wy)) < tol


def test_ray_shoot_empty(jt):
    import torch
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    bx, by = jt.ray_shoot(e, e.clone(), (1.0, 0, 0, 0, 0), None, None)
    assert bx.numel() == 0 and by.numel() == 0


# ------------------------------------------------------------------ step 2: jt_source_brightness
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_source_brightness(jt, orc, dtype):
    rng = np.random.default_rng(11)
    n = 10007
    bx, by = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    bx[:3], by[:3] = [0.1, 0.1 + 1e-9, 5.0], [-0.05, -0.05, 5.0]       # exactly on a centre; just off; far out
    src = np.array([[10.0, 0.2, 1.5, 0.05, 0.02, 0.1, -0.05], [7.0, 0.4, 4.0, -0.15, 0.1, -0.2, 0.1],
                    [12.0, 0.15, 0.5, 0.0, 0.0, 0.0, 0.0]])
    if dtype == "f32":
        bx, by, src = _f32r(bx), _f32r(by), _f32r(src)
    got = jt.source_brightness(to_dev(bx, dtype), to_dev(by, dtype), src).double().cpu().numpy()
    want = orc.source_brightness(bx, by, src)
    assert rel_err(got, want) < (1e-13 if dtype == "f64" else 2e-5)


# ------------------------------------------------------------------ step 3: jt_psf_convolve (direct)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("ny,nx,ky,kx", [(8, 8, 3, 3), (8, 8, 5, 3), (60, 60, 11, 11), (100, 100, 31, 31),
                                         (64, 64, 21, 21), (37, 91, 7, 13), (130, 75, 45, 45), (5, 7, 11, 9),
                                         (200, 200, 21, 21), (33, 31, 1, 1), (180, 180, 135, 135), (301, 203, 101, 7),
                                         (300, 420, 101, 101), (64, 1000, 3, 201), (70, 66, 151, 9)])
def test_convolve_direct(jt, orc, dtype, ny, nx, ky, kx):
    plan = jt.psf_convolve_plan(dtype, ny, nx, ky, kx, method="direct")
    assert plan["method"] == "direct"
    # every launch shape of the direct convolution is named by a case here (jt_psf_convolve_plan)
    expect = {(8, 8, 3, 3): "small", (60, 60, 11, 11): "small", (37, 91, 7, 13): "small", (33, 31, 1, 1): "small",
              (100, 100, 31, 31): "tile", (64, 64, 21, 21): "tile", (130, 75, 45, 45): "tile", (200, 200, 21, 21): "tile",
              (180, 180, 135, 135): "tile", (300, 420, 101, 101): "tile"}
    if (ny, nx, ky, kx) in expect:
        assert plan["path"] == expect[(ny, nx, ky, kx)], plan
    if (ny, nx, ky, kx) in ((100, 100, 31, 31), (64, 64, 21, 21), (200, 200, 21, 21)):
        assert plan["tma"] == 1 and plan["z_split"] > 1 and plan["row_bands"] == 1, plan     # TMA tile, column pairs split (L2 reduction)
    if (ny, nx, ky, kx) == (130, 75, 45, 45):
        assert plan["tma"] == 0, plan                                    # 75-element rows: pitch not a multiple of 16 bytes -> plain loads
    if (ny, nx, ky, kx) == (180, 180, 135, 135):
        assert plan["row_bands"] > 1 and plan["tma"] == 1, plan          # taps exceed the 60 KB constant bank: bands of kernel rows
    rng = np.random.default_rng(ny * 1000 + nx + ky)
    img = rng.uniform(0, 1, (ny, nx))
    ker = rng.uniform(0, 1, (ky, kx))
    ker /= ker.sum()
    if dtype == "f32":
        img, ker = _f32r(img), _f32r(ker)
    got = jt.psf_convolve(to_dev(img, dtype), to_dev(ker, dtype), method="direct").double().cpu().numpy()
    want = orc.convolve(img, ker)
    # f32: ky*kx sequential float additions of positive terms, random-walk rounding ~ sqrt(ky kx) 2^-24
    assert rel_err(got, want) < (1e-13 if dtype == "f64" else max(2e-6, 3.0 * (ky * kx) ** 0.5 * 2.0 ** -24))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("B,ny,nx,k", [(5, 60, 60, 21), (3, 100, 100, 13), (7, 33, 47, 45), (2, 180, 180, 135), (130, 16, 20, 5)])
def test_convolve_batch(jt, orc, dtype, B, ny, nx, k):
    """jt_psf_convolve_batch (B images, one kernel) = the oracle's convolution image by image, both methods;
    covers the TMA tile path (aligned pitch) and the plain-load fallback (33 x 47: odd pitch)."""
    plan = jt.psf_convolve_plan(dtype, ny, nx, k, k, method="direct", B=B)
    assert plan["path"] == "tile", plan                                  # the one-launch kernel is for single images only
    assert plan["tma"] == (0 if (ny, nx) == (33, 47) else 1), plan
    if B == 130:
        assert plan["z_split"] == 1, plan                                # enough tiles: no split, no L2 reduction
    if k == 135:
        assert plan["row_bands"] > 1, plan
    assert jt.psf_convolve_plan(dtype, ny, nx, k, k, method="fft", B=B)["path"] == "fft"
    rng = np.random.default_rng(B * 100 + k)
    imgs = rng.uniform(0, 1, (B, ny, nx))
    ker = rng.uniform(0, 1, (k, k))
    ker /= ker.sum()
    if dtype == "f32":
        imgs, ker = _f32r(imgs), _f32r(ker)
    want = np.stack([orc.convolve(imgs[b], ker) for b in range(B)])
    for method in ("direct", "fft", "auto"):
        got = jt.psf_convolve_batch(to_dev(imgs, dtype), to_dev(ker, dtype), method=method).double().cpu().numpy()
        assert rel_err(got, want) < (1e-12 if dtype == "f64" else max(2e-6, 3.0 * k * 2.0 ** -24)), method


def test_convolve_direct_unaligned_view(jt, orc):
    """An image whose base address is not 16-byte aligned takes the plain-load tile fill, same result."""
    rng = np.random.default_rng(12)
    flat = to_dev(rng.uniform(0, 1, 64 * 64 + 1), "f32")
    img = flat[1:].view(64, 64)
    ker = to_dev(rng.uniform(0, 1, (21, 21)) / 220.0, "f32")             # 21 x 21: the tile kernel (9 x 9 would take the one-launch path)
    aligned = jt.psf_convolve_plan("f32", 64, 64, 21, 21, method="direct")
    plan = jt.psf_convolve_plan("f32", 64, 64, 21, 21, method="direct", image=img)
    assert aligned["path"] == plan["path"] == "tile" and aligned["tma"] == 1 and plan["tma"] == 0, (aligned, plan)
    got = jt.psf_convolve(img, ker, method="direct").double().cpu().numpy()
    want = orc.convolve(img.double().cpu().numpy(), ker.double().cpu().numpy())
    assert rel_err(got, want) < max(2e-6, 3.0 * 21 * 2.0 ** -24)


def test_convolve_delta_and_shift(jt):
    """delta kernel = identity; a single off-centre tap shifts by (+du, +dv) (definition P orientation)."""
    import torch
    rng = np.random.default_rng(5)
    img = to_dev(rng.uniform(0, 1, (40, 50)), "f64")
    k = torch.zeros(7, 5, dtype=torch.float64, device="cuda")
    k[3, 2] = 1.0
    assert torch.equal(jt.psf_convolve(img, k, method="direct"), img)
    k.zero_()
    k[3 + 1, 2 + 2] = 1.0
    out = jt.psf_convolve(img, k, method="direct")
    assert torch.equal(out[1:, 2:], img[:-1, :-2]) and float(out[0].abs().max()) == 0.0


# ------------------------------------------------------------------ step 3: jt_psf_convolve (hand-written FFT)
FFT_SHAPES = [(8, 8, 3, 3), (8, 8, 5, 3), (60, 60, 11, 11), (100, 100, 31, 31), (64, 64, 21, 21), (37, 91, 7, 13),
              (130, 75, 45, 45), (5, 7, 11, 9), (200, 200, 21, 21), (33, 31, 1, 1), (180, 180, 135, 135),
              (60, 60, 45, 45), (300, 420, 101, 101), (17, 1000, 3, 61), (1100, 9, 77, 5)]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("ny,nx,ky,kx", FFT_SHAPES)
def test_convolve_fft(jt, orc, dtype, ny, nx, ky, kx):
    """FFT path against the oracle's literal quadruple loop (the FFT reaches the direct result up to rounding)."""
    rng = np.random.default_rng(ny * 1000 + nx + ky)
    img = rng.uniform(0, 1, (ny, nx))
    ker = rng.uniform(0, 1, (ky, kx))
    ker /= ker.sum()
    if dtype == "f32":
        img, ker = _f32r(img), _f32r(ker)
    got = jt.psf_convolve(to_dev(img, dtype), to_dev(ker, dtype), method="fft").double().cpu().numpy()
    want = orc.convolve(img, ker)
    # ~log2(Py Px) <= 24 butterfly levels, each adding one rounding of relative size eps to values of size <= max|img|
    assert rel_err(got, want) < (1e-12 if dtype == "f64" else 2e-6)     # f32: transforms run in double, output rounding only


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_convolve_fft_vs_direct_vs_cufft(jt, dtype):
    """Three-way agreement: own FFT path, direct path, and a cuFFT-based convolution (torch.fft; test only)."""
    import torch
    rng = np.random.default_rng(77)
    ny, nx, ky, kx = 150, 170, 41, 37
    img = to_dev(rng.uniform(0, 1, (ny, nx)), dtype)
    ker = to_dev(rng.uniform(0, 1, (ky, kx)) / (ky * kx * 0.5), dtype)
    a = jt.psf_convolve(img, ker, method="fft")
    b = jt.psf_convolve(img, ker, method="direct")
    sy, sx = ny + ky - 1, nx + kx - 1
    full = torch.fft.irfft2(torch.fft.rfft2(img.double(), s=(sy, sx)) * torch.fft.rfft2(ker.double(), s=(sy, sx)), s=(sy, sx))
    c = full[ky // 2:ky // 2 + ny, kx // 2:kx // 2 + nx]
    tol = 1e-12 if dtype == "f64" else 2e-5
    m = float(c.abs().max())
    assert float((a.double() - c).abs().max()) < tol * m
    assert float((b.double() - c).abs().max()) < tol * m
    assert float((a.double() - b.double()).abs().max()) < tol * m


def test_convolve_fft_delta_shift_and_auto(jt):
    """delta kernel = identity and single-tap shift through the FFT path; AUTO resolves to a working method."""
    import torch
    rng = np.random.default_rng(6)
    img = to_dev(rng.uniform(0, 1, (40, 50)), "f64")
    k = torch.zeros(7, 5, dtype=torch.float64, device="cuda")
    k[3, 2] = 1.0
    assert float((jt.psf_convolve(img, k, method="fft") - img).abs().max()) < 1e-13
    k.zero_()
    k[3 + 1, 2 + 2] = 1.0
    out = jt.psf_convolve(img, k, method="fft")
    assert float((out[1:, 2:] - img[:-1, :-2]).abs().max()) < 1e-13 and float(out[0].abs().max()) < 1e-13
    big = to_dev(rng.uniform(0, 1, (61, 61)), "f64")
    big /= big.sum()
    a = jt.psf_convolve(img, big, method="auto")
    b = jt.psf_convolve(img, big, method="direct")
    assert float((a - b).abs().max()) < 1e-13


# ------------------------------------------------------------------ fused: jt_simulate_image
def _check_image(jt, orc, w, method="auto", tol=None):
    pre, want = orc.simulate_image(w)
    got = gpu_simulate(jt, w, method=method)
    got_pre = gpu_simulate(jt, w, conv=False)
    tol = TOL_IMG[w.dtype] if tol is None else tol
    assert rel_err(got_pre, pre) < tol, "pre-PSF image"
    assert rel_err(got, want) < tol, "convolved image"


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config_c0(jt, orc, dtype):
    w = workloads.config_c0(dtype=dtype)
    plan = _trace_plan(jt, w)
    assert plan["rays_per_thread"] == w.supersample == 1 and plan["n_chunks"] == 1, plan      # latency shape: one pixel row per thread
    assert jt.psf_convolve_plan(dtype, w.ny, w.nx, *w.psf.shape, method="direct")["path"] == "small"   # one-launch convolution
    _check_image(jt, orc, workloads.config_c0(dtype=dtype), method="direct")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config_c1(jt, orc, dtype):
    plan = _trace_plan(jt, workloads.config_c1(dtype=dtype))
    assert plan["rays_per_thread"] == 3 and plan["wide"] == 1 and plan["n_chunks"] == 1, plan  # R = s row mode, CTA-wide tiles (s = 3)
    _check_image(jt, orc, workloads.config_c1(dtype=dtype), method="direct")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config_c2_reduced(jt, orc, dtype):
    """C2's recipe at 48x48 pixels and 1,500 subhalos: several subhalo tiles plus a ragged tail, split list."""
    plan = _trace_plan(jt, workloads.config_c2(nx=48, n_tnfw=1500, dtype=dtype))
    assert plan["n_chunks"] > 1 and plan["wide"] == 0 and plan["rays_per_thread"] == 8, plan
    _check_image(jt, orc, workloads.config_c2(nx=48, n_tnfw=1500, dtype=dtype), method="direct")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config_c4_reduced(jt, orc, dtype):
    """C4's recipe (s=5, 3 sources, AiryMix PSF) at 30x30 pixels, 700 subhalos, K=41."""
    plan = _trace_plan(jt, workloads.config_c4(nx=30, n_tnfw=700, K=41, half_width=0.6, dtype=dtype))
    assert plan["wide"] == 1 and plan["rays_per_thread"] == 10 and plan["n_chunks"] > 1, plan  # CTA-wide tiles AND a split list
    _check_image(jt, orc, workloads.config_c4(nx=30, n_tnfw=700, K=41, half_width=0.6, dtype=dtype), method="direct")


@pytest.mark.parametrize("s", [1, 2, 3, 4, 5, 6, 7, 8, 11, 16])
def test_supersampling_factors(jt, orc, s):
    """Every supported s: the warp-shuffle binning (definition B) with ragged tiles, off-centre, non-square grid."""
    w = workloads.config_c1(nx=23, supersample=s, K=9)
    w.ny, w.cx, w.cy = 17, 0.013, -0.021
    assert _trace_plan(jt, w)["wide"] == (1 if 32 % s else 0)              # warp-shuffle binning vs CTA-wide shared-memory binning
    _check_image(jt, orc, w, method="direct")


def test_no_lens_constant_source_invariant(jt):
    """No deflector, very wide n=1 source: image ~ c * pixel_scale^2 (pins G/B independently of the oracle)."""
    g = jt.Grid(16, 12, 0.05, supersample=3)
    src = np.array([[2.0, 1e6, 1.0, 0.0, 0.0, 0.0, 0.0]])
    img = jt.simulate_image(g, None, None, None, src, None, dtype="f64").cpu().numpy()
    b = 1.9992 - 0.3271
    assert np.allclose(img, 2.0 * np.exp(b) * 0.05 ** 2, rtol=1e-5)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_image_edge_cases(jt, orc, dtype):
    """Degenerate shapes of jt_simulate_image: no sources (image = 0), 16 sources (JT_MAX_SOURCES), a 1 x 1 grid,
    s = 16 on a 3 x 2 grid, a non-square PSF through both convolution paths, one subhalo list entry."""
    import torch
    rng = np.random.default_rng(31)
    w = workloads.config_c1(nx=21, supersample=2, K=9, dtype=dtype)
    # no sources
    g = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
    img = jt.simulate_image(g, w.sie, w.shear, to_dev(w.tnfw, dtype), np.zeros((0, 7)), to_dev(w.psf, dtype), dtype=dtype)
    assert float(img.abs().max()) == 0.0
    # 16 sources
    src = np.tile(w.sources[:1], (16, 1))
    src[:, 0] = rng.uniform(1, 3, 16)
    src[:, 5:7] = rng.uniform(-0.3, 0.3, (16, 2))
    w16 = workloads.config_c1(nx=21, supersample=2, K=9, dtype=dtype)
    w16.sources = _f32r(src) if dtype == "f32" else src
    _check_image(jt, orc, w16, method="direct")
    # 1 x 1 grid and s = 16
    for nx, ny, s in ((1, 1, 1), (3, 2, 16)):
        we = workloads.config_c1(nx=nx, supersample=s, K=3, dtype=dtype)
        we.ny = ny
        _check_image(jt, orc, we, method="direct")
    # non-square PSF, both paths
    wn = workloads.config_c1(nx=40, supersample=1, K=9, dtype=dtype)
    psf = rng.uniform(0, 1, (5, 13))
    wn.psf = _f32r(psf / psf.sum()) if dtype == "f32" else psf / psf.sum()
    _check_image(jt, orc, wn, method="direct")
    _check_image(jt, orc, wn, method="fft")
    _check_image(jt, orc, wn, method="auto")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("s", [1, 2, 5])
def test_image_series_levels_and_cores(jt, orc, dtype, s):
    """jt_simulate_image's per-warp-tile sort: a few VERY strong subhalos (alpha_Rs = 0.5-2 arcsec,
    hundreds of times the priors') whose three far-far radii (9 / 20 / 44 max(1, tau) Rs in double, 6.5 / 18 / 32 in float),
    far and near zones all fall inside the grid, so that every warp tile puts some of them in every class; two of them
    sit exactly on a ray and exactly between rays.  The source is broad and shallow (n = 1), so max|img| does not dwarf
    the pixels the subhalos act on.  The float64 tolerance here is 1e-12, a hundred times tighter than the north-star
    bar: the series' truncation bound is 1e-13 of each deflection (measured: 3e-15 ... 7e-15 on this case), while a
    series shortened one level too early (K = 7 from the K = 13 radius on -- tried as a mutation) gives 1.2e-11 ... 7.8e-11."""
    nx, ny, h = 96, 64, 0.05
    tn = np.array([  # cx, cy, Rs, alpha_Rs, r_trunc
        [0.31, -0.22, 0.010, 2.00, 0.010],       # tau = 1: radii 0.09, 0.20, 0.44
        [-1.20, 0.45, 0.004, 2.00, 0.020],       # tau = 5: 0.18, 0.40, 0.88
        [1.05, 0.90, 0.020, 1.00, 0.010],        # tau = 0.5 (max(1, tau) = 1): 0.18, 0.40, 0.88
        [-0.60, -1.10, 0.002, 1.00, 0.040],      # tau = 20: 0.36, 0.80, 1.76
        [0.0, 0.0, 0.006, 0.50, 0.030],          # moved onto a ray below
        [0.0, 0.0, 0.006, 0.50, 0.030],          # moved between four rays below
    ]).T.copy()
    w = workloads.config_c4(nx=nx, n_tnfw=6, K=9, dtype="f64")
    w.ny, w.supersample, w.pixel_scale, w.cx, w.cy = ny, s, h, 0.0, 0.0
    hs = h / s
    x0 = -(nx * s - 1) / 2 * hs
    y0 = -(ny * s - 1) / 2 * hs
    tn[0, 4], tn[1, 4] = x0 + 37 * hs, y0 + 21 * hs                  # exactly on ray (J = 21, I = 37)
    tn[0, 5], tn[1, 5] = x0 + 60.5 * hs, y0 + 40.5 * hs              # centre of a ray cell
    w.tnfw = tn
    w.sources = np.array([[3.0, 0.8, 1.0, 0.0, 0.1, -0.3, 0.2]])
    w = w.as_dtype(dtype)
    _check_image(jt, orc, w, method="direct", tol=1e-12 if dtype == "f64" else None)


@pytest.mark.parametrize("seed", range(16))
def test_image_random_shapes(jt, orc, seed):
    """Seeded random configurations of the fused call: grid shape and offset, supersampling, subhalo count (around the
    staging-tile and chunk-split boundaries), tau from 0.5 to 20 (all four tiers of definition T), 1-3 sources, PSF shape,
    dtype and convolution method."""
    rng = np.random.default_rng(9000 + seed)
    dtype = "f64" if seed % 2 == 0 else "f32"
    nx, ny = int(rng.integers(3, 70)), int(rng.integers(3, 70))
    s = int(rng.choice([1, 2, 3, 4, 5, 7]))
    M = int(rng.choice([0, 1, 31, 255, 257, 700, 1537, 3000]))
    K = (int(rng.choice([1, 3, 9, 21, 33])), int(rng.choice([1, 5, 13, 27])))
    w = workloads.config_c4(nx=nx, n_tnfw=M, K=9, half_width=0.04 * max(nx, ny) * 0.6, dtype="f64")
    w.ny = ny
    w.supersample = s
    w.pixel_scale = 0.04
    w.cx, w.cy = float(rng.uniform(-0.05, 0.05)), float(rng.uniform(-0.05, 0.05))
    if M:
        w.tnfw[4] = w.tnfw[2] * rng.uniform(0.5, 20.0, M)
    w.sources = w.sources[: int(rng.integers(1, 4))]
    psf = rng.uniform(0, 1, K)
    w.psf = psf / psf.sum()
    w = w.as_dtype(dtype)
    _check_image(jt, orc, w, method=str(rng.choice(["direct", "fft", "auto"])))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_c2_full_size_whole_image(jt, orc, dtype):
    """Full-size C2 (200x200, s=2, 10,000 subhalos) in the launch configuration bench.py times: the WHOLE pre-PSF
    image and the whole convolved image against the oracle (1.6e9 ray x deflector evaluations: seconds on the GPU
    box's host cores).  Every warp tile of the grid -- centre, Einstein ring, edges -- takes part, so the
    position-dependent tier decisions (far-far / far / mid / cold) are all covered."""
    w = workloads.config_c2(dtype=dtype)
    plan = _trace_plan(jt, w)
    assert plan["n_chunks"] > 1 and plan["wide"] == 0 and plan["chunk_len"] > 4 * plan["tile_recs"], plan     # split list, long ring runs
    want_pre = orc.prepsf_rows(w, 0, w.ny)
    got_pre = gpu_simulate(jt, w, conv=False)
    assert rel_err(got_pre, want_pre) < TOL_IMG[dtype]
    want = orc.convolve(want_pre, w.psf)
    for method in ("direct", "fft"):
        assert rel_err(gpu_simulate(jt, w, method=method), want) < TOL_IMG[dtype], method


def test_c4_full_size_rows(jt, orc):
    """Full-size C4 (500x500, s=5, 50,000 subhalos, f64, 101x101 AiryMix PSF) in the launch configuration bench.py
    times.  (1) 20 WHOLE pixel rows of the pre-PSF image, spread from the first to the last row, against the oracle
    with all 50,002 deflectors (1.25e10 evaluations, SURVEY.md section 8(d) C4 plan); (2) both convolution methods on
    the FULL image: the oracle's direct convolution of the GPU's pre-PSF image against the GPU's convolved images."""
    w = workloads.config_c4(dtype="f64")
    plan = _trace_plan(jt, w)
    assert plan["wide"] == 1 and plan["rays_per_thread"] == 10 and plan["n_chunks"] == 1 and plan["n_ctas"] == 5000, plan
    cp = jt.psf_convolve_plan("f64", w.ny, w.nx, *w.psf.shape, method="direct")
    assert cp["path"] == "tile" and cp["row_bands"] > 1 and cp["z_split"] > 1, cp
    assert jt.psf_convolve_plan("f64", w.ny, w.nx, *w.psf.shape, method="auto")["path"] == "fft"
    pre = gpu_simulate(jt, w, conv=False)
    scale = np.max(np.abs(pre))
    for j in np.linspace(0, w.ny - 1, 20).astype(int):
        want = orc.prepsf_rows(w, int(j), int(j) + 1)[0]
        assert np.max(np.abs(pre[j] - want)) < TOL_IMG["f64"] * scale, j
    want = orc.convolve(pre, w.psf)
    for method in ("direct", "fft"):
        got = gpu_simulate(jt, w, method=method)
        assert rel_err(got, want) < TOL_IMG["f64"], method


# ------------------------------------------------------------------ batched: jt_simulate_batch
def _gpu_batch(jt, bw, conv=True):
    g = jt.Grid(bw.nx, bw.ny, bw.pixel_scale, bw.cx, bw.cy, bw.supersample)
    d = lambda a: to_dev(a, bw.dtype)
    tn = d(bw.tnfw) if bw.tnfw.shape[2] > 0 else None
    out = jt.simulate_batch(g, d(bw.sie), d(bw.shear), tn, d(bw.sources), d(bw.psf) if conv else None)
    return out.double().cpu().numpy()


def _check_batch(jt, orc, bw):
    want = orc.simulate_batch(bw)
    got = _gpu_batch(jt, bw)
    worst = max(rel_err(got[b], want[b]) for b in range(bw.B))          # reading Q20: per image, worst of the batch
    assert worst < TOL_IMG[bw.dtype], worst


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_batch_c3_reduced(jt, orc, dtype):
    """C3's recipe, 12 systems of 64x64 (s=2, 100 subhalos, own 21x21 PSF): the launch shape bench.py times."""
    _check_batch(jt, orc, workloads.config_c3(B=12, dtype=dtype))


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("nx,s,M,K", [(20, 1, 0, 5), (33, 3, 7, 9), (17, 5, 600, 13), (40, 2, 1100, 31), (9, 4, 3, 21)])
def test_batch_shapes(jt, orc, dtype, nx, s, M, K):
    """Ragged grids, every path of the subhalo staging (none, resident, re-staged in rounds), kernels wider than the image."""
    _check_batch(jt, orc, workloads.config_c3(B=3, nx=nx, supersample=s, n_tnfw=M, K=K, dtype=dtype))


def test_batch_matches_single_image_call(jt):
    """jt_simulate_batch on one system == jt_simulate_image on the same system (same arithmetic, f64)."""
    bw = workloads.config_c3(B=2, nx=48, n_tnfw=300, dtype="f64")
    got = _gpu_batch(jt, bw)
    g = jt.Grid(bw.nx, bw.ny, bw.pixel_scale, bw.cx, bw.cy, bw.supersample)
    for b in range(bw.B):
        one = jt.simulate_image(g, tuple(bw.sie[b]), tuple(bw.shear[b]), to_dev(bw.tnfw[b], "f64"), bw.sources[b],
                                to_dev(bw.psf[b], "f64"), dtype="f64", method="direct").cpu().numpy()
        assert rel_err(got[b], one) < 1e-12


def test_batch_no_psf_and_empty(jt, orc):
    import torch
    bw = workloads.config_c3(B=2, nx=24, n_tnfw=50, dtype="f64")
    got = _gpu_batch(jt, bw, conv=False)
    g = jt.Grid(bw.nx, bw.ny, bw.pixel_scale, bw.cx, bw.cy, bw.supersample)
    for b in range(bw.B):
        one = jt.simulate_image(g, tuple(bw.sie[b]), tuple(bw.shear[b]), to_dev(bw.tnfw[b], "f64"), bw.sources[b],
                                None, dtype="f64").cpu().numpy()
        assert rel_err(got[b], one) < 1e-12
    e = lambda *s: torch.empty(s, dtype=torch.float64, device="cuda")
    out = jt.simulate_batch(g, e(0, 5), e(0, 2), None, e(0, 1, 7), None)
    assert out.shape[0] == 0


def test_batch_c3_full_size(jt, orc):
    """Full C3 (4,096 systems, f32; BASELINE.json configs[3], PAPER.md:47 training-set generation) in the launch
    configuration bench.py times: EVERY system against the oracle ("C0-C3 get full end-to-end
    parity"; 6.8e9 double evaluations, a few tens of seconds on the host cores), each image at the north_star bar."""
    bw = workloads.config_c3(dtype="f32")
    got = _gpu_batch(jt, bw)
    assert np.isfinite(got).all() and (got >= 0).all()
    want = orc.simulate_batch(bw)
    assert want.shape == got.shape == (4096, 64, 64)
    err = np.max(np.abs(got - want), axis=(1, 2)) / np.max(np.abs(want), axis=(1, 2))
    assert float(err.max()) < TOL_IMG["f32"], (int(err.argmax()), float(err.max()))


def test_results_are_bitwise_reproducible(jt):
    """Arrival-order mechanisms (last warp / CTA to arrive reduces the split subhalo list, warp tiles handed out by a
    counter in the batch kernel, convolution partial sums meeting in L2) must not leak into the numbers: every reduction
    runs in a fixed order, so repeated calls agree bit for bit."""
    import torch
    for dtype in ("f64", "f32"):
        w = workloads.config_c2(nx=48, n_tnfw=3000, dtype=dtype)          # few ray tiles: the subhalo list is split
        a = gpu_simulate(jt, w, method="direct")
        for _ in range(3):
            assert np.array_equal(a, gpu_simulate(jt, w, method="direct"))
        w5 = workloads.config_c4(nx=40, n_tnfw=2000, K=31, dtype=dtype)   # s = 5: CTA-wide tiles, per-CTA completion
        b = gpu_simulate(jt, w5, method="direct")
        for _ in range(3):
            assert np.array_equal(b, gpu_simulate(jt, w5, method="direct"))
    bw = workloads.config_c3(B=24, nx=32, n_tnfw=60, dtype="f32")
    c = _gpu_batch(jt, bw)
    for _ in range(3):
        assert np.array_equal(c, _gpu_batch(jt, bw))


def test_second_device_in_one_process(jt, orc):
    """The per-kernel shared-memory attribute (cudaFuncSetAttribute) belongs to a device: the library remembers it per
    device, so the first call on a SECOND device of the same process works too (every kernel here needs > 48 KB)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two visible GPUs")
    w = workloads.config_c1()
    want = orc.simulate_image(w)
    bw = workloads.config_c3(B=8, dtype="f32")
    want_b = orc.simulate_batch(bw)
    for dev in (0, 1):
        with torch.cuda.device(dev):                   # "cuda" in to_dev() now means this device
            for method in ("direct", "fft"):
                assert rel_err(gpu_simulate(jt, w, method=method), want) < TOL_IMG["f64"], (dev, method)
            got_b = _gpu_batch(jt, bw)
            assert max(rel_err(got_b[b], want_b[b]) for b in range(bw.B)) < TOL_IMG["f32"], dev


def test_prepared_image_equals_simulate_image(jt):
    """binding.PreparedImage (marshalling done once, one ctypes call per image) returns bit for bit what simulate_image
    returns, call after call, and sees in-place updates of the subhalo tensor."""
    import torch
    for w in (workloads.config_c0(), workloads.config_c1(), workloads.config_c2(nx=48, n_tnfw=1500, dtype="f32")):
        g = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
        tn = to_dev(w.tnfw, w.dtype) if w.n_tnfw > 0 else None
        psf = to_dev(w.psf, w.dtype)
        want = jt.simulate_image(g, w.sie, w.shear, tn, w.sources, psf, dtype=w.dtype)
        prep = jt.PreparedImage(g, w.sie, w.shear, tn, w.sources, psf, dtype=w.dtype)
        for _ in range(3):
            assert torch.equal(prep(), want)
        if tn is not None:
            tn[3] *= 2.0                                   # alpha_Rs doubled in place
            want2 = jt.simulate_image(g, w.sie, w.shear, tn, w.sources, psf, dtype=w.dtype)
            assert torch.equal(prep(), want2) and not torch.equal(want2, want)
