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


# ------------------------------------------------------------------ step 1: jt_ray_shoot
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("n,M", [(1, 0), (5000, 0), (4097, 1), (3001, 700), (20000, 513)])
def test_ray_shoot_random(jt, orc, dtype, n, M):
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
                                         (200, 200, 21, 21), (33, 31, 1, 1)])
def test_convolve_direct(jt, orc, dtype, ny, nx, ky, kx):
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
    _check_image(jt, orc, workloads.config_c0(dtype=dtype), method="direct")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config_c1(jt, orc, dtype):
    _check_image(jt, orc, workloads.config_c1(dtype=dtype), method="direct")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config_c2_reduced(jt, orc, dtype):
    """C2's recipe at 48x48 pixels and 1,500 subhalos: several subhalo tiles plus a ragged tail, split list."""
    _check_image(jt, orc, workloads.config_c2(nx=48, n_tnfw=1500, dtype=dtype), method="direct")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config_c4_reduced(jt, orc, dtype):
    """C4's recipe (s=5, 3 sources, AiryMix PSF) at 30x30 pixels, 700 subhalos, K=41."""
    _check_image(jt, orc, workloads.config_c4(nx=30, n_tnfw=700, K=41, half_width=0.6, dtype=dtype), method="direct")


@pytest.mark.parametrize("s", [1, 2, 3, 4, 5, 6, 7, 8, 11, 16])
def test_supersampling_factors(jt, orc, s):
    """Every supported s: the warp-shuffle binning (definition B) with ragged tiles, off-centre, non-square grid."""
    w = workloads.config_c1(nx=23, supersample=s, K=9)
    w.ny, w.cx, w.cy = 17, 0.013, -0.021
    _check_image(jt, orc, w, method="direct")


def test_no_lens_constant_source_invariant(jt):
    """No deflector, very wide n=1 source: image ~ c * pixel_scale^2 (pins G/B independently of the oracle)."""
    g = jt.Grid(16, 12, 0.05, supersample=3)
    src = np.array([[2.0, 1e6, 1.0, 0.0, 0.0, 0.0, 0.0]])
    img = jt.simulate_image(g, None, None, None, src, None, dtype="f64").cpu().numpy()
    b = 1.9992 - 0.3271
    assert np.allclose(img, 2.0 * np.exp(b) * 0.05 ** 2, rtol=1e-5)


def test_c2_full_size_sampled_rows(jt, orc):
    """Full-size C2 (200x200, s=2, 10,000 subhalos) in the launch configuration bench.py times:
    three pixel rows of the pre-PSF image against the oracle, f64 and f32."""
    for dtype in ("f64", "f32"):
        w = workloads.config_c2(dtype=dtype)
        got = gpu_simulate(jt, w, conv=False)
        scale = np.max(np.abs(got))
        for j in (0, 97, 163):
            want = orc.prepsf_rows(w, j, j + 1)[0]
            assert np.max(np.abs(got[j] - want)) < TOL_IMG[dtype] * scale, (dtype, j)
