"""GPU parity for the SURVEY.md section 8(f) rows (through the C ABI) against oracle/oracle_next.c:
NEXT-3 chi^2 (standalone and fused into the batch kernel), NEXT-2 lensing maps, NEXT-1 typed profile lists."""
import numpy as np
import pytest

import workloads
from conftest import rel_err, to_dev

pytestmark = pytest.mark.gpu


def _f32r(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)


# ------------------------------------------------------------------ NEXT-3
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("B,ny,nx", [(1, 8, 8), (5, 100, 100), (64, 33, 47), (3, 257, 300)])
def test_chi2_batch(jt, orc, dtype, B, ny, nx):
    """jt_chi2_batch = the oracle's plain loop; includes image vs itself (0) and image + sigma (N pixels)."""
    rng = np.random.default_rng(B * 7 + nx)
    data = rng.uniform(1, 5, (ny, nx))
    sigma = rng.uniform(0.05, 0.3, (ny, nx))
    models = rng.uniform(1, 5, (B, ny, nx))
    models[0] = data
    if B > 1:
        models[1] = data + sigma
    if dtype == "f32":
        data, sigma, models = _f32r(data), _f32r(sigma), _f32r(models)
    got = jt.chi2_batch(to_dev(models, dtype), to_dev(data, dtype), to_dev(sigma, dtype)).cpu().numpy()
    want = orc.chi2_batch(models, data, sigma)
    assert got[0] == 0.0
    assert np.max(np.abs(got - want)) <= 1e-12 * np.max(want)         # double accumulation on both sides, different order
    if B > 1 and dtype == "f64":
        assert abs(got[1] - ny * nx) < 1e-9 * ny * nx


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("conv", [True, False])
def test_swarm_fused_chi2(jt, orc, dtype, conv):
    """jt_simulate_batch_chi2 on the swarm shape (100x100 grid, 13-pixel PSF): chi^2 of every particle =
    oracle chi^2 of the oracle's images; the images it optionally returns = jt_simulate_batch's; particle 0 (the truth)
    against data = truth + noise gives the noise's own chi^2."""
    w = workloads.config_swarm(B=12, dtype=dtype)
    truth = orc.simulate_batch(w, systems=[0])[0] if conv else None
    g = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
    d = lambda a: to_dev(a, dtype)
    psf = d(w.psf) if conv else None
    imgs = jt.simulate_batch(g, d(w.sie), d(w.shear), None, d(w.sources), psf)
    want_imgs = imgs.double().cpu().numpy()
    if not conv:
        truth = want_imgs[0]
    data = truth + w.data
    if dtype == "f32":
        data = _f32r(data)
    chi, got_imgs = jt.simulate_batch_chi2(g, d(w.sie), d(w.shear), None, d(w.sources), psf, d(data), d(w.sigma), images=True)
    assert np.array_equal(got_imgs.double().cpu().numpy(), want_imgs)
    only = jt.simulate_batch_chi2(g, d(w.sie), d(w.shear), None, d(w.sources), psf, d(data), d(w.sigma))
    assert np.array_equal(only.cpu().numpy(), chi.cpu().numpy())          # images not requested: same numbers
    # against the oracle end to end: its images, its chi^2
    orc_imgs = orc.simulate_batch(w) if conv else np.stack([orc.prepsf_rows(w.system(b)) for b in range(w.B)])
    want = orc.chi2_batch(orc_imgs, data, w.sigma)
    tol = 1e-8 if dtype == "f64" else 2e-2          # chi^2 amplifies image error by |residual| / sigma^2; float images carry ~1e-6
    assert np.max(np.abs(chi.cpu().numpy() - want) / np.maximum(want, 1.0)) < tol
    assert np.max(np.abs(chi.cpu().numpy() - orc.chi2_batch(want_imgs, data, w.sigma))) <= 1e-11 * np.max(want)
    noise_chi2 = float(np.sum((w.data / w.sigma) ** 2))
    assert abs(chi.cpu().numpy()[0] / noise_chi2 - 1.0) < (1e-6 if dtype == "f64" else 5e-3)


# ------------------------------------------------------------------ NEXT-2
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_lensing_maps(jt, orc, dtype):
    """kappa, gamma1, gamma2, mu of SIE + shear + 700 TNFW at 5000 points (incl. points at X = 1e-4 ... 30 around
    subhalo centres) against the oracle's analytic Jacobian."""
    rng = np.random.default_rng(31)
    M = 700
    tn = np.zeros((5, M))
    tn[0], tn[1] = rng.uniform(-1.5, 1.5, M), rng.uniform(-1.5, 1.5, M)
    tn[2] = np.exp(rng.uniform(np.log(0.005), np.log(0.05), M))
    tn[3] = np.exp(rng.uniform(np.log(1e-4), np.log(1e-2), M))
    tn[4] = tn[2] * np.exp(rng.uniform(np.log(0.5), np.log(20.0), M))
    x, y = rng.uniform(-1.5, 1.5, 5000), rng.uniform(-1.5, 1.5, 5000)
    Xs = np.logspace(-4, np.log10(30.0), 400)
    ang = rng.uniform(0, 2 * np.pi, 400)
    j = rng.integers(0, M, 400)
    x[:400] = tn[0, j] + Xs * tn[2, j] * np.cos(ang)
    y[:400] = tn[1, j] + Xs * tn[2, j] * np.sin(ang)
    sie, shear = (1.1, 0.15, -0.1, 0.02, 0.01), (0.03, -0.02)
    if dtype == "f32":
        x, y, tn = _f32r(x), _f32r(y), _f32r(tn)
        sie, shear = tuple(_f32r(sie)), tuple(_f32r(shear))
    got = [t.double().cpu().numpy() for t in jt.lensing_maps(to_dev(x, dtype), to_dev(y, dtype), sie, shear, to_dev(tn, dtype))]
    want = orc.lensing_maps(x, y, sie, shear, tn)
    # double: definition T's closed form loses digits just above the series switch (brace ~ X^2 ln X from terms of size
    # tau^2: relative error 3e-15 / (X^2 ln(2/X)) = 4e-10 at X = 1e-3) on BOTH sides independently; harmless for the
    # deflection alpha = f R, but the mean convergence alpha / R that enters gamma keeps it (reading Q25)
    tol = 5e-9 if dtype == "f64" else 3e-6
    for name, g_, w_ in zip(("kappa", "gamma1", "gamma2"), got[:3], want[:3]):
        assert np.max(np.abs(g_ - w_) / np.maximum(np.abs(w_), 1.0)) < tol, name
        assert np.max(np.abs(g_[400:] - w_[400:]) / np.maximum(np.abs(w_[400:]), 1.0)) < (1e-11 if dtype == "f64" else 3e-6), name
    ok = np.abs(want[3]) < 30
    assert np.max(np.abs(got[3][ok] / want[3][ok] - 1.0)) < (1e-8 if dtype == "f64" else 2e-3)
    # no subhalos, SIE only: |gamma| = kappa (closed form), through the kernel
    k, g1, g2, _ = [t.double().cpu().numpy() for t in jt.lensing_maps(to_dev(x, dtype), to_dev(y, dtype), sie, None, None)]
    assert np.max(np.abs(np.hypot(g1, g2) - k)) < (1e-13 if dtype == "f64" else 2e-6) * np.max(k)


# ------------------------------------------------------------------ NEXT-1
DEFLECTORS = [("CONVERGENCE", [0.07, 0.1, -0.2]), ("SIS", [1.2, 0.05, -0.1]), ("NFW", [0.3, 0.15, -0.1, 0.2]),
              ("HERNQUIST", [0.4, 0.8, 0.1, 0.0]), ("PJAFFE", [0.9, 0.05, 0.6, -0.1, 0.1]),
              ("SIE", [1.0, 0.1, -0.05, 0.0, 0.0]), ("SHEAR", [0.03, 0.01]), ("TNFW", [0.2, 0.1, 1.0, 0.8, 0.3])]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ray_shoot_profiles(jt, orc, dtype):
    """Every deflector type alone and all together (plus 150 NFW subhalos: three staging rounds of the list), rays incl.
    X = 1 +- 1e-7 of the NFW / Hernquist scale radii and a ray exactly on a centre."""
    rng = np.random.default_rng(41)
    x, y = rng.uniform(-2, 2, 3000), rng.uniform(-2, 2, 3000)
    x[:6] = [-0.1 + 0.3 * (1 + e) for e in (-1e-7, 0.0, 1e-7)] + [0.1 + 0.4 * (1 + e) for e in (-1e-7, 0.0, 1e-7)]
    y[:6] = [0.2, 0.2, 0.2, 0.0, 0.0, 0.0]
    x[6], y[6] = 0.05, -0.1                                          # on the SIS centre
    many = [("NFW", [float(r), float(a), float(cx), float(cy)]) for r, a, cx, cy in
            zip(np.exp(rng.uniform(np.log(0.005), np.log(0.05), 150)), np.exp(rng.uniform(np.log(1e-4), np.log(1e-2), 150)),
                rng.uniform(-2, 2, 150), rng.uniform(-2, 2, 150))]
    lists = [[d] for d in DEFLECTORS] + [DEFLECTORS + many]
    for defl in lists:
        xx, yy, dd = x, y, defl
        if dtype == "f32":
            xx, yy = _f32r(x), _f32r(y)
        bx, by = jt.ray_shoot_profiles(to_dev(xx, dtype), to_dev(yy, dtype), dd)
        wx, wy = orc.ray_shoot_profiles(xx, yy, dd)
        tol = 2e-13 if dtype == "f64" else 6e-7                      # float: storage of beta (|beta| up to ~3)
        assert np.max(np.abs(bx.double().cpu().numpy() - wx)) < tol * (1 + len(dd) / 50), dd[0][0]
        assert np.max(np.abs(by.double().cpu().numpy() - wy)) < tol * (1 + len(dd) / 50), dd[0][0]
    # the hot path's three profiles through the typed list = jt_ray_shoot
    tn = np.array([[0.8], [0.3], [0.2], [0.1], [1.0]])
    a = jt.ray_shoot(to_dev(x, "f64"), to_dev(y, "f64"), (1.0, 0.1, -0.05, 0.0, 0.0), (0.03, 0.01), to_dev(tn, "f64"))
    b = jt.ray_shoot_profiles(to_dev(x, "f64"), to_dev(y, "f64"), DEFLECTORS[5:])
    assert float((a[0] - b[0]).abs().max()) < 2e-13 and float((a[1] - b[1]).abs().max()) < 2e-13


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_light_profiles(jt, orc, dtype):
    """MULTI_GAUSSIAN_ELLIPSE (5 components) + a Sersic component, and 70 Gaussians (two staging rounds)."""
    rng = np.random.default_rng(43)
    bx, by = rng.uniform(-1, 1, 4000), rng.uniform(-1, 1, 4000)
    mg = [("GAUSSIAN_ELLIPSE", [a, s, 0.2, -0.1, 0.05, 0.0]) for a, s in zip((1.0, 2.0, 0.5, 0.3, 1.2), (0.05, 0.1, 0.2, 0.4, 0.8))]
    ser = [("SERSIC_ELLIPSE", [10.0, 0.2, 1.5, 0.05, 0.02, 0.05, 0.0])]
    lots = [("GAUSSIAN_ELLIPSE", [1.0, 0.1 + 0.01 * k, 0.0, 0.0, 0.02 * k - 0.7, 0.1]) for k in range(70)]
    if dtype == "f32":
        bx, by = _f32r(bx), _f32r(by)
    for comps in (mg, mg + ser, lots, ser):
        got = jt.light_profiles(to_dev(bx, dtype), to_dev(by, dtype), comps).double().cpu().numpy()
        want = orc.light_profiles(bx, by, comps)
        assert rel_err(got, want) < (1e-13 if dtype == "f64" else 2e-7)
    # Sersic through the typed list = jt_source_brightness
    a = jt.source_brightness(to_dev(bx, "f64"), to_dev(by, "f64"), [ser[0][1]])
    b = jt.light_profiles(to_dev(bx, "f64"), to_dev(by, "f64"), ser)
    assert float((a - b).abs().max()) < 1e-12 * float(a.abs().max())


def test_unknown_profile_types_contribute_nothing(jt):
    """include/jt.h: "Unknown types contribute nothing" -- a record of a type the library does not know (its parameters
    all zero, so a Gaussian reading of it would be 0/0) must leave the light sum and the deflection untouched."""
    import torch
    from paper_2606_01547_b200 import binding as b
    rng = np.random.default_rng(47)
    x, y = to_dev(rng.uniform(-1, 1, 3000), "f64"), to_dev(rng.uniform(-1, 1, 3000), "f64")
    ser = [("SERSIC_ELLIPSE", [10.0, 0.2, 1.5, 0.05, 0.02, 0.05, 0.0])]
    light = dict(b.LIGHT_TYPES, UNKNOWN=99, NEGATIVE=-3)
    recs = b.profile_records(ser + [("UNKNOWN", []), ("NEGATIVE", [])], light)
    assert torch.equal(jt.light_profiles(x, y, recs), jt.light_profiles(x, y, ser))
    sis = [("SIS", [1.0, 0.01, -0.02])]
    defl = dict(b.DEFLECTOR_TYPES, UNKNOWN=99)
    a = jt.ray_shoot_profiles(x, y, b.profile_records(sis + [("UNKNOWN", [])], defl))
    w = jt.ray_shoot_profiles(x, y, sis)
    assert torch.equal(a[0], w[0]) and torch.equal(a[1], w[1])


# ------------------------------------------------------------------ NEXT-1, second set
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ray_shoot_profiles_nie_epl(jt, orc, dtype):
    """NIE (readings Q31), EPL (Q32: the Tessore-Metcalf series, summed to the same tolerance on both sides) and
    MULTIPOLE (Q36; EPL + m = 3, 4 about one centre is the paper's EPL_MULTIPOLE row without its m = 1 term) in a typed
    list with members of the first set; includes s_scale = 0, gamma = 2, round lenses and a ray on a centre."""
    rng = np.random.default_rng(91)
    n = 3000
    tx, ty = rng.uniform(-2, 2, n), rng.uniform(-2, 2, n)
    tx[0], ty[0] = 0.3, -0.1                                   # on the centre of the first NIE
    defl = [("NIE", [1.1, 0.2, -0.1, 0.15, 0.3, -0.1]), ("NIE", [0.4, 0.0, 0.0, 0.05, -0.8, 0.6]),
            ("NIE", [0.7, -0.3, 0.25, 0.0, 1.2, 1.1]), ("EPL", [1.0, 2.0, 0.15, 0.1, -0.2, 0.3]),
            ("EPL", [0.8, 1.45, -0.35, 0.3, 0.9, -0.7]), ("EPL", [0.5, 2.7, 0.5, -0.2, -1.1, -1.2]),
            ("EPL", [0.6, 2.3, 0.0, 0.0, 0.1, 1.4]), ("SHEAR", [0.03, -0.02]), ("SIS", [0.2, 1.5, -1.5]),
            ("MULTIPOLE", [3.0, 0.04, 0.2, -0.2, 0.3]), ("MULTIPOLE", [4.0, -0.03, 1.1, -0.2, 0.3]),
            ("MULTIPOLE", [2.0, 0.02, -0.4, 0.3, -0.1]),                # centred on ray 0
            ("CSE", [0.05, 0.2, 0.3, -0.15, 0.5, 0.5]), ("CSE", [0.02, 0.05, 0.0, 0.0, -1.0, -0.4]),
            ("PJAFFE_ELLIPSE_POTENTIAL", [0.3, 0.1, 0.8, 0.25, -0.2, 0.9, 0.1])]
    if dtype == "f32":
        tx, ty = _f32r(tx), _f32r(ty)
    bx, by = jt.ray_shoot_profiles(to_dev(tx, dtype), to_dev(ty, dtype), defl)
    wx, wy = orc.ray_shoot_profiles(tx, ty, defl)
    tol = 2e-12 if dtype == "f64" else 6e-7
    assert np.max(np.abs(bx.double().cpu().numpy() - wx)) < tol
    assert np.max(np.abs(by.double().cpu().numpy() - wy)) < tol


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_light_core_sersic_and_shapelets(jt, orc, dtype):
    """CORE_SERSIC (Q33) and SHAPELETS (Q34) at n_max = 0, 6, 10 (the paper's two orders, 28 and 66 coefficients) and 12."""
    rng = np.random.default_rng(92)
    n = 5000
    bx, by = rng.uniform(-1.5, 1.5, n), rng.uniform(-1.5, 1.5, n)
    if dtype == "f32":
        bx, by = _f32r(bx), _f32r(by)
    p = [3.0, 0.4, 2.5, 0.05, 0.3, 2.0, 0.1, -0.2, 0.05, 0.02]
    got = jt.light_core_sersic(to_dev(bx, dtype), to_dev(by, dtype), p).double().cpu().numpy()
    want = orc.core_sersic(bx, by, *p)
    assert np.max(np.abs(got / want - 1.0)) < (1e-12 if dtype == "f64" else 2e-6)
    for n_max in (0, 6, 10, 12):
        coef = rng.normal(size=orc.shapelet_count(n_max))
        if dtype == "f32":
            coef = _f32r(coef)
        got = jt.light_shapelets(to_dev(bx, dtype), to_dev(by, dtype), n_max, 0.37, 0.1, -0.2, to_dev(coef, dtype)).double().cpu().numpy()
        want = orc.shapelets(bx, by, n_max, 0.37, 0.1, -0.2, coef)
        assert np.max(np.abs(got - want)) < (1e-12 if dtype == "f64" else 2e-6) * np.max(np.abs(want)), n_max


# ------------------------------------------------------------------ NEXT-4
@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("s,method", [(1, "direct"), (2, "direct"), (3, "fft"), (4, "auto")])
def test_simulate_image_supersampled_psf(jt, orc, dtype, s, method):
    """Convolution at ray resolution, then s x s binning = the oracle's composition (its ray image is the s = 1 pre-PSF
    image on the ray grid; PSF sampled on that grid, asymmetric on purpose)."""
    nx = 36
    w = workloads.config_c2(nx=nx, supersample=s, n_tnfw=300, K=9, dtype=dtype)
    rng = np.random.default_rng(93 + s)
    kf = rng.uniform(0, 1, (4 * s + 1, 2 * s + 3))
    kf /= kf.sum()
    if dtype == "f32":
        kf = _f32r(kf)
    fine = workloads.config_c2(nx=nx, supersample=s, n_tnfw=300, K=9, dtype=dtype)
    fine.nx, fine.ny, fine.pixel_scale, fine.supersample = nx * s, nx * s, w.pixel_scale / s, 1
    rays, _ = orc.simulate_image(fine)
    want = orc.convolve_supersampled(rays, s, kf)
    g = jt.Grid(w.nx, w.ny, w.pixel_scale, w.cx, w.cy, w.supersample)
    got = jt.simulate_image_supersampled_psf(g, w.sie, w.shear, to_dev(w.tnfw, dtype), w.sources, to_dev(kf, dtype), dtype=dtype,
                                             method=method).double().cpu().numpy()
    assert rel_err(got, want) < (1e-10 if dtype == "f64" else 2e-4)


def test_wrappers_on_a_side_stream(jt):
    """A caller-chosen stream that is not torch's current one: the binding uploads the profile records and allocates its
    outputs and scratch on THAT stream, so the result equals the default-stream result (no upload still in flight when
    the kernel starts, no temporary recycled under it).  Repeated, with allocator churn on the default stream between."""
    import torch
    rng = np.random.default_rng(53)
    x, y = to_dev(rng.uniform(-1, 1, 50000), "f64"), to_dev(rng.uniform(-1, 1, 50000), "f64")
    comps = [("GAUSSIAN_ELLIPSE", [1.0, 0.1 + 0.01 * k, 0.0, 0.0, 0.02 * k - 0.7, 0.1]) for k in range(70)]
    defl = [("SIS", [1.0, 0.01, -0.02]), ("NFW", [0.3, 0.2, -0.1, 0.1]), ("SHEAR", [0.03, -0.02])]
    tn = to_dev(np.array([[0.3], [0.2], [0.05], [0.01], [0.25]]) * np.ones((1, 3000)), "f64")
    want_l, want_d = jt.light_profiles(x, y, comps), jt.ray_shoot_profiles(x, y, defl)
    want_r = jt.ray_shoot(x[:2000], y[:2000], (1.0, 0.1, 0.0, 0.0, 0.0), None, tn)        # split list: scratch workspace
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    for _ in range(5):
        got_l = jt.light_profiles(x, y, comps, stream=side)
        got_d = jt.ray_shoot_profiles(x, y, defl, stream=side)
        got_r = jt.ray_shoot(x[:2000], y[:2000], (1.0, 0.1, 0.0, 0.0, 0.0), None, tn, stream=side)
        junk = [torch.full((50000,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(8)]   # default stream
        del junk
        side.synchronize()
        assert torch.equal(got_l, want_l)
        assert torch.equal(got_d[0], want_d[0]) and torch.equal(got_d[1], want_d[1])
        assert torch.equal(got_r[0], want_r[0]) and torch.equal(got_r[1], want_r[1])
