"""Pins for the oracle of the SURVEY.md section 8(f) rows (oracle/oracle_next.c): chi^2 (NEXT-3), lensing Jacobian
(NEXT-2), further deflector and light profiles (NEXT-1).  Nothing here touches the CUDA path; every pin is a closed
form, an invariant, a library routine or brute force (mpmath / scipy quadrature)."""
import math

import numpy as np
import pytest
from scipy import integrate

from conftest import rel_err


# ------------------------------------------------------------------ NEXT-3: chi^2
def test_chi2_self_zero_sigma_shift_and_numpy(orc):
    """chi2(image, image) = 0; data + sigma in every pixel gives N; scaling sigma by c divides chi2 by c^2; numpy."""
    rng = np.random.default_rng(3)
    data = rng.uniform(1, 5, (17, 23))
    sigma = rng.uniform(0.1, 0.4, (17, 23))
    models = np.stack([data, data + sigma, data - 2 * sigma, rng.uniform(1, 5, (17, 23))])
    got = orc.chi2_batch(models, data, sigma)
    assert got[0] == 0.0
    assert abs(got[1] - data.size) < 1e-10 * data.size and abs(got[2] - 4 * data.size) < 1e-10 * data.size
    want = (((models[3] - data) / sigma) ** 2).sum()
    assert abs(got[3] - want) < 1e-12 * want
    assert abs(orc.chi2_batch(models[3:], data, 3.0 * sigma)[0] - want / 9.0) < 1e-12 * want


# ------------------------------------------------------------------ NEXT-2: Jacobian
def _fd_maps(orc, x, y, sie, shear, tnfw, h=1e-6):
    """kappa, gamma1, gamma2 from central differences of the (already pinned) lens equation: A = d beta / d theta."""
    bxp, byp = orc.ray_shoot(x + h, y, sie, shear, tnfw)
    bxm, bym = orc.ray_shoot(x - h, y, sie, shear, tnfw)
    cxp, cyp = orc.ray_shoot(x, y + h, sie, shear, tnfw)
    cxm, cym = orc.ray_shoot(x, y - h, sie, shear, tnfw)
    a11, a21 = (bxp - bxm) / (2 * h), (byp - bym) / (2 * h)
    a12, a22 = (cxp - cxm) / (2 * h), (cyp - cym) / (2 * h)
    assert np.max(np.abs(a12 - a21)) < 1e-7                      # curl alpha = 0
    return 1.0 - 0.5 * (a11 + a22), 0.5 * (a22 - a11), -0.5 * (a12 + a21), 1.0 / (a11 * a22 - a12 * a21)


def test_lensing_maps_against_finite_differences(orc):
    """Analytic kappa / gamma / mu of SIE + shear + TNFW = central differences of the lens equation, at five SIE
    ellipticities and for subhalos of tau = 0.5 ... 20 probed from X = 0.05 to 50."""
    rng = np.random.default_rng(11)
    tn = np.array([[0.6, -0.4, 0.1, 0.9], [0.3, 0.5, -0.8, -0.2], [0.05, 0.02, 0.2, 0.1], [0.01, 0.003, 0.1, 0.02],
                   [0.025, 0.02, 4.0, 0.1]])               # tau = 0.5, 1, 20, 1
    for e1, e2 in ((0.1, -0.05), (0.0, 0.0), (-0.2, 0.2), (0.3, 0.1), (1e-9, 0.0)):
        sie, shear = (1.3, e1, e2, 0.02, -0.01), (0.03, 0.01)
        x, y = rng.uniform(-1.8, 1.8, 300), rng.uniform(-1.8, 1.8, 300)
        keep = np.hypot(x - sie[3], y - sie[4]) > 0.15
        for j in range(tn.shape[1]):
            keep &= np.hypot(x - tn[0, j], y - tn[1, j]) > 0.02
        x, y = x[keep], y[keep]
        k, g1, g2, mu = orc.lensing_maps(x, y, sie, shear, tn)
        fk, fg1, fg2, fmu = _fd_maps(orc, x, y, sie, shear, tn)
        assert np.max(np.abs(k - fk)) < 2e-7 and np.max(np.abs(g1 - fg1)) < 2e-7 and np.max(np.abs(g2 - fg2)) < 2e-7
        ok = np.abs(fmu) < 50
        assert np.max(np.abs(mu[ok] / fmu[ok] - 1.0)) < 1e-4
    # one subhalo alone, rays placed at chosen X
    for tau in (0.5, 1.0, 5.0, 20.0):
        one = np.array([[0.0], [0.0], [0.1], [0.05], [0.1 * tau]])
        X = np.array([0.05, 0.5, 0.999, 1.001, 2.0, 7.0, 50.0])
        ang = rng.uniform(0, 2 * np.pi, X.size)
        x, y = 0.1 * X * np.cos(ang), 0.1 * X * np.sin(ang)
        k, g1, g2, _ = orc.lensing_maps(x, y, None, None, one)
        fk, fg1, fg2, _ = _fd_maps(orc, x, y, None, None, one, h=1e-7)
        assert np.max(np.abs(k - fk)) < 5e-6 * np.max(np.abs(k)) + 1e-8
        assert np.max(np.abs(g1 - fg1)) < 5e-6 * np.max(np.abs(g1)) + 1e-8
        assert np.max(np.abs(g2 - fg2)) < 5e-6 * np.max(np.abs(g2)) + 1e-8


def test_lensing_maps_closed_forms(orc):
    """SIS: kappa = theta_E / (2 r) = |gamma|, gamma tangential, mu = r / (r - theta_E).  Shear alone: kappa = 0,
    gamma = (g1, g2), mu = 1 / (1 - g^2).  Far from a TNFW (R >> r_trunc): point mass, kappa -> 0, |gamma| -> alpha / R."""
    rng = np.random.default_rng(5)
    x, y = rng.uniform(-2, 2, 200), rng.uniform(-2, 2, 200)
    r = np.hypot(x, y)
    tE = 1.1
    k, g1, g2, mu = orc.lensing_maps(x, y, (tE, 0.0, 0.0, 0.0, 0.0), None, None)
    assert np.max(np.abs(k - tE / (2 * r))) < 1e-14 * np.max(k)
    assert np.max(np.abs(np.hypot(g1, g2) - k)) < 1e-13 * np.max(k)
    assert np.max(np.abs(g1 + k * (x * x - y * y) / r ** 2)) < 1e-13 * np.max(k)      # tangential: -kappa cos 2phi
    far = np.abs(r - tE) > 0.05
    assert np.max(np.abs(mu[far] / (r[far] / (r[far] - tE)) - 1.0)) < 1e-11
    k, g1, g2, mu = orc.lensing_maps(x, y, None, (0.04, -0.03), None)
    assert np.all(k == 0.0) and np.all(g1 == 0.04) and np.all(g2 == -0.03)
    assert np.max(np.abs(mu - 1.0 / (1.0 - 0.04 ** 2 - 0.03 ** 2))) < 1e-15
    one = np.array([[0.0], [0.0], [0.01], [0.002], [0.05]])
    xf, yf = 40.0 * np.cos(np.linspace(0.1, 6, 7)), 40.0 * np.sin(np.linspace(0.1, 6, 7))     # X = 4000, 800 r_trunc
    k, g1, g2, _ = orc.lensing_maps(xf, yf, None, None, one)
    bx, by = orc.ray_shoot(xf, yf, None, None, one)
    a = np.hypot(xf - bx, yf - by)
    assert np.max(np.abs(k)) < 1e-6 * np.max(np.hypot(g1, g2))
    assert np.max(np.abs(np.hypot(g1, g2) / (a / 40.0) - 1.0)) < 1e-6


# ------------------------------------------------------------------ NEXT-1: deflectors
PROFILES = [("CONVERGENCE", [0.07, 0.1, -0.2]), ("SIS", [1.2, 0.05, -0.1]), ("NFW", [0.3, 0.15, -0.1, 0.2]),
            ("HERNQUIST", [0.4, 0.8, 0.1, 0.0]), ("PJAFFE", [0.9, 0.05, 0.6, -0.1, 0.1])]


@pytest.mark.parametrize("name,p", PROFILES)
def test_profile_divergence_curl_and_gauss_law(orc, name, p):
    """div alpha = 2 kappa, curl alpha = 0 (central differences) and, for the axisymmetric profiles, the Gauss-law
    integral alpha(R) R = 2 int_0^R kappa R' dR' by scipy quadrature of the oracle's own kappa."""
    rng = np.random.default_rng(len(name))
    cx, cy = (p[1], p[2]) if name in ("CONVERGENCE", "SIS") else (p[-2], p[-1])
    h = 1e-6
    for _ in range(40):
        ang, R = rng.uniform(0, 2 * np.pi), np.exp(rng.uniform(np.log(0.03), np.log(3.0)))
        x, y = cx + R * np.cos(ang), cy + R * np.sin(ang)
        axp, ayp = orc.profile_alpha(name, p, x + h, y)
        axm, aym = orc.profile_alpha(name, p, x - h, y)
        bxp, byp = orc.profile_alpha(name, p, x, y + h)
        bxm, bym = orc.profile_alpha(name, p, x, y - h)
        div = (axp - axm) / (2 * h) + (byp - bym) / (2 * h)
        curl = (ayp - aym) / (2 * h) - (bxp - bxm) / (2 * h)
        kap = orc.profile_kappa(name, p, x, y)
        assert abs(div - 2 * kap) < 3e-8 * max(1.0, abs(kap)) and abs(curl) < 3e-8 * max(1.0, abs(kap))
    if name != "CONVERGENCE":
        for R in (0.05, 0.3999, 0.4001, 1.7):
            ax, ay = orc.profile_alpha(name, p, cx + R, cy)
            m, _ = integrate.quad(lambda r: 2.0 * orc.profile_kappa(name, p, cx + r, cy) * r, 0.0, R, epsabs=1e-13, epsrel=1e-12,
                                  points=[min(R, p[0])] if name in ("NFW", "HERNQUIST") and p[0] < R else None, limit=400)
            assert abs(ax * R - m) < 2e-9 * abs(m) and abs(ay) < 1e-15
    assert orc.profile_alpha(name, p, cx, cy) == (0.0, 0.0)


def test_profile_closed_forms_and_limits(orc):
    """CONVERGENCE: alpha = kappa (theta - c).  SIS = SIE with e = 0.  NFW = TNFW with tau = 1e6.  NFW
    alpha(Rs) = alpha_Rs (the meaning of the parameter, reading Q7).  Hernquist and NFW convergence against the
    line-of-sight projection of their 3-D densities (mpmath quadrature), including X = 1 +- 1e-6 where the closed
    forms cancel.  PJAFFE: total mass pi alpha R -> 2 pi sigma0 Ra Rs at large R."""
    import mpmath as mp
    assert orc.profile_alpha("CONVERGENCE", [0.07, 0.1, -0.2], 0.6, 0.3) == pytest.approx((0.07 * 0.5, 0.07 * 0.5), rel=1e-15)
    a1 = orc.profile_alpha("SIS", [1.2, 0.05, -0.1], 0.7, 0.4)
    a2 = orc.profile_alpha("SIE", [1.2, 0.0, 0.0, 0.05, -0.1], 0.7, 0.4)
    assert a1 == pytest.approx(a2, rel=1e-14)
    Rs, aRs = 0.3, 0.15
    for X in (0.01, 0.5, 1.0, 3.0, 40.0):
        n = orc.profile_alpha("NFW", [Rs, aRs, 0.0, 0.0], X * Rs, 0.0)[0]
        t = orc.profile_alpha("TNFW", [Rs, aRs, 1e6 * Rs, 0.0, 0.0], X * Rs, 0.0)[0]
        assert abs(n / t - 1.0) < 1e-10 + 3e-12 * X * X      # the truncated halo misses ~ (X / tau)^2 of the mass at large X
    assert abs(orc.profile_alpha("NFW", [Rs, aRs, 0.0, 0.0], Rs, 0.0)[0] - aRs) < 1e-15
    mp.mp.dps = 30
    for name, rho in (("HERNQUIST", lambda x: 1 / (x * (1 + x) ** 3)), ("NFW", lambda x: 1 / (x * (1 + x) ** 2))):
        for X in (0.05, 0.5, 1 - 1e-6, 1.0, 1 + 1e-6, 1.02, 2.0, 30.0):
            sig = 2 * mp.quad(lambda z: rho(mp.sqrt(mp.mpf(X) ** 2 + z * z)), [0, 1, 10, mp.inf])       # rho0 = Rs = 1
            if name == "HERNQUIST":
                got = orc.profile_kappa(name, [1.0, 1.0, 0.0, 0.0], X, 0.0)                             # sigma0 = rho0 Rs = 1
            else:
                got = orc.profile_kappa(name, [1.0, 4.0 * (1 - math.log(2)), 0.0, 0.0], X, 0.0)         # 4 rho0 Rs^2 = aRs/(1-ln2)
            assert abs(got / float(sig) - 1.0) < 1e-11, (name, X)
    s0, Ra, Rsj = 0.9, 0.05, 0.6
    R = 1e5
    assert abs(orc.profile_alpha("PJAFFE", [s0, Ra, Rsj, 0.0, 0.0], R, 0.0)[0] * R / (2 * s0 * Ra * Rsj) - 1.0) < 1e-5


def test_ray_shoot_profiles_is_sum_of_parts(orc):
    rng = np.random.default_rng(2)
    defl = PROFILES + [("SIE", [1.0, 0.1, -0.05, 0.0, 0.0]), ("SHEAR", [0.03, 0.01]), ("TNFW", [0.2, 0.1, 1.0, 0.8, 0.3])]
    x, y = rng.uniform(-2, 2, 50), rng.uniform(-2, 2, 50)
    bx, by = orc.ray_shoot_profiles(x, y, defl)
    for i in range(50):
        sx = sum(orc.profile_alpha(n, p, x[i], y[i])[0] for n, p in defl)
        sy = sum(orc.profile_alpha(n, p, x[i], y[i])[1] for n, p in defl)
        assert abs(bx[i] - (x[i] - sx)) < 1e-14 and abs(by[i] - (y[i] - sy)) < 1e-14
    # the typed list restricted to the hot path's profiles = the hot path's oracle
    tn = np.array([[0.8], [0.3], [0.2], [0.1], [1.0]])
    wx, wy = orc.ray_shoot(x, y, (1.0, 0.1, -0.05, 0.0, 0.0), (0.03, 0.01), tn)
    hx, hy = orc.ray_shoot_profiles(x, y, defl[5:])
    assert np.max(np.abs(wx - hx)) < 1e-15 and np.max(np.abs(wy - hy)) < 1e-15


# ------------------------------------------------------------------ NEXT-1: light
def test_gaussian_light_flux_centre_and_half_light(orc):
    """amp is the total flux for any ellipticity (2-D quadrature); centre value amp / (2 pi sigma^2); half of the flux
    lies inside the elliptical radius sigma sqrt(2 ln 2); e = 0 is the circular Gaussian."""
    amp, sig = 3.0, 0.25
    for e1, e2 in ((0.0, 0.0), (0.3, -0.2)):
        p = [amp, sig, e1, e2, 0.1, -0.05]
        f = lambda r, t: orc.light("GAUSSIAN_ELLIPSE", p, 0.1 + r * math.cos(t), -0.05 + r * math.sin(t)) * r
        tot, _ = integrate.dblquad(f, 0, 2 * math.pi, 0, 12 * sig, epsabs=1e-12, epsrel=1e-11)
        assert abs(tot - amp) < 1e-8 * amp
        assert abs(orc.light("GAUSSIAN_ELLIPSE", p, 0.1, -0.05) - amp / (2 * math.pi * sig * sig)) < 1e-14
    r = 0.4
    want = amp / (2 * math.pi * sig * sig) * math.exp(-r * r / (2 * sig * sig))
    assert abs(orc.light("GAUSSIAN_ELLIPSE", [amp, sig, 0, 0, 0, 0], r * 0.6, r * 0.8) - want) < 1e-15 * want
    prof = lambda u: orc.light("GAUSSIAN_ELLIPSE", [amp, sig, 0, 0, 0, 0], u, 0.0) * 2 * math.pi * u
    inner, _ = integrate.quad(prof, 0, sig * math.sqrt(2 * math.log(2)), epsabs=1e-14)
    assert abs(inner / amp - 0.5) < 1e-12


def test_light_profiles_sum(orc):
    """MULTI_GAUSSIAN_ELLIPSE = the sum of its Gaussians; mixed lists add Sersic and Gaussian components; the typed
    list restricted to Sersic components = the hot path's oracle."""
    rng = np.random.default_rng(8)
    bx, by = rng.uniform(-1, 1, 40), rng.uniform(-1, 1, 40)
    mg = [("GAUSSIAN_ELLIPSE", [a, s, 0.2, -0.1, 0.05, 0.0]) for a, s in zip((1.0, 2.0, 0.5, 0.3, 1.2), (0.05, 0.1, 0.2, 0.4, 0.8))]
    ser = [("SERSIC_ELLIPSE", [10.0, 0.2, 1.5, 0.05, 0.02, 0.05, 0.0])]
    got = orc.light_profiles(bx, by, mg + ser)
    for i in range(40):
        want = sum(orc.light(n, p, bx[i], by[i]) for n, p in mg + ser)
        assert abs(got[i] - want) < 1e-13 * abs(want)
    assert rel_err(orc.light_profiles(bx, by, ser), orc.source_brightness(bx, by, [ser[0][1]])) < 1e-15
