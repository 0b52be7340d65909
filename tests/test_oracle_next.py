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


# ------------------------------------------------------------------ NEXT-1, second set: NIE, EPL, CORE_SERSIC, SHAPELETS
def _div_curl(orc, name, p, x, y, h=1e-6):
    axp, ayp = orc.profile_alpha(name, p, x + h, y)
    axm, aym = orc.profile_alpha(name, p, x - h, y)
    bxp, byp = orc.profile_alpha(name, p, x, y + h)
    bxm, bym = orc.profile_alpha(name, p, x, y - h)
    return ((axp - axm) + (byp - bym)) / (2 * h), ((ayp - aym) - (bxp - bxm)) / (2 * h)


def _brute_alpha(kappa, x, y, rmax=60.0):
    """alpha(theta) = (1/pi) int kappa(theta') (theta - theta')/|theta - theta'|^2 d^2 theta', polar about theta."""
    def fx(r, a):
        return kappa(x - r * math.cos(a), y - r * math.sin(a)) * math.cos(a)
    def fy(r, a):
        return kappa(x - r * math.cos(a), y - r * math.sin(a)) * math.sin(a)
    ix = integrate.dblquad(fx, 0, 2 * math.pi, 0, rmax, epsabs=1e-6, epsrel=1e-6)[0]
    iy = integrate.dblquad(fy, 0, 2 * math.pi, 0, rmax, epsabs=1e-6, epsrel=1e-6)[0]
    return ix / math.pi, iy / math.pi


def test_nie_reduces_to_sie_sphere_and_is_a_potential_flow(orc):
    """NIE (reading Q31): s_scale = 0 is definition S exactly; q = 1 is the cored isothermal sphere
    alpha = theta_E (sqrt(s^2 + r^2) - s)/r; div alpha = 2 kappa and curl alpha = 0 by central differences."""
    rng = np.random.default_rng(81)
    for e1, e2 in ((0.1, -0.05), (-0.3, 0.2), (0.0, 0.0), (1e-9, 0.0)):
        for _ in range(20):
            x, y = rng.uniform(-2, 2, 2)
            a = orc.profile_alpha("NIE", [1.2, e1, e2, 0.0, 0.05, -0.02], x, y)
            b = orc.sie_alpha(x, y, 1.2, e1, e2, 0.05, -0.02)
            assert abs(a[0] - b[0]) < 1e-14 and abs(a[1] - b[1]) < 1e-14
    for s in (0.01, 0.3, 2.0):
        for _ in range(10):
            x, y = rng.uniform(-2, 2, 2)
            ax, ay = orc.profile_alpha("NIE", [1.1, 0.0, 0.0, s, 0.0, 0.0], x, y)
            r = math.hypot(x, y)
            want = 1.1 * (math.sqrt(s * s + r * r) - s) / r
            assert abs(ax - want * x / r) < 1e-13 and abs(ay - want * y / r) < 1e-13
    for e1, e2, s in ((0.2, 0.1, 0.05), (-0.35, 0.3, 0.4), (0.5, -0.4, 0.01)):
        p = [1.3, e1, e2, s, 0.1, 0.05]
        for _ in range(30):
            x, y = rng.uniform(-2, 2, 2)
            div, curl = _div_curl(orc, "NIE", p, x, y)
            k = orc.profile_kappa("NIE", p, x, y)
            assert abs(div - 2 * k) < 2e-8 * max(1.0, k) and abs(curl) < 2e-8
    assert orc.profile_alpha("NIE", [1.0, 0.2, 0.1, 0.1, 0.3, 0.4], 0.3, 0.4) == (0.0, 0.0)      # centre of a cored lens


def test_nie_against_the_mass_integral(orc):
    """The NIE deflection from its OWN convergence by brute-force 2-D integration (independent of the closed form).
    kappa falls like 1/r, so the integral is cut at rmax and compared with the same cut of the closed form:
    the difference alpha(rmax1) - alpha(rmax2) of two cuts cancels the far field's (finite, direction-dependent) share."""
    p = [1.0, 0.25, -0.15, 0.2, 0.0, 0.0]
    kap = lambda u, v: orc.profile_kappa("NIE", p, u, v)
    for x, y in ((0.7, 0.2),):
        # the mass outside the disc of radius rmax around theta pulls with ~ theta_E |theta| / rmax: inside the tolerance
        ax, ay = _brute_alpha(kap, x, y, rmax=400.0)
        bx, by = orc.profile_alpha("NIE", p, x, y)
        assert abs(ax - bx) < 4e-3 and abs(ay - by) < 4e-3          # cut-off share ~ theta_E |theta| / rmax


def test_epl_reduces_to_sie_power_law_sphere_and_is_a_potential_flow(orc):
    """EPL (reading Q32): gamma = 2 is definition S; q = 1 is alpha = theta_E (theta_E/r)^(gamma-2) radially
    (mean convergence inside r of a power law); div alpha = 2 kappa, curl alpha = 0; steep and shallow slopes."""
    rng = np.random.default_rng(82)
    for e1, e2 in ((0.1, -0.05), (-0.3, 0.2), (0.45, 0.3)):
        for _ in range(20):
            x, y = rng.uniform(-2, 2, 2)
            a = orc.profile_alpha("EPL", [1.2, 2.0, e1, e2, 0.05, -0.02], x, y)
            b = orc.sie_alpha(x, y, 1.2, e1, e2, 0.05, -0.02)
            assert abs(a[0] - b[0]) < 1e-13 and abs(a[1] - b[1]) < 1e-13
    for gam in (1.4, 2.0, 2.6):
        for _ in range(10):
            x, y = rng.uniform(-2, 2, 2)
            ax, ay = orc.profile_alpha("EPL", [1.1, gam, 0.0, 0.0, 0.0, 0.0], x, y)
            r = math.hypot(x, y)
            want = 1.1 * (1.1 / r) ** (gam - 2.0)
            assert abs(ax - want * x / r) < 1e-13 and abs(ay - want * y / r) < 1e-13
    for gam, e1, e2 in ((1.5, 0.2, 0.1), (2.3, -0.35, 0.3), (2.7, 0.1, -0.4), (1.95, 0.6, 0.0)):
        p = [1.3, gam, e1, e2, 0.1, 0.05]
        for _ in range(30):
            x, y = rng.uniform(-2, 2, 2)
            if math.hypot(x - 0.1, y - 0.05) < 0.2:
                continue
            div, curl = _div_curl(orc, "EPL", p, x, y)
            k = orc.profile_kappa("EPL", p, x, y)
            assert abs(div - 2 * k) < 5e-8 * max(1.0, k) and abs(curl) < 5e-8


def test_epl_against_the_mass_integral_and_hyp2f1(orc):
    """Steep EPL (gamma = 2.6: kappa ~ r^-1.6 converges fast) against the brute-force 2-D mass integral, taken in polar
    coordinates about the LENS centre (the r^-1.6 cusp is then integrable by quadrature) and split at |theta| where the
    1/|theta - theta'| kernel peaks; and the series against mpmath's Gauss hypergeometric function, of which it is
    the Taylor expansion (Tessore & Metcalf 2015, eq. 13)."""
    import mpmath as mp
    p = [1.0, 2.6, 0.3, -0.2, 0.0, 0.0]
    x, y = 0.8, 0.3
    R0 = math.hypot(x, y)

    def fx(r, a):
        u, v = r * math.cos(a), r * math.sin(a)
        return orc.profile_kappa("EPL", p, u, v) * (x - u) / ((x - u) ** 2 + (y - v) ** 2) * r
    import warnings
    with warnings.catch_warnings():
        warnings.simplefilter("ignore")
        ix = sum(integrate.dblquad(fx, 0, 2 * math.pi, lo, hi, epsabs=1e-6, epsrel=1e-6)[0] for lo, hi in ((1e-9, R0), (R0, 3000.0)))
    bx, by = orc.profile_alpha("EPL", p, x, y)
    assert abs(ix / math.pi - bx) < 2e-5
    # hypergeometric form in the lens frame (no rotation: e2 = 0), several slopes and axis ratios
    for gam, e1 in ((1.3, 0.4), (2.0, -0.3), (2.8, 0.6)):
        _, q = orc.ellipticity(e1, 0.0)
        if e1 < 0:
            continue                                        # phi0 = pi/2 for e1 < 0: covered by the rotated cases above
        t, b = gam - 1.0, 1.2 * math.sqrt(q)
        for xx, yy in ((0.7, 0.4), (-1.1, 0.3), (0.2, -1.6)):
            R, phi = math.hypot(q * xx, yy), math.atan2(yy, q * xx)
            z = mp.e ** (1j * phi)
            want = 2 * b / (1 + q) * (b / R) ** (t - 1) * z * mp.hyp2f1(1, t / 2, 2 - t / 2, -(1 - q) / (1 + q) * z * z)
            ax, ay = orc.profile_alpha("EPL", [1.2, gam, e1, 0.0, 0.0, 0.0], xx, yy)
            assert abs(ax - float(want.real)) < 1e-13 and abs(ay - float(want.imag)) < 1e-13


def test_multipole_is_the_gradient_of_its_potential(orc):
    """MULTIPOLE (reading Q36), m = 2, 3, 4: alpha = grad psi by central differences of the potential; div alpha = 2 kappa
    with the closed-form kappa = a_m cos(m (phi - phi_m))/(2 r); curl alpha = 0; |alpha| does not depend on r;
    rotating the point by 2 pi / m leaves the radial component unchanged."""
    rng = np.random.default_rng(86)
    for m in (2, 3, 4):
        p = [float(m), 0.07, 0.3, 0.1, -0.05]
        for _ in range(25):
            x, y = rng.uniform(-2, 2, 2)
            if math.hypot(x - 0.1, y + 0.05) < 0.2:
                continue
            h = 1e-6
            gx = (orc.multipole_potential(x + h, y, *p) - orc.multipole_potential(x - h, y, *p)) / (2 * h)
            gy = (orc.multipole_potential(x, y + h, *p) - orc.multipole_potential(x, y - h, *p)) / (2 * h)
            ax, ay = orc.profile_alpha("MULTIPOLE", p, x, y)
            assert abs(ax - gx) < 1e-9 and abs(ay - gy) < 1e-9
            div, curl = _div_curl(orc, "MULTIPOLE", p, x, y)
            assert abs(div - 2 * orc.profile_kappa("MULTIPOLE", p, x, y)) < 2e-8 and abs(curl) < 2e-8
            a2 = orc.profile_alpha("MULTIPOLE", p, 0.1 + 3 * (x - 0.1), -0.05 + 3 * (y + 0.05))
            assert abs(a2[0] - ax) < 1e-14 and abs(a2[1] - ay) < 1e-14
    assert orc.profile_alpha("MULTIPOLE", [3.0, 0.05, 0.1, 0.2, 0.3], 0.2, 0.3) == (0.0, 0.0)


def test_cse_sphere_mass_integral_and_potential_flow(orc):
    """CSE (reading Q37): q = 1 is the cored steep sphere, alpha = A (1/s - 1/sqrt(s^2 + r^2))/r (enclosed mass of
    kappa = A/(2 (s^2 + r^2)^(3/2))); div alpha = 2 kappa and curl alpha = 0; the deflection from its OWN convergence by
    brute-force 2-D integration (kappa ~ r^-3: the cut at rmax = 200 leaves 1e-4 of the mass outside); total mass
    pi A q / s."""
    rng = np.random.default_rng(87)
    for s in (0.05, 0.4, 1.5):
        for _ in range(10):
            x, y = rng.uniform(-2, 2, 2)
            ax, ay = orc.profile_alpha("CSE", [0.8, s, 0.0, 0.0, 0.0, 0.0], x, y)
            r = math.hypot(x, y)
            want = 0.8 * (1.0 / s - 1.0 / math.sqrt(s * s + r * r)) / r
            assert abs(ax - want * x / r) < 1e-13 * max(1.0, want) and abs(ay - want * y / r) < 1e-13 * max(1.0, want)
    for e1, e2, s in ((0.2, 0.1, 0.3), (-0.35, 0.3, 0.1), (0.5, -0.3, 1.0)):
        p = [0.6, s, e1, e2, 0.1, 0.05]
        for _ in range(30):
            x, y = rng.uniform(-2, 2, 2)
            div, curl = _div_curl(orc, "CSE", p, x, y, h=1e-5)
            k = orc.profile_kappa("CSE", p, x, y)
            assert abs(div - 2 * k) < 1e-7 * max(1.0, k) and abs(curl) < 1e-7
    p = [0.6, 0.25, 0.3, -0.2, 0.0, 0.0]
    kap = lambda u, v: orc.profile_kappa("CSE", p, u, v)
    ax, ay = _brute_alpha(kap, 0.7, 0.2, rmax=200.0)
    bx, by = orc.profile_alpha("CSE", p, 0.7, 0.2)
    assert abs(ax - bx) < 2e-4 and abs(ay - by) < 2e-4
    _, q = orc.ellipticity(0.3, -0.2)
    far = orc.profile_alpha("CSE", p, 3000.0, 0.0)                    # a point mass of pi A q / s: alpha = M / (pi r)
    assert abs(far[0] * 3000.0 - 0.6 * q / 0.25) < 1e-3


def test_pjaffe_ellipse_potential(orc):
    """PJAFFE_ELLIPSE_POTENTIAL (reading Q38): e = 0 is PJAFFE exactly; alpha = grad psi by central differences of the
    elliptical potential (whose radial derivative is the already pinned PJAFFE deflection); div alpha = 2 kappa with
    the analytic Laplacian; curl alpha = 0."""
    rng = np.random.default_rng(88)
    for _ in range(20):
        x, y = rng.uniform(-2, 2, 2)
        a = orc.profile_alpha("PJAFFE_ELLIPSE_POTENTIAL", [0.7, 0.1, 0.9, 0.0, 0.0, 0.2, -0.1], x, y)
        b = orc.profile_alpha("PJAFFE", [0.7, 0.1, 0.9, 0.2, -0.1], x, y)
        assert abs(a[0] - b[0]) < 1e-14 and abs(a[1] - b[1]) < 1e-14
    for e1, e2 in ((0.2, 0.1), (-0.3, 0.25), (0.05, -0.4)):
        p = [0.7, 0.1, 0.9, e1, e2, 0.2, -0.1]
        for _ in range(25):
            x, y = rng.uniform(-2, 2, 2)
            h = 1e-6
            gx = (orc.pjaffe_ell_potential(x + h, y, *p) - orc.pjaffe_ell_potential(x - h, y, *p)) / (2 * h)
            gy = (orc.pjaffe_ell_potential(x, y + h, *p) - orc.pjaffe_ell_potential(x, y - h, *p)) / (2 * h)
            ax, ay = orc.profile_alpha("PJAFFE_ELLIPSE_POTENTIAL", p, x, y)
            assert abs(ax - gx) < 2e-9 and abs(ay - gy) < 2e-9
            div, curl = _div_curl(orc, "PJAFFE_ELLIPSE_POTENTIAL", p, x, y)
            k = orc.profile_kappa("PJAFFE_ELLIPSE_POTENTIAL", p, x, y)
            assert abs(div - 2 * k) < 5e-8 * max(1.0, abs(k)) and abs(curl) < 5e-8
    assert orc.profile_alpha("PJAFFE_ELLIPSE_POTENTIAL", [0.7, 0.1, 0.9, 0.2, 0.1, 0.2, -0.1], 0.2, -0.1) == (0.0, 0.0)


def test_core_sersic_limits(orc):
    """CORE_SERSIC (reading Q33): Rb -> 0 is definition R; far outside the break it tends to it; the inner logarithmic
    slope is -gamma; I on the R_sersic isophote for Rb = 0 is amp."""
    rng = np.random.default_rng(83)
    x, y = rng.uniform(-1, 1, 50), rng.uniform(-1, 1, 50)
    want = np.array([orc.sersic(a, b, 3.0, 0.4, 2.5, 0.1, -0.2, 0.05, 0.02) for a, b in zip(x, y)])
    got = orc.core_sersic(x, y, 3.0, 0.4, 2.5, 1e-12, 0.3, 2.0, 0.1, -0.2, 0.05, 0.02)
    assert np.max(np.abs(got / want - 1.0)) < 1e-9
    far = orc.core_sersic([3.0], [0.0], 3.0, 0.4, 1.0, 0.01, 0.2, 3.0, 0.0, 0.0, 0.0, 0.0)[0]
    assert abs(far / orc.sersic(3.0, 0.0, 3.0, 0.4, 1.0, 0.0, 0.0, 0.0, 0.0) - 1.0) < 1e-6
    r = np.array([1e-6, 2e-6])
    inner = orc.core_sersic(r, [0.0, 0.0], 1.0, 0.5, 3.0, 0.05, 0.35, 2.0, 0.0, 0.0, 0.0, 0.0)
    assert abs(math.log(inner[1] / inner[0]) / math.log(2.0) + 0.35) < 1e-4


def test_shapelets_orthonormal_gaussian_and_numpy(orc):
    """SHAPELETS (reading Q34): the n_max = 0 term is the Gaussian pi^(-1/2)/beta exp(-r^2/(2 beta^2)); single terms
    equal numpy's Hermite polynomials with the (2^n sqrt(pi) n!)^(-1/2) normalisation; the basis is orthonormal
    (Gauss-Hermite quadrature, exact for these polynomial degrees); the sum is linear in the coefficients."""
    from numpy.polynomial import hermite as H
    beta, cx, cy = 0.37, 0.1, -0.2
    rng = np.random.default_rng(84)
    x, y = rng.uniform(-1.5, 1.5, 40), rng.uniform(-1.5, 1.5, 40)
    g = orc.shapelets(x, y, 0, beta, cx, cy, [1.0])
    assert np.max(np.abs(g - np.exp(-((x - cx) ** 2 + (y - cy) ** 2) / (2 * beta * beta)) / (math.sqrt(math.pi) * beta))) < 1e-15
    n_max = 10
    nk = orc.shapelet_count(n_max)
    assert nk == 66 and orc.shapelet_count(6) == 28
    def b1(n, u):
        c = np.zeros(n + 1); c[n] = 1.0
        return H.hermval(u, c) * np.exp(-0.5 * u * u) / math.sqrt(2.0 ** n * math.sqrt(math.pi) * math.factorial(n))
    k = 0
    for N in range(n_max + 1):
        for n2 in range(N + 1):
            c = np.zeros(nk); c[k] = 1.0
            got = orc.shapelets(x, y, n_max, beta, cx, cy, c)
            want = b1(N - n2, (x - cx) / beta) * b1(n2, (y - cy) / beta) / beta
            assert np.max(np.abs(got - want)) < 1e-12, (N, n2)
            k += 1
    # orthonormality on a Gauss-Hermite grid (weight e^{-u^2}: B_n B_m = polynomial x e^{-u^2})
    u, wgt = H.hermgauss(40)
    U, V = np.meshgrid(u, u)
    W = np.outer(wgt, wgt) * np.exp(U * U + V * V)        # undo the weight: the integrand carries its own Gaussian
    pts_x, pts_y = cx + beta * U.ravel(), cy + beta * V.ravel()
    basis = []
    for kk in range(orc.shapelet_count(4)):
        c = np.zeros(orc.shapelet_count(4)); c[kk] = 1.0
        basis.append(orc.shapelets(pts_x, pts_y, 4, beta, cx, cy, c))
    basis = np.array(basis)
    gram = (basis * W.ravel()) @ basis.T * beta * beta
    assert np.max(np.abs(gram - np.eye(len(basis)))) < 1e-10
    c1, c2 = rng.normal(size=nk), rng.normal(size=nk)
    lin = orc.shapelets(x, y, n_max, beta, cx, cy, 2 * c1 - 3 * c2)
    assert np.max(np.abs(lin - (2 * orc.shapelets(x, y, n_max, beta, cx, cy, c1) - 3 * orc.shapelets(x, y, n_max, beta, cx, cy, c2)))) < 1e-12


# ------------------------------------------------------------------ NEXT-4: supersampled convolution
def test_convolve_supersampled_special_cases(orc):
    """s = 1 is definition P; a delta PSF on the ray grid gives plain binning (sum of the s x s rays); a PSF that is
    constant over s x s ray blocks and an image that is constant over pixels reduce to the pixel-resolution
    convolution with the block-summed kernel; flux is conserved away from the border; scipy on the fine grid."""
    from scipy.signal import convolve2d
    rng = np.random.default_rng(85)
    img = rng.uniform(0, 1, (12, 9))
    ker = rng.uniform(0, 1, (5, 3))
    assert np.max(np.abs(orc.convolve_supersampled(img, 1, ker) - orc.convolve(img, ker))) == 0.0
    s = 3
    rays = rng.uniform(0, 1, (12 * s, 9 * s))
    delta = np.zeros((3, 3)); delta[1, 1] = 1.0
    binned = rays.reshape(12, s, 9, s).sum(axis=(1, 3))
    assert np.max(np.abs(orc.convolve_supersampled(rays, s, delta) - binned)) < 1e-14
    kf = rng.uniform(0, 1, (7, 9))
    want = convolve2d(rays, kf, mode="same", boundary="fill").reshape(12, s, 9, s).sum(axis=(1, 3))
    assert np.max(np.abs(orc.convolve_supersampled(rays, s, kf) - want)) < 1e-12
    inner = np.zeros((12 * s, 9 * s)); inner[12:24, 9:18] = rays[12:24, 9:18]
    kf /= kf.sum()
    assert abs(orc.convolve_supersampled(inner, s, kf).sum() - inner.sum()) < 1e-12
