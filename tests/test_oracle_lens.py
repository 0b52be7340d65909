"""Pins for the oracle's deflectors (definitions E, S, H, T; SURVEY.md §8(c) pins table).

None of these re-type the oracle's formula: they are closed forms, invariants (div alpha =
2 kappa, curl alpha = 0), textbook limits and numerical line-of-sight projections of the 3-D
density (mpmath), chosen so a dropped term / wrong sign / swapped operand fails one of them.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")
LN2 = math.log(2.0)


def _read_table(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


def _div_curl(alpha, x, y, h=1e-5):
    axp, ayp = alpha(x + h, y)
    axm, aym = alpha(x - h, y)
    bxp, byp = alpha(x, y + h)
    bxm, bym = alpha(x, y - h)
    div = (axp - axm) / (2 * h) + (byp - bym) / (2 * h)
    curl = (ayp - aym) / (2 * h) - (bxp - bxm) / (2 * h)
    return div, curl


# ---------------------------------------------------------------- E
def test_ellipticity_golden(orc):
    for e1, e2, phi, q, tol in _read_table("ellipticity_c0.txt"):
        p, qq = orc.ellipticity(float(e1), float(e2))
        assert abs(p - float(phi)) < float(tol)
        assert abs(qq - float(q)) < float(tol)


def test_ellipticity_special_cases(orc):
    assert orc.ellipticity(0.0, 0.0) == (0.0, 1.0)
    phi, q = orc.ellipticity(0.5, 0.0)          # along x: phi = 0, q = (1-.5)/(1+.5)
    assert phi == 0.0 and abs(q - 1.0 / 3.0) < 1e-15
    phi, q = orc.ellipticity(0.0, 0.5)          # 45 degrees
    assert abs(phi - math.pi / 4) < 1e-15
    phi, q = orc.ellipticity(3.0, 4.0)          # clamp |e| at 0.9999
    assert abs(q - (1 - 0.9999) / (1 + 0.9999)) < 1e-15


# ---------------------------------------------------------------- S
def test_sis_constant_magnitude_radial(orc):
    """Circular SIE == SIS: |alpha| = theta_E, direction radial (north_star closed form)."""
    rng = np.random.default_rng(1)
    for _ in range(200):
        x, y = rng.uniform(-3, 3, size=2)
        cx, cy = rng.uniform(-0.5, 0.5, size=2)
        ax, ay = orc.sie_alpha(x, y, 1.3, 0.0, 0.0, cx, cy)
        r = math.hypot(x - cx, y - cy)
        assert abs(math.hypot(ax, ay) - 1.3) < 5e-15
        assert abs(ax - 1.3 * (x - cx) / r) < 5e-15 and abs(ay - 1.3 * (y - cy) / r) < 5e-15


def test_sie_q_to_one_continuity(orc):
    rng = np.random.default_rng(2)
    for _ in range(100):
        x, y = rng.uniform(-2, 2, size=2)
        a0 = orc.sie_alpha(x, y, 1.1, 0.0, 0.0)
        a1 = orc.sie_alpha(x, y, 1.1, 1e-9, 0.0)
        assert abs(a0[0] - a1[0]) < 2e-9 and abs(a0[1] - a1[1]) < 2e-9


@pytest.mark.parametrize("e1,e2", [(0.1, -0.05), (0.0, 0.0), (-0.2, 0.2), (0.3, 0.1), (1e-9, 0.0)])
def test_sie_div_equals_2kappa_curl_zero(orc, e1, e2):
    rng = np.random.default_rng(3)
    n = 0
    while n < 300:
        x, y = rng.uniform(-2.5, 2.5, size=2)
        if math.hypot(x - 0.1, y + 0.2) < 0.2:
            continue
        n += 1
        f = lambda a, b: orc.sie_alpha(a, b, 1.3, e1, e2, 0.1, -0.2)
        div, curl = _div_curl(f, x, y)
        kap = orc.sie_kappa(x, y, 1.3, e1, e2, 0.1, -0.2)
        assert abs(div - 2 * kap) < 1e-7 * kap
        assert abs(curl) < 1e-7


def test_sie_kappa_half_on_einstein_ellipse(orc):
    """Rays on q x'^2 + y'^2/q = theta_E^2 have kappa = 1/2 (theta_E = circularised Einstein radius)."""
    e1, e2, tE = 0.25, -0.1, 1.2
    phi, q = orc.ellipticity(e1, e2)
    for t in np.linspace(0, 2 * math.pi, 17):
        xr = tE / math.sqrt(q) * math.cos(t)
        yr = tE * math.sqrt(q) * math.sin(t)
        x = math.cos(phi) * xr - math.sin(phi) * yr
        y = math.sin(phi) * xr + math.cos(phi) * yr
        assert abs(orc.sie_kappa(x, y, tE, e1, e2) - 0.5) < 1e-14


def test_sie_antisymmetric_and_origin(orc):
    assert orc.sie_alpha(0.3, -0.1, 1.0, 0.2, 0.1, 0.3, -0.1) == (0.0, 0.0)
    a = orc.sie_alpha(0.7, 0.2, 1.0, 0.2, 0.1)
    b = orc.sie_alpha(-0.7, -0.2, 1.0, 0.2, 0.1)
    assert abs(a[0] + b[0]) < 1e-15 and abs(a[1] + b[1]) < 1e-15


def test_sie_deflection_from_mass_integral(orc):
    """alpha_r averaged on a circle = M(<r)/(pi r): Gauss's theorem in 2-D, for an ELLIPTICAL SIE.
    M(<r) is integrated numerically from the oracle's kappa (itself pinned by the kappa=1/2 ellipse)."""
    from scipy import integrate
    e1, e2, tE, r = 0.3, 0.1, 1.0, 0.8
    # flux of alpha through the circle
    ts = np.linspace(0, 2 * math.pi, 2001)[:-1]
    flux = 0.0
    for t in ts:
        ax, ay = orc.sie_alpha(r * math.cos(t), r * math.sin(t), tE, e1, e2)
        flux += (ax * math.cos(t) + ay * math.sin(t))
    flux *= r * (2 * math.pi / ts.size)
    # 2 * integral of kappa over the disc (kappa ~ 1/rho is integrable; polar coordinates remove it)
    f = lambda rho, t: 2 * orc.sie_kappa(rho * math.cos(t), rho * math.sin(t), tE, e1, e2) * rho
    mass2, _ = integrate.dblquad(f, 0, 2 * math.pi, 0, r, epsabs=1e-10, epsrel=1e-10)
    assert abs(flux - mass2) < 1e-8 * mass2


# ---------------------------------------------------------------- H
def test_shear_closed_form(orc):
    ax, ay = orc.shear_alpha(0.7, -0.3, 0.03, 0.01)
    assert abs(ax - (0.03 * 0.7 + 0.01 * -0.3)) < 1e-17
    assert abs(ay - (0.01 * 0.7 - 0.03 * -0.3)) < 1e-17
    f = lambda a, b: orc.shear_alpha(a, b, 0.03, 0.01)
    div, curl = _div_curl(f, 0.4, 0.9)
    assert abs(div) < 1e-10 and abs(curl) < 1e-10     # kappa = 0


def test_pointmass_closed_form(orc):
    ax, ay = orc.pointmass_alpha(0.6, 0.8, 1.5)
    assert abs(math.hypot(ax, ay) - 1.5 ** 2 / 1.0) < 1e-15
    assert abs(ax - 2.25 * 0.6) < 1e-15 and abs(ay - 2.25 * 0.8) < 1e-15


# ---------------------------------------------------------------- T
def _rho(r, Rs, rho0, tau):
    x = r / Rs
    return rho0 / (x * (1 + x) ** 2) * tau ** 2 / (tau ** 2 + x ** 2)


def _alpha_from_density(R, Rs, alpha_Rs, r_trunc):
    """alpha(R) = M_cyl(R)/(pi R) with Sigma_cr = 1; M_cyl from the 3-D density by 1-D quadrature:
    M_cyl(R) = int_0^R 4 pi r^2 rho dr + int_R^inf 4 pi r^2 rho (1 - sqrt(1 - R^2/r^2)) dr."""
    mp.mp.dps = 30
    Rs, R = mp.mpf(Rs), mp.mpf(R)
    tau = mp.mpf(r_trunc) / Rs
    rho0 = mp.mpf(alpha_Rs) / (4 * Rs ** 2 * (1 - mp.log(2)))
    inner = mp.quad(lambda r: 4 * mp.pi * r ** 2 * _rho(r, Rs, rho0, tau), [0, R / 2, R])
    outer = mp.quad(lambda r: 4 * mp.pi * r ** 2 * _rho(r, Rs, rho0, tau) * (1 - mp.sqrt(1 - (R / r) ** 2)),
                    [R, 2 * R, 10 * R + 10 * Rs * tau, mp.inf])
    return float((inner + outer) / (mp.pi * R))


@pytest.mark.parametrize("tau", [0.5, 1.0, 5.0, 20.0])
def test_tnfw_alpha_against_projected_density(orc, tau):
    Rs, aRs = 0.2, 0.1
    for X in (0.05, 0.5, 0.999, 1.001, 2.0, 7.0, 50.0):
        R = X * Rs
        want = _alpha_from_density(R, Rs, aRs, tau * Rs)
        ax, ay = orc.tnfw_alpha(0.3 + R * 0.6, -0.1 + R * 0.8, 0.3, -0.1, Rs, aRs, tau * Rs)
        got = math.hypot(ax, ay)
        assert abs(got - want) < 2e-10 * want, (tau, X, got, want)
        assert abs(ax / got - 0.6) < 1e-12 and abs(ay / got - 0.8) < 1e-12     # radial, outward


def test_tnfw_kappa_against_projected_density(orc):
    mp.mp.dps = 30
    Rs, aRs = 0.2, 0.1
    for tau in (0.5, 5.0):
        rho0 = mp.mpf(aRs) / (4 * mp.mpf(Rs) ** 2 * (1 - mp.log(2)))
        for X in (0.05, 0.5, 2.0, 7.0):
            R = mp.mpf(X) * Rs
            sig = 2 * mp.quad(lambda z: _rho(mp.sqrt(R * R + z * z), mp.mpf(Rs), rho0, mp.mpf(tau)),
                              [0, R, 10 * R + 10 * Rs * tau, mp.inf])
            got = orc.tnfw_kappa(float(R), 0.0, 0.0, 0.0, Rs, aRs, tau * Rs)
            assert abs(got - float(sig)) < 1e-9 * float(sig)


def test_tnfw_golden_values(orc):
    for X, g, tol in _read_table("tnfw_g_tau5.txt"):
        want, tol = float(g), float(tol)
        if X == "inf":
            tau = 5.0
            t = tau * tau
            closed = t / (t + 1) ** 2 * ((t - 1) * math.log(tau) + tau * math.pi - (t + 1))
            assert abs(closed - want) < tol * want                      # g_inf closed form == printed value
            got = orc.tnfw_g(1e7, 5.0)
            assert abs(got - want) < 1e-7 * want
        else:
            got = orc.tnfw_g(float(X), 5.0)
            assert abs(got - want) < tol * want, (X, got, want)


def test_tnfw_nfw_limit(orc):
    """tau -> inf: deflection at Rs equals alpha_Rs (Q7) and g -> ln(X/2) + F(X) (textbook NFW)."""
    ax, ay = orc.tnfw_alpha(0.2, 0.0, 0.0, 0.0, 0.2, 0.1, 0.2 * 1e6)
    assert abs(ax - 0.1) < 3e-11 * 0.1 * 10 and ay == 0.0
    for X in (0.2, 0.9, 1.0, 1.7, 12.0):
        if X < 1:
            F = math.acosh(1 / X) / math.sqrt(1 - X * X)
        elif X > 1:
            F = math.acos(1 / X) / math.sqrt(X * X - 1)
        else:
            F = 1.0
        assert abs(orc.tnfw_g(X, 1e6) - (math.log(X / 2) + F)) < 2e-9


def test_tnfw_total_mass_limit(orc):
    """R >> r_trunc: alpha R -> alpha_Rs Rs g_inf/(1-ln2); relative deficit ~ -8/X^2 at tau=5."""
    tau, Rs, aRs = 5.0, 0.02, 1e-3
    t = tau * tau
    ginf = t / (t + 1) ** 2 * ((t - 1) * math.log(tau) + tau * math.pi - (t + 1))
    for X, tol in ((1e3, 1e-6), (1e4, 1e-8)):
        ax, _ = orc.tnfw_alpha(X * Rs, 0.0, 0.0, 0.0, Rs, aRs, tau * Rs)
        rel = ax * X * Rs / (aRs * Rs * ginf / (1 - LN2)) - 1.0
        assert abs(rel + 8.0 / X ** 2) < tol


def test_tnfw_series_matches_closed_in_overlap(orc):
    for tau in (0.3, 1.0, 5.0, 30.0):
        for X in (1e-3, 2e-3, 5e-3):
            a, b = orc.tnfw_g_series(X, tau), orc.tnfw_g_closed(X, tau)
            assert abs(a - b) < (20 * X ** 4 + 1e-9) * abs(b)      # series truncation O(X^6)/X^2 + closed-form cancellation
        # the switch at X = 1e-3 is continuous to the closed form's own accuracy
        assert abs(orc.tnfw_g(0.999e-3, tau) / orc.tnfw_g(1.001e-3, tau) - (0.999 / 1.001) ** 2) < 1e-3


def test_tnfw_small_x_against_mpmath_closed_form(orc):
    """X < 1e-3 (series branch): compare with the closed form evaluated in 40-digit arithmetic."""
    mp.mp.dps = 40
    for tau in (0.5, 5.0):
        for X in (1e-5, 1e-4, 5e-4):
            Xm, tm = mp.mpf(X), mp.mpf(tau)
            t = tm * tm
            F = mp.acosh(1 / Xm) / mp.sqrt(1 - Xm * Xm)
            S = mp.sqrt(t + Xm * Xm)
            L = mp.log(Xm / (S + tm))
            brace = (t + 1 + 2 * (Xm * Xm - 1)) * F + tm * mp.pi + (t - 1) * mp.log(tm) + S * (-mp.pi + (t - 1) / tm * L)
            want = float(t / (t + 1) ** 2 * brace)
            assert abs(orc.tnfw_g(X, tau) - want) < 1e-6 * want


@pytest.mark.parametrize("tau", [0.5, 5.0, 20.0])
def test_tnfw_div_equals_2kappa_curl_zero(orc, tau):
    rng = np.random.default_rng(4)
    Rs, aRs = 0.2, 0.1
    for _ in range(200):
        X = math.exp(rng.uniform(math.log(0.05), math.log(30.0)))
        if abs(X - 1.0) < 1e-3:
            continue
        ang = rng.uniform(0, 2 * math.pi)
        x, y = 0.8 + X * Rs * math.cos(ang), 0.3 + X * Rs * math.sin(ang)
        f = lambda a, b: orc.tnfw_alpha(a, b, 0.8, 0.3, Rs, aRs, tau * Rs)
        div, curl = _div_curl(f, x, y, h=1e-5 * max(1.0, X) * Rs / 0.2)
        kap = orc.tnfw_kappa(x, y, 0.8, 0.3, Rs, aRs, tau * Rs)
        assert abs(div - 2 * kap) < 2e-6 * abs(kap) + 1e-9
        assert abs(curl) < 2e-7 * max(1.0, abs(kap))     # finite-difference noise floor


def test_tnfw_at_centre_and_x_equal_one(orc):
    assert orc.tnfw_alpha(0.8, 0.3, 0.8, 0.3, 0.2, 0.1, 1.0) == (0.0, 0.0)
    assert orc.tnfw_F(1.0) == 1.0
    # F is continuous through X = 1 (F = 1 - (2/3)(X-1) + ...)
    assert abs(orc.tnfw_F(1 - 1e-7) - 1.0) < 1e-6 and abs(orc.tnfw_F(1 + 1e-7) - 1.0) < 1e-6


def test_tnfw_F_against_mpmath_literal_definition(orc):
    """F(X) as literally defined (arccosh(1/X)/sqrt(1-X^2), arccos(1/X)/sqrt(X^2-1)) evaluated with 40 digits,
    on both sides of X = 1 down to the last representable neighbours, and over the whole range."""
    mp.mp.dps = 40
    xs = [1e-6, 1e-3, 0.03, 0.5, 0.9, 1.1, 2.0, 7.0, 50.0, 1e4]
    for k in range(3, 16):
        xs += [1.0 - 10.0 ** -k, 1.0 + 10.0 ** -k]
    xs += [np.nextafter(1.0, 0.0), np.nextafter(1.0, 2.0)]
    for X in xs:
        Xm = mp.mpf(float(X))
        want = mp.acosh(1 / Xm) / mp.sqrt(1 - Xm * Xm) if X < 1 else mp.acos(1 / Xm) / mp.sqrt(Xm * Xm - 1)
        assert abs(orc.tnfw_F(float(X)) / float(want) - 1.0) < 4e-15, X


# ---------------------------------------------------------------- lens equation
def test_lens_equation_closed_forms(orc):
    # no lens: beta = theta
    tx = np.array([0.3, -1.2, 0.0])
    ty = np.array([0.1, 0.4, -2.0])
    bx, by = orc.ray_shoot(tx, ty)
    assert np.array_equal(bx, tx) and np.array_equal(by, ty)
    # SIS: a point on the Einstein ring maps to beta = 0
    ang = np.linspace(0, 2 * math.pi, 13)
    bx, by = orc.ray_shoot(1.3 * np.cos(ang), 1.3 * np.sin(ang), sie=(1.3, 0, 0, 0, 0))
    assert np.max(np.abs(bx)) < 1e-15 and np.max(np.abs(by)) < 1e-15


def test_ray_shoot_is_sum_of_parts(orc):
    """beta = theta - alpha_SIE - alpha_shear - sum_j alpha_TNFW,j  (sign: Q2; single plane: Q23)."""
    rng = np.random.default_rng(5)
    M = 7
    tnfw = np.stack([rng.uniform(-1, 1, M), rng.uniform(-1, 1, M), rng.uniform(0.01, 0.2, M),
                     rng.uniform(1e-3, 1e-1, M), rng.uniform(0.1, 1.0, M)])
    sie = (1.1, 0.1, -0.2, 0.05, -0.02)
    shear = (0.04, -0.02)
    tx = rng.uniform(-2, 2, 20)
    ty = rng.uniform(-2, 2, 20)
    bx, by = orc.ray_shoot(tx, ty, sie, shear, tnfw)
    for i in range(20):
        ax, ay = orc.sie_alpha(tx[i], ty[i], *sie)
        sx, sy = orc.shear_alpha(tx[i], ty[i], *shear)
        ax += sx
        ay += sy
        for j in range(M):
            qx, qy = orc.tnfw_alpha(tx[i], ty[i], *tnfw[:, j])
            ax += qx
            ay += qy
        assert abs(bx[i] - (tx[i] - ax)) < 1e-14 and abs(by[i] - (ty[i] - ay)) < 1e-14
