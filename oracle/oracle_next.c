/*
 * oracle_next.c -- oracle for the SURVEY.md section 8(f) "next" rows (compiled into liboracle.so beside oracle.c).
 *
 * TEST INFRASTRUCTURE ONLY (same rules as oracle.c: only tests/, smoke() and bench.py's cpu legs may use it; it shares
 * nothing with the CUDA path).  Plain double arithmetic in the order of the definitions.
 *
 *   NEXT-2  lensing Jacobian A = d beta / d theta = I - H, H_ij = d alpha_i / d theta_j of the hot path's deflectors
 *           (SIE, shear, TNFW):  kappa = (H_xx + H_yy)/2, gamma1 = (H_xx - H_yy)/2, gamma2 = H_xy,
 *           mu = 1 / ((1 - kappa)^2 - gamma1^2 - gamma2^2).  PAPER.md:35 and :135 obtain derivatives by automatic
 *           differentiation; here they are the analytic derivatives of definitions S, H, T (reading Q25).
 *   NEXT-1  further profiles of PAPER.md:63-87 (deflectors) and :95-108 (light): CONVERGENCE :65, HERNQUIST :71, NFW :81,
 *           PJAFFE :83, SIS :86, and GAUSSIAN :98 / GAUSSIAN_ELLIPSE :99 / MULTI_GAUSSIAN(_ELLIPSE) :100-101.  The paper
 *           prints names only; the formulas are the readings Q26-Q30 of DESIGN.md (standard lensing literature).
 *
 * Pins (tests/test_oracle_next.py): central differences of the already pinned deflections for every Hessian;
 * SIS closed forms (kappa = theta_E / 2r = |gamma|, mu = r / (r - theta_E)); div alpha = 2 kappa and the Gauss-law mass
 * integral alpha R = 2 int kappa R dR for every new deflector; projection of the 3-D Hernquist and NFW densities by
 * mpmath quadrature; NFW = TNFW at tau -> infinity; Gaussian total flux = amp, half-flux radius; multi-Gaussian = sum.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>

#define ORC_PI 3.14159265358979323846264338327950288

/* from oracle.c */
void orc_ellipticity(double e1, double e2, double *phi, double *q);
double orc_sie_kappa(double x, double y, const double *p);
double orc_tnfw_F(double X);
double orc_tnfw_kappa(double x, double y, double cx, double cy, double Rs, double alpha_Rs, double r_trunc);
void orc_tnfw_alpha(double x, double y, double cx, double cy, double Rs, double alpha_Rs, double r_trunc, double *ax, double *ay);
void orc_sie_alpha(double x, double y, const double *p, double *ax, double *ay);
void orc_shear_alpha(double x, double y, double g1, double g2, double *ax, double *ay);

/* ================================================================== NEXT-2: Hessians
 * Each routine ADDS its (kappa, gamma1, gamma2) to the running sums. */

/* SIE (definition S, core 0): the shear of a singular isothermal ellipsoid has the size of its convergence and points
 * along the position angle phi' of the ray in the lens frame (Kormann, Schneider & Bartelmann 1994):
 *   gamma1' = -kappa cos 2phi', gamma2' = -kappa sin 2phi';  back-rotation by the lens angle phi0 is a spin-2 rotation. */
static void sie_hessian(double x, double y, const double *p, double *k, double *g1, double *g2) {
    double phi0, q;
    orc_ellipticity(p[1], p[2], &phi0, &q);
    const double c = cos(phi0), s = sin(phi0);
    const double dx = x - p[3], dy = y - p[4];
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    const double r2 = xr * xr + yr * yr;
    if (r2 == 0.0) return;
    const double kap = orc_sie_kappa(x, y, p);
    const double c2 = (xr * xr - yr * yr) / r2, s2 = 2.0 * xr * yr / r2;          /* cos 2phi', sin 2phi' */
    const double g1r = -kap * c2, g2r = -kap * s2;
    const double C2 = cos(2.0 * phi0), S2 = sin(2.0 * phi0);
    *k += kap;
    *g1 += g1r * C2 - g2r * S2;
    *g2 += g1r * S2 + g2r * C2;
}

/* axisymmetric deflector about (cx, cy) with deflection a(R) and convergence kap(R): mean convergence inside R is a/R,
 * tangential shear gamma_t = a/R - kap, gamma1 = -gamma_t cos 2phi, gamma2 = -gamma_t sin 2phi. */
static void radial_hessian(double dx, double dy, double a, double kap, double *k, double *g1, double *g2) {
    const double R2 = dx * dx + dy * dy;
    if (R2 == 0.0) return;
    const double gt = a / sqrt(R2) - kap;
    *k += kap;
    *g1 += -gt * (dx * dx - dy * dy) / R2;
    *g2 += -gt * 2.0 * dx * dy / R2;
}

/* kappa, gamma1, gamma2 and magnification of SIE + shear + M TNFW at n points.
 * sie: 5 doubles or NULL; shear: 2 doubles or NULL; tnfw: [5][M] rows cx, cy, Rs, alpha_Rs, r_trunc. */
void orc_lensing_maps(int64_t n, const double *tx, const double *ty, const double *sie, const double *shear, int64_t M,
                      const double *tnfw, double *kappa, double *gamma1, double *gamma2, double *mu) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        const double x = tx[i], y = ty[i];
        double k = 0.0, g1 = 0.0, g2 = 0.0;
        if (sie) sie_hessian(x, y, sie, &k, &g1, &g2);
        if (shear) { g1 += shear[0]; g2 += shear[1]; }                    /* definition H: H_xx = g1, H_yy = -g1, H_xy = g2 */
        for (int64_t j = 0; j < M; ++j) {
            const double cx = tnfw[j], cy = tnfw[M + j], Rs = tnfw[2 * M + j], aRs = tnfw[3 * M + j], rt = tnfw[4 * M + j];
            double ax, ay;
            orc_tnfw_alpha(x, y, cx, cy, Rs, aRs, rt, &ax, &ay);
            const double a = sqrt(ax * ax + ay * ay);
            radial_hessian(x - cx, y - cy, a, orc_tnfw_kappa(x, y, cx, cy, Rs, aRs, rt), &k, &g1, &g2);
        }
        kappa[i] = k;
        gamma1[i] = g1;
        gamma2[i] = g2;
        mu[i] = 1.0 / ((1.0 - k) * (1.0 - k) - g1 * g1 - g2 * g2);
    }
}

/* ================================================================== NEXT-1: typed deflector list
 * A deflector is (type, p[8]).  Types and parameters (readings Q26-Q29):
 *   0 CONVERGENCE  p = {kappa, cx, cy}                 alpha = kappa (theta - c)                       (mass sheet)
 *   1 SIS          p = {theta_E, cx, cy}               alpha = theta_E (theta - c)/R
 *   2 NFW          p = {Rs, alpha_Rs, cx, cy}          alpha = alpha_Rs/(1 - ln 2) [ln(X/2) + F(X)]/X, X = R/Rs
 *   3 HERNQUIST    p = {Rs, sigma0, cx, cy}            rho = rho0/[x (1+x)^3], sigma0 = rho0 Rs:
 *                                                      kappa = sigma0 [(2 + X^2) F - 3]/(X^2 - 1)^2,
 *                                                      alpha = 2 sigma0 Rs X (1 - F)/(X^2 - 1)
 *   4 PJAFFE       p = {sigma0, Ra, Rs, cx, cy}        kappa = sigma0 Ra Rs/(Rs - Ra) [1/sqrt(Ra^2+R^2) - 1/sqrt(Rs^2+R^2)],
 *                                                      alpha = 2 sigma0 Ra Rs/(Rs - Ra) [f(Ra) - f(Rs)]/R,
 *                                                      f(a) = sqrt(a^2 + R^2) - a
 *   5 SIE          p = {theta_E, e1, e2, cx, cy}       definition S
 *   6 SHEAR        p = {gamma1, gamma2}                definition H
 *   7 TNFW         p = {Rs, alpha_Rs, r_trunc, cx, cy} definition T
 * X = 1 limits: F = 1, (1 - F)/(X^2 - 1) -> 1/3, [(2 + X^2) F - 3]/(X^2 - 1)^2 -> 4/15 (Taylor series for |X^2 - 1| < 0.05).
 * Every profile: alpha = 0 at R = 0. */
enum { ORC_CONVERGENCE = 0, ORC_SIS = 1, ORC_NFW = 2, ORC_HERNQUIST = 3, ORC_PJAFFE = 4, ORC_SIE = 5, ORC_SHEAR = 6, ORC_TNFW = 7 };

/* (1 - F(X))/(X^2 - 1) with u = X^2 - 1: the closed form cancels near X = 1 (1 - F ~ u/3), so for |u| < 0.05 the
 * Taylor series sum_k (-u)^k/(2k+3) is summed instead (12 terms: remainder < 1e-16); checked against 60-digit mpmath. */
static double one_minus_F_over(double X) {
    const double u = X * X - 1.0;
    if (fabs(u) < 0.05) {
        double acc = 0.0, pw = 1.0;
        for (int k = 0; k < 12; ++k) { acc += pw / (double)(2 * k + 3); pw *= -u; }
        return acc;
    }
    return (1.0 - orc_tnfw_F(X)) / u;
}
/* [(2 + X^2) F - 3]/(X^2 - 1)^2: cancels twice near X = 1; series sum_k (-u)^k 4(k+1)/((2k+3)(2k+5)) for |u| < 0.05 */
static double hernquist_shape(double X) {
    const double u = X * X - 1.0;
    if (fabs(u) < 0.05) {
        double acc = 0.0, pw = 1.0;
        for (int k = 0; k < 12; ++k) { acc += pw * 4.0 * (double)(k + 1) / (double)((2 * k + 3) * (2 * k + 5)); pw *= -u; }
        return acc;
    }
    return ((2.0 + X * X) * orc_tnfw_F(X) - 3.0) / (u * u);
}

void orc_profile_alpha(int type, const double *p, double x, double y, double *ax, double *ay) {
    *ax = 0.0;
    *ay = 0.0;
    if (type == ORC_SIE) { orc_sie_alpha(x, y, p, ax, ay); return; }
    if (type == ORC_SHEAR) { orc_shear_alpha(x, y, p[0], p[1], ax, ay); return; }
    if (type == ORC_TNFW) { orc_tnfw_alpha(x, y, p[3], p[4], p[0], p[1], p[2], ax, ay); return; }
    if (type == ORC_CONVERGENCE) { *ax = p[0] * (x - p[1]); *ay = p[0] * (y - p[2]); return; }
    double cx, cy;
    if (type == ORC_SIS) { cx = p[1]; cy = p[2]; }
    else if (type == ORC_PJAFFE) { cx = p[3]; cy = p[4]; }
    else { cx = p[2]; cy = p[3]; }
    const double dx = x - cx, dy = y - cy;
    const double R = sqrt(dx * dx + dy * dy);
    if (R == 0.0) return;
    double a = 0.0;
    if (type == ORC_SIS) {
        a = p[0];
    } else if (type == ORC_NFW) {
        const double X = R / p[0];
        a = p[1] / (1.0 - log(2.0)) * (log(0.5 * X) + orc_tnfw_F(X)) / X;
    } else if (type == ORC_HERNQUIST) {
        const double X = R / p[0];
        a = 2.0 * p[1] * p[0] * X * one_minus_F_over(X);
    } else if (type == ORC_PJAFFE) {
        const double Ra = p[1], Rs = p[2];
        a = 2.0 * p[0] * Ra * Rs / (Rs - Ra) * ((sqrt(Ra * Ra + R * R) - Ra) - (sqrt(Rs * Rs + R * R) - Rs)) / R;
    }
    *ax = a * dx / R;
    *ay = a * dy / R;
}

double orc_profile_kappa(int type, const double *p, double x, double y) {
    if (type == ORC_SIE) return orc_sie_kappa(x, y, p);
    if (type == ORC_SHEAR) return 0.0;
    if (type == ORC_TNFW) return orc_tnfw_kappa(x, y, p[3], p[4], p[0], p[1], p[2]);
    if (type == ORC_CONVERGENCE) return p[0];
    double cx, cy;
    if (type == ORC_SIS) { cx = p[1]; cy = p[2]; }
    else if (type == ORC_PJAFFE) { cx = p[3]; cy = p[4]; }
    else { cx = p[2]; cy = p[3]; }
    const double R = sqrt((x - cx) * (x - cx) + (y - cy) * (y - cy));
    if (type == ORC_SIS) return 0.5 * p[0] / R;
    if (type == ORC_NFW) return p[1] / ((1.0 - log(2.0)) * p[0]) * 0.5 * one_minus_F_over(R / p[0]);
    if (type == ORC_HERNQUIST) return p[1] * hernquist_shape(R / p[0]);
    if (type == ORC_PJAFFE) {
        const double Ra = p[1], Rs = p[2];
        return p[0] * Ra * Rs / (Rs - Ra) * (1.0 / sqrt(Ra * Ra + R * R) - 1.0 / sqrt(Rs * Rs + R * R));
    }
    return 0.0;
}

/* beta = theta - sum_d alpha_d(theta) over a typed list: types [n_def], params [n_def][8] */
void orc_ray_shoot_profiles(int64_t n, const double *tx, const double *ty, int64_t n_def, const int32_t *types,
                            const double *params, double *bx, double *by) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        double sx = 0.0, sy = 0.0;
        for (int64_t d = 0; d < n_def; ++d) {
            double ax, ay;
            orc_profile_alpha(types[d], params + 8 * d, tx[i], ty[i], &ax, &ay);
            sx += ax;
            sy += ay;
        }
        bx[i] = tx[i] - sx;
        by[i] = ty[i] - sy;
    }
}

/* ================================================================== NEXT-1: light profiles
 *   0 SERSIC_ELLIPSE    p = {amp, R_sersic, n_sersic, e1, e2, cx, cy}   definition R
 *   1 GAUSSIAN_ELLIPSE  p = {amp, sigma, e1, e2, cx, cy}   I = amp/(2 pi sigma^2) exp(-R^2/(2 sigma^2)),
 *                       R^2 = q x'^2 + y'^2/q (the product-averaged radius of definition R, so amp is the total flux for
 *                       any ellipticity); GAUSSIAN is e1 = e2 = 0; MULTI_GAUSSIAN(_ELLIPSE) (:100-101) is a
 *                       list of these sharing centre and ellipticity. */
double orc_sersic(double x, double y, const double *p);
enum { ORC_LIGHT_SERSIC = 0, ORC_LIGHT_GAUSSIAN = 1 };

double orc_light(int type, const double *p, double x, double y) {
    if (type == ORC_LIGHT_SERSIC) return orc_sersic(x, y, p);
    double phi, q;
    orc_ellipticity(p[2], p[3], &phi, &q);
    const double c = cos(phi), s = sin(phi);
    const double dx = x - p[4], dy = y - p[5];
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    const double R2 = q * xr * xr + yr * yr / q;
    return p[0] / (2.0 * ORC_PI * p[1] * p[1]) * exp(-R2 / (2.0 * p[1] * p[1]));
}

void orc_light_profiles(int64_t n, const double *bx, const double *by, int64_t n_comp, const int32_t *types,
                        const double *params, double *flux) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double acc = 0.0;
        for (int64_t k = 0; k < n_comp; ++k) acc += orc_light(types[k], params + 8 * k, bx[i], by[i]);
        flux[i] = acc;
    }
}

/* ================================================================== NEXT-1, second set (readings Q31-Q34 of DESIGN.md)
 *   8 NIE  ("NIE/SIE")   p = {theta_E, e1, e2, s_scale, cx, cy}
 *        kappa = (theta_E / 2) / sqrt(s^2 + q x'^2 + y'^2/q): definition S with a core; s_scale = 0 IS definition S.
 *        Deflection (Kormann et al. 1994, Keeton 2001), with b = theta_E / sqrt q, sk = s / sqrt q,
 *        psi = sqrt(q^2 (sk^2 + x'^2) + y'^2), f = sqrt(1 - q^2), A(z) = atan z / z, Bh(z) = atanh z / z:
 *          a'x = b q x'/(psi + sk) A(f x'/(psi + sk)),   a'y = b q y'/(psi + q^2 sk) Bh(f y'/(psi + q^2 sk))
 *        (regular at q = 1, where a = theta_E (sqrt(s^2 + r^2) - s) / r).
 *   9 EPL          p = {theta_E, gamma, e1, e2, cx, cy}
 *        kappa = (3 - gamma)/2 (theta_E / sqrt(q x'^2 + y'^2/q))^(gamma - 1), 1 < gamma < 3; gamma = 2 IS definition S.
 *        Deflection by the series of Tessore & Metcalf (2015, eq. 13 and 29): t = gamma - 1, b = theta_E sqrt q,
 *        R = sqrt(q^2 x'^2 + y'^2), phi = atan2(y', q x'), f = (1 - q)/(1 + q):
 *          a'x + i a'y = 2 b/(1 + q) (b/R)^(t-1) sum_n a_n,  a_0 = e^(i phi),
 *          a_n = -f (2n - (2 - t))/(2n + (2 - t)) e^(2 i phi) a_(n-1),  summed until |a_n| < 1e-17 |sum| (<= 400 terms).
 */
enum { ORC_NIE = 8, ORC_EPL = 9, ORC_MULTIPOLE = 10, ORC_CSE = 11, ORC_PJAFFE_ELL = 12 };

static double atan_over(double z) { return fabs(z) < 1e-4 ? 1.0 - z * z / 3.0 + z * z * z * z / 5.0 : atan(z) / z; }
static double atanh_over(double z) { return fabs(z) < 1e-4 ? 1.0 + z * z / 3.0 + z * z * z * z / 5.0 : atanh(z) / z; }

void orc_nie_alpha(double x, double y, const double *p, double *ax, double *ay) {
    double phi0, q;
    orc_ellipticity(p[1], p[2], &phi0, &q);
    const double c = cos(phi0), s = sin(phi0);
    const double dx = x - p[4], dy = y - p[5];
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    const double b = p[0] / sqrt(q), sk = p[3] / sqrt(q), f = sqrt(1.0 - q * q);
    const double psi = sqrt(q * q * (sk * sk + xr * xr) + yr * yr);
    *ax = 0.0;
    *ay = 0.0;
    if (psi + sk == 0.0) return;                                  /* the centre of a singular lens */
    const double ux = xr / (psi + sk), uy = yr / (psi + q * q * sk);
    const double axr = b * q * ux * atan_over(f * ux), ayr = b * q * uy * atanh_over(f * uy);
    *ax = c * axr - s * ayr;
    *ay = s * axr + c * ayr;
}
double orc_nie_kappa(double x, double y, const double *p) {
    double phi0, q;
    orc_ellipticity(p[1], p[2], &phi0, &q);
    const double c = cos(phi0), s = sin(phi0);
    const double dx = x - p[4], dy = y - p[5];
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    return 0.5 * p[0] / sqrt(p[3] * p[3] + q * xr * xr + yr * yr / q);
}

void orc_epl_alpha(double x, double y, const double *p, double *ax, double *ay) {
    double phi0, q;
    orc_ellipticity(p[2], p[3], &phi0, &q);
    const double c = cos(phi0), s = sin(phi0);
    const double dx = x - p[4], dy = y - p[5];
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    const double t = p[1] - 1.0, b = p[0] * sqrt(q);
    const double R = sqrt(q * q * xr * xr + yr * yr);
    *ax = 0.0;
    *ay = 0.0;
    if (R == 0.0) return;
    const double cph = q * xr / R, sph = yr / R;                  /* e^(i phi) */
    const double c2 = cph * cph - sph * sph, s2 = 2.0 * cph * sph;
    const double f = (1.0 - q) / (1.0 + q);
    double are = cph, aim = sph, sre = cph, sim = sph;
    for (int n = 1; n <= 400; ++n) {
        const double g = -f * (2.0 * n - (2.0 - t)) / (2.0 * n + (2.0 - t));
        const double nre = g * (c2 * are - s2 * aim), nim = g * (c2 * aim + s2 * are);
        are = nre;
        aim = nim;
        sre += are;
        sim += aim;
        if (are * are + aim * aim < 1e-34 * (sre * sre + sim * sim)) break;
    }
    const double pre = 2.0 * b / (1.0 + q) * pow(b / R, t - 1.0);
    const double axr = pre * sre, ayr = pre * sim;
    *ax = c * axr - s * ayr;
    *ay = s * axr + c * ayr;
}
double orc_epl_kappa(double x, double y, const double *p) {
    double phi0, q;
    orc_ellipticity(p[2], p[3], &phi0, &q);
    const double c = cos(phi0), s = sin(phi0);
    const double dx = x - p[4], dy = y - p[5];
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    return 0.5 * (3.0 - p[1]) * pow(p[0] / sqrt(q * xr * xr + yr * yr / q), p[1] - 1.0);
}

/*  10 MULTIPOLE  p = {m, a_m, phi_m, cx, cy}, integer m >= 2 (reading Q36): the potential
 *        psi = r a_m/(1 - m^2) cos(m (phi - phi_m)), whose Laplacian gives kappa = a_m cos(m (phi - phi_m))/(2 r);
 *        alpha_r = dpsi/dr = a_m/(1 - m^2) cos(m (phi - phi_m)), alpha_phi = (1/r) dpsi/dphi = -m a_m/(1 - m^2) sin(m (phi - phi_m)),
 *        (alpha_x, alpha_y) = (alpha_r cos phi - alpha_phi sin phi, alpha_r sin phi + alpha_phi cos phi); alpha(0) = 0. */
double orc_multipole_potential(double x, double y, const double *p) {
    const double dx = x - p[3], dy = y - p[4], m = p[0];
    return sqrt(dx * dx + dy * dy) * p[1] / (1.0 - m * m) * cos(m * (atan2(dy, dx) - p[2]));
}
void orc_multipole_alpha(double x, double y, const double *p, double *ax, double *ay) {
    const double dx = x - p[3], dy = y - p[4], m = p[0];
    *ax = 0.0;
    *ay = 0.0;
    if (dx == 0.0 && dy == 0.0) return;
    const double phi = atan2(dy, dx);
    const double ar = p[1] / (1.0 - m * m) * cos(m * (phi - p[2])), aphi = -m * p[1] / (1.0 - m * m) * sin(m * (phi - p[2]));
    *ax = ar * cos(phi) - aphi * sin(phi);
    *ay = ar * sin(phi) + aphi * cos(phi);
}
double orc_multipole_kappa(double x, double y, const double *p) {
    const double dx = x - p[3], dy = y - p[4];
    return 0.5 * p[1] * cos(p[0] * (atan2(dy, dx) - p[2])) / sqrt(dx * dx + dy * dy);
}

/*  11 CSE (cored steep ellipsoid; reading Q37)  p = {A, s, e1, e2, cx, cy}
 *        kappa = A / (2 (s^2 + x'^2 + y'^2/q^2)^(3/2))  (Oguri 2021: the major axis along x', NOT the product-averaged
 *        radius of definitions S and R), deflection in the lens frame with psi = sqrt(q^2 (s^2 + x'^2) + y'^2):
 *          a'x = A q x' (psi + q^2 s) / (s psi [(psi + s)^2 + (1 - q^2) x'^2]),
 *          a'y = A q y' (psi + s)     / (s psi [(psi + s)^2 + (1 - q^2) x'^2]). */
void orc_cse_alpha(double x, double y, const double *p, double *ax, double *ay) {
    double phi0, q;
    orc_ellipticity(p[2], p[3], &phi0, &q);
    const double c = cos(phi0), sn = sin(phi0), s = p[1];
    const double dx = x - p[4], dy = y - p[5];
    const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
    const double psi = sqrt(q * q * (s * s + xr * xr) + yr * yr);
    const double den = s * psi * ((psi + s) * (psi + s) + (1.0 - q * q) * xr * xr);
    const double axr = p[0] * q * xr * (psi + q * q * s) / den, ayr = p[0] * q * yr * (psi + s) / den;
    *ax = c * axr - sn * ayr;
    *ay = sn * axr + c * ayr;
}
double orc_cse_kappa(double x, double y, const double *p) {
    double phi0, q;
    orc_ellipticity(p[2], p[3], &phi0, &q);
    const double c = cos(phi0), sn = sin(phi0);
    const double dx = x - p[4], dy = y - p[5];
    const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
    return 0.5 * p[0] / pow(p[1] * p[1] + xr * xr + yr * yr / (q * q), 1.5);
}

/*  12 PJAFFE_ELLIPSE_POTENTIAL (reading Q38)  p = {sigma0, Ra, Rs, e1, e2, cx, cy}: the PJAFFE lensing
 *        POTENTIAL made elliptical, psi(x', y') = psi_PJ(Re), Re = sqrt(q x'^2 + y'^2/q) (the product-averaged radius of
 *        definitions S and R), psi_PJ(R) = C [f(Ra) - f(Rs)], f(a) = sqrt(a^2 + R^2) - a ln(a + sqrt(a^2 + R^2)),
 *        C = 2 sigma0 Ra Rs/(Rs - Ra), so that dpsi_PJ/dR is the PJAFFE deflection a(R) of reading Q29.  Then
 *          a'x = a(Re) q x'/Re,  a'y = a(Re) y'/(q Re);   kappa = (psi_xx + psi_yy)/2 with a'(R) = 2 kappa_PJ(R) - a(R)/R. */
static double pjaffe_a(const double *p, double R) {            /* p = sigma0, Ra, Rs */
    const double Ra = p[1], Rs = p[2];
    return 2.0 * p[0] * Ra * Rs / (Rs - Ra) * ((sqrt(Ra * Ra + R * R) - Ra) - (sqrt(Rs * Rs + R * R) - Rs)) / R;
}
static double pjaffe_kappa(const double *p, double R) {
    const double Ra = p[1], Rs = p[2];
    return p[0] * Ra * Rs / (Rs - Ra) * (1.0 / sqrt(Ra * Ra + R * R) - 1.0 / sqrt(Rs * Rs + R * R));
}
double orc_pjaffe_ell_potential(double x, double y, const double *p) {
    double phi0, q;
    orc_ellipticity(p[3], p[4], &phi0, &q);
    const double c = cos(phi0), sn = sin(phi0);
    const double dx = x - p[5], dy = y - p[6];
    const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
    const double R2 = q * xr * xr + yr * yr / q, Ra = p[1], Rs = p[2];
    const double sa = sqrt(Ra * Ra + R2), ss = sqrt(Rs * Rs + R2);
    return 2.0 * p[0] * Ra * Rs / (Rs - Ra) * ((sa - Ra * log(Ra + sa)) - (ss - Rs * log(Rs + ss)));
}
void orc_pjaffe_ell_alpha(double x, double y, const double *p, double *ax, double *ay) {
    double phi0, q;
    orc_ellipticity(p[3], p[4], &phi0, &q);
    const double c = cos(phi0), sn = sin(phi0);
    const double dx = x - p[5], dy = y - p[6];
    const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
    const double Re = sqrt(q * xr * xr + yr * yr / q);
    *ax = 0.0;
    *ay = 0.0;
    if (Re == 0.0) return;
    const double a = pjaffe_a(p, Re);
    const double axr = a * q * xr / Re, ayr = a * yr / (q * Re);
    *ax = c * axr - sn * ayr;
    *ay = sn * axr + c * ayr;
}
double orc_pjaffe_ell_kappa(double x, double y, const double *p) {
    double phi0, q;
    orc_ellipticity(p[3], p[4], &phi0, &q);
    const double c = cos(phi0), sn = sin(phi0);
    const double dx = x - p[5], dy = y - p[6];
    const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
    const double R2 = q * xr * xr + yr * yr / q, R = sqrt(R2);
    const double a = pjaffe_a(p, R), da = 2.0 * pjaffe_kappa(p, R) - a / R;
    const double gx = q * xr / R, gy = yr / (q * R);                 /* grad Re */
    const double pxx = da * gx * gx + a * (q / R - q * q * xr * xr / (R2 * R));
    const double pyy = da * gy * gy + a * (1.0 / (q * R) - yr * yr / (q * q * R2 * R));
    return 0.5 * (pxx + pyy);
}

/* the typed list with the second set: types [n_def], params [n_def][8] */
void orc_profile_alpha2(int type, const double *p, double x, double y, double *ax, double *ay) {
    if (type == ORC_NIE) orc_nie_alpha(x, y, p, ax, ay);
    else if (type == ORC_EPL) orc_epl_alpha(x, y, p, ax, ay);
    else if (type == ORC_MULTIPOLE) orc_multipole_alpha(x, y, p, ax, ay);
    else if (type == ORC_CSE) orc_cse_alpha(x, y, p, ax, ay);
    else if (type == ORC_PJAFFE_ELL) orc_pjaffe_ell_alpha(x, y, p, ax, ay);
    else orc_profile_alpha(type, p, x, y, ax, ay);
}
double orc_profile_kappa2(int type, const double *p, double x, double y) {
    if (type == ORC_NIE) return orc_nie_kappa(x, y, p);
    if (type == ORC_EPL) return orc_epl_kappa(x, y, p);
    if (type == ORC_MULTIPOLE) return orc_multipole_kappa(x, y, p);
    if (type == ORC_CSE) return orc_cse_kappa(x, y, p);
    if (type == ORC_PJAFFE_ELL) return orc_pjaffe_ell_kappa(x, y, p);
    return orc_profile_kappa(type, p, x, y);
}
void orc_ray_shoot_profiles2(int64_t n, const double *tx, const double *ty, int64_t n_def, const int32_t *types,
                             const double *params, double *bx, double *by) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        double sx = 0.0, sy = 0.0;
        for (int64_t d = 0; d < n_def; ++d) {
            double ax, ay;
            orc_profile_alpha2(types[d], params + 8 * d, tx[i], ty[i], &ax, &ay);
            sx += ax;
            sy += ay;
        }
        bx[i] = tx[i] - sx;
        by[i] = ty[i] - sy;
    }
}

/*   light 2 CORE_SERSIC   p = {amp, R_sersic, n_sersic, Rb, gamma, alpha, e1, e2}, centre passed apart
 *        (eight parameters fill the record): with R the product-averaged radius of definition R about (cx, cy),
 *          I = amp (1 + (Rb/R)^alpha)^(gamma/alpha) exp(-b_n [ ((R^alpha + Rb^alpha)/R_sersic^alpha)^(1/(alpha n)) - 1 ])
 *        (Graham et al. 2003 / Trujillo et al. 2004 core-Sersic with b_n of reading Q10): Rb -> 0 IS definition R; the
 *        inner logarithmic slope is -gamma. */
double orc_core_sersic(double x, double y, const double *p, double cx, double cy) {
    double phi, q;
    orc_ellipticity(p[6], p[7], &phi, &q);
    const double c = cos(phi), s = sin(phi);
    const double dx = x - cx, dy = y - cy;
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    const double R = sqrt(q * xr * xr + yr * yr / q);
    const double bn = 1.9992 * p[2] - 0.3271;
    const double Rb = p[3], gam = p[4], al = p[5];
    const double core = R > 0.0 ? pow(1.0 + pow(Rb / R, al), gam / al) : (gam > 0.0 ? INFINITY : 1.0);
    const double arg = pow((pow(R, al) + pow(Rb, al)) / pow(p[1], al), 1.0 / (al * p[2]));
    return p[0] * core * exp(-bn * (arg - 1.0));
}
void orc_core_sersic_n(int64_t n, const double *bx, const double *by, const double *p, double cx, double cy, double *flux) {
    for (int64_t i = 0; i < n; ++i) flux[i] = orc_core_sersic(bx[i], by[i], p, cx, cy);
}

/*   SHAPELETS (n_max = 6 and 10): Cartesian Gauss-Hermite basis (Refregier 2003),
 *          I(x, y) = sum_{n1 + n2 <= n_max} c[k] B_n1(u) B_n2(v) / beta,  u = (x - cx)/beta, v = (y - cy)/beta,
 *          B_n(u) = (2^n sqrt(pi) n!)^(-1/2) H_n(u) exp(-u^2/2)       (H_n: physicists' Hermite polynomials)
 *        coefficient order k: N = n1 + n2 ascending, within N: n2 = 0 ... N (n1 = N - n2); (n_max+1)(n_max+2)/2 of them.
 *        B_n by the stable three-term recurrence of the NORMALISED functions:
 *          B_0 = pi^(-1/4) e^(-u^2/2), B_1 = sqrt 2 u B_0, B_n = sqrt(2/n) u B_(n-1) - sqrt((n-1)/n) B_(n-2). */
#define ORC_SHAPELET_MAX 32
static void shapelet_1d(double u, int n_max, double *B) {
    B[0] = pow(ORC_PI, -0.25) * exp(-0.5 * u * u);
    if (n_max >= 1) B[1] = sqrt(2.0) * u * B[0];
    for (int n = 2; n <= n_max; ++n) B[n] = sqrt(2.0 / n) * u * B[n - 1] - sqrt((n - 1.0) / n) * B[n - 2];
}
double orc_shapelets(double x, double y, int n_max, double beta, double cx, double cy, const double *coef) {
    double Bx[ORC_SHAPELET_MAX + 1], By[ORC_SHAPELET_MAX + 1];
    if (n_max > ORC_SHAPELET_MAX) n_max = ORC_SHAPELET_MAX;
    shapelet_1d((x - cx) / beta, n_max, Bx);
    shapelet_1d((y - cy) / beta, n_max, By);
    double acc = 0.0;
    int k = 0;
    for (int N = 0; N <= n_max; ++N)
        for (int n2 = 0; n2 <= N; ++n2) acc += coef[k++] * Bx[N - n2] * By[n2];
    return acc / beta;
}
void orc_shapelets_n(int64_t n, const double *bx, const double *by, int n_max, double beta, double cx, double cy,
                     const double *coef, double *flux) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) flux[i] = orc_shapelets(bx[i], by[i], n_max, beta, cx, cy, coef);
}

/* ================================================================== NEXT-4: supersampled convolution
 * Reading Q15 convolves at pixel resolution; the variant convolves the UNBINNED ray image (ny s x nx s, each ray
 * carrying its share pixel_scale^2/s^2 of the flux) with a PSF sampled on the ray grid [ky][kx] (odd sizes, in rays)
 * and bins s x s afterwards:  out[j][i] = sum over the pixel's s x s rays of (ray image conv PSF_fine). */
void orc_convolve(int ny, int nx, const double *img, int ky, int kx, const double *ker, double *out);
void orc_convolve_supersampled(int ny, int nx, int s, const double *rays, int ky, int kx, const double *ker_fine, double *tmp,
                               double *out) {
    const int NY = ny * s, NX = nx * s;
    orc_convolve(NY, NX, rays, ky, kx, ker_fine, tmp);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double acc = 0.0;
            for (int a = 0; a < s; ++a)
                for (int b = 0; b < s; ++b) acc += tmp[(size_t)(j * s + a) * NX + (i * s + b)];
            out[(size_t)j * nx + i] = acc;
        }
}
