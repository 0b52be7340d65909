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
