/*
 * oracle.c -- plain, slow, obviously-correct CPU oracle for the lensed-image hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  The product
 * (paper_2606_01547_b200/, include/jt.h) shares no code, header, table or helper with it.
 *
 * What it computes: the three steps of PAPER.md:55 (section "Improvements over lenstronomy
 * in image simulation"): (1) a coordinate grid in the observer's angles is ray-traced through
 * the deflectors back to the source plane, (2) the source surface brightness is evaluated on
 * the traced grid, (3) the lensed image is convolved with the PSF.  The paper prints profile
 * NAMES only (PAPER.md:80 NIE/SIE, :85 SHEAR, :87 TNFW, :103 SERSIC_ELLIPSE); every formula
 * below is the reading fixed in SURVEY.md §8(c) (definitions G, E, S, H, T, R, B, P) and
 * listed in DESIGN.md "Readings".  Everything is IEEE double, naive loops, no blocking, no
 * fusion, no reordering beyond the definitions.  `#pragma omp parallel for` on the outermost
 * independent loop only spreads identical per-element work over host cores.
 *
 * Pins (tests/test_oracle_*.py): SIS |alpha|=theta_E; point mass theta_E^2/r; div alpha =
 * 2 kappa and curl alpha = 0 by central differences for S, H, T; NFW limit of T; total-mass
 * limit of T; projected TNFW mass against numerical line-of-sight quadrature (mpmath);
 * Sersic isophote / total flux closed forms and the half-light fraction inside R_sersic (pins the two
 * constants of b_n, reading Q10); grid + bin invariants; convolution against
 * scipy.signal.convolve2d, delta / shift kernels, flux conservation, 8x8 brute force.
 * The composed pipeline has no external implementation to compare with: "parity unpinned"
 * end-to-end, pinned per step (SURVEY.md §8(c) last pin row).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------ threads */
void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_get_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ G: grid
 * SURVEY §8(c) G.  Sub-ray (J,I): theta_x = cx + (I - (nx*s-1)/2) h, theta_y = cy + (J - (ny*s-1)/2) h,
 * h = pixel_scale/s.  Row-major, x fastest. */
void orc_grid(int nx, int ny, double pixel_scale, double cx, double cy, int s,
              double *theta_x, double *theta_y) {
    const int NX = nx * s, NY = ny * s;
    const double h = pixel_scale / (double)s;
    for (int J = 0; J < NY; ++J)
        for (int I = 0; I < NX; ++I) {
            theta_x[(size_t)J * NX + I] = cx + ((double)I - 0.5 * (double)(NX - 1)) * h;
            theta_y[(size_t)J * NX + I] = cy + ((double)J - 0.5 * (double)(NY - 1)) * h;
        }
}

/* ------------------------------------------------------------------ E: ellipticity
 * (e1,e2) -> phi = atan2(e2,e1)/2; c = min(|e|, 0.9999); q = (1-c)/(1+c). */
void orc_ellipticity(double e1, double e2, double *phi, double *q) {
    double c = sqrt(e1 * e1 + e2 * e2);
    if (c > 0.9999) c = 0.9999;
    *phi = 0.5 * atan2(e2, e1);
    *q = (1.0 - c) / (1.0 + c);
}

/* A(z) = atan(z)/z, Bh(z) = atanh(z)/z, both 1 at z = 0 (series below 1e-4). */
static double fn_A(double z) {
    if (fabs(z) < 1e-4) { double z2 = z * z; return 1.0 - z2 / 3.0 + z2 * z2 / 5.0; }
    return atan(z) / z;
}
static double fn_Bh(double z) {
    if (fabs(z) < 1e-4) { double z2 = z * z; return 1.0 + z2 / 3.0 + z2 * z2 / 5.0; }
    return atanh(z) / z;
}

/* ------------------------------------------------------------------ S: SIE
 * p = {theta_E, e1, e2, cx, cy}.  kappa = theta_E / (2 sqrt(q x'^2 + y'^2/q)).
 * b = theta_E sqrt(q), f = sqrt(1-q^2), psi = sqrt(q^2 x'^2 + y'^2):
 *   a'x = b (x'/psi) A(f x'/psi),  a'y = b (y'/psi) Bh(f y'/psi); rotate back by phi.  alpha(psi=0) = 0. */
void orc_sie_alpha(double x, double y, const double *p, double *ax, double *ay) {
    double phi, q;
    orc_ellipticity(p[1], p[2], &phi, &q);
    const double c = cos(phi), s = sin(phi);
    const double dx = x - p[3], dy = y - p[4];
    const double xr = c * dx + s * dy;
    const double yr = -s * dx + c * dy;
    const double psi = sqrt(q * q * xr * xr + yr * yr);
    if (psi == 0.0) { *ax = 0.0; *ay = 0.0; return; }
    const double b = p[0] * sqrt(q);
    const double f = sqrt(1.0 - q * q);
    const double axr = b * (xr / psi) * fn_A(f * xr / psi);
    const double ayr = b * (yr / psi) * fn_Bh(f * yr / psi);
    *ax = c * axr - s * ayr;
    *ay = s * axr + c * ayr;
}

double orc_sie_kappa(double x, double y, const double *p) {
    double phi, q;
    orc_ellipticity(p[1], p[2], &phi, &q);
    const double c = cos(phi), s = sin(phi);
    const double dx = x - p[3], dy = y - p[4];
    const double xr = c * dx + s * dy;
    const double yr = -s * dx + c * dy;
    return 0.5 * p[0] / sqrt(q * xr * xr + yr * yr / q);
}

/* ------------------------------------------------------------------ H: external shear about the origin */
void orc_shear_alpha(double x, double y, double g1, double g2, double *ax, double *ay) {
    *ax = g1 * x + g2 * y;
    *ay = g2 * x - g1 * y;
}

/* ------------------------------------------------------------------ point mass (oracle-only pin) */
void orc_pointmass_alpha(double x, double y, double theta_E, double cx, double cy, double *ax, double *ay) {
    const double dx = x - cx, dy = y - cy;
    const double r2 = dx * dx + dy * dy;
    if (r2 == 0.0) { *ax = 0.0; *ay = 0.0; return; }
    *ax = theta_E * theta_E * dx / r2;
    *ay = theta_E * theta_E * dy / r2;
}

/* ------------------------------------------------------------------ T: truncated NFW
 * rho(r) = rho0 / [x (1+x)^2] * tau^2/(tau^2+x^2), x = r/Rs, tau = r_trunc/Rs.
 * alpha_Rs = deflection at Rs of the UNtruncated NFW with the same rho0: 4 rho0 Rs^2 = alpha_Rs/(1-ln2). */
/* F(X) = arccosh(1/X)/sqrt(1-X^2) (X<1), 1 (X=1), arccos(1/X)/sqrt(X^2-1) (X>1)   [definition T].
 * Written with the identities arccosh(1/X) = ln((1+s)/X), s = sqrt((1-X)(1+X)), and
 * arccos(1/X) = 2 arctan(sqrt((X-1)/(X+1))): the same function, but 1-X is exact in floating point
 * near X = 1 whereas 1/X rounds to 1 there and the literal form loses every digit for |X-1| < 1e-8
 * (reading Q9a; pinned against the literal definition in 40-digit mpmath at
 * X = 1 +- 1e-3 ... 1 ulp and over 1e-6 ... 1e4 in tests/test_oracle_lens.py). */
double orc_tnfw_F(double X) {
    if (X < 1.0) { const double s = sqrt((1.0 - X) * (1.0 + X)); return (log1p(s) - log(X)) / s; }
    if (X > 1.0) return 2.0 * atan(sqrt((X - 1.0) / (X + 1.0))) / sqrt((X - 1.0) * (X + 1.0));
    return 1.0;
}

double orc_tnfw_L(double X, double tau) {
    return log(X / (sqrt(tau * tau + X * X) + tau));
}

/* closed form of g(X,tau) */
double orc_tnfw_g_closed(double X, double tau) {
    const double t = tau * tau;
    const double F = orc_tnfw_F(X);
    const double L = orc_tnfw_L(X, tau);
    const double S = sqrt(t + X * X);
    const double brace = (t + 1.0 + 2.0 * (X * X - 1.0)) * F + tau * ORC_PI + (t - 1.0) * log(tau)
                       + S * (-ORC_PI + ((t - 1.0) / tau) * L);
    return t / ((t + 1.0) * (t + 1.0)) * brace;
}

/* two-term small-X series of the brace, l = ln(2/X), t = tau^2 */
double orc_tnfw_g_series(double X, double tau) {
    const double t = tau * tau;
    const double l = log(2.0 / X);
    const double lt = log(tau);
    const double X2 = X * X;
    const double c2 = (t + 1.0) * (t + 1.0) / (2.0 * t) * l - (t * t - 1.0) / (4.0 * t)
                    - (t - 1.0) / (2.0 * t) * lt - ORC_PI / (2.0 * tau);
    const double c4 = (3.0 * t / 8.0 + 5.0 / 8.0 + 1.0 / (8.0 * t) - 1.0 / (8.0 * t * t)) * l
                    - 7.0 * t / 32.0 - 9.0 / 32.0 - 1.0 / (32.0 * t) + 1.0 / (32.0 * t * t)
                    + lt * (1.0 / (8.0 * t) - 1.0 / (8.0 * t * t)) + ORC_PI / (8.0 * tau * tau * tau);
    const double brace = X2 * c2 + X2 * X2 * c4;
    return t / ((t + 1.0) * (t + 1.0)) * brace;
}

/* oracle rule: closed form for X >= 1e-3, series below */
double orc_tnfw_g(double X, double tau) {
    return (X < 1e-3) ? orc_tnfw_g_series(X, tau) : orc_tnfw_g_closed(X, tau);
}

/* alpha(R) = alpha_Rs/(1-ln2) * g(X,tau)/X along (theta-c)/R; 0 at R = 0 */
void orc_tnfw_alpha(double x, double y, double cx, double cy, double Rs, double alpha_Rs, double r_trunc,
                    double *ax, double *ay) {
    const double dx = x - cx, dy = y - cy;
    const double R = sqrt(dx * dx + dy * dy);
    if (R == 0.0) { *ax = 0.0; *ay = 0.0; return; }
    const double X = R / Rs;
    const double tau = r_trunc / Rs;
    const double a = alpha_Rs / (1.0 - log(2.0)) * orc_tnfw_g(X, tau) / X;
    *ax = a * dx / R;
    *ay = a * dy / R;
}

/* convergence, used only by the div(alpha) = 2 kappa pin */
double orc_tnfw_kappa(double x, double y, double cx, double cy, double Rs, double alpha_Rs, double r_trunc) {
    const double dx = x - cx, dy = y - cy;
    const double X = sqrt(dx * dx + dy * dy) / Rs;
    const double tau = r_trunc / Rs;
    const double t = tau * tau;
    const double F = orc_tnfw_F(X);
    const double L = orc_tnfw_L(X, tau);
    const double S = sqrt(t + X * X);
    const double brace = (t + 1.0) / (X * X - 1.0) * (1.0 - F) + 2.0 * F - ORC_PI / S + (t - 1.0) / (tau * S) * L;
    return alpha_Rs / ((1.0 - log(2.0)) * Rs) * t / (2.0 * (t + 1.0) * (t + 1.0)) * brace;
}

/* ------------------------------------------------------------------ lens equation
 * beta = theta - alpha_SIE - alpha_shear - sum_j alpha_TNFW,j   (single plane)
 * sie: 5 doubles or NULL; shear: 2 doubles or NULL; tnfw: [5][M] rows cx,cy,Rs,alpha_Rs,r_trunc. */
static void ray_beta(double x, double y, const double *sie, const double *shear, int64_t M, const double *tnfw,
                     double *bx, double *by) {
    double sx = 0.0, sy = 0.0, ax, ay;
    if (sie) { orc_sie_alpha(x, y, sie, &ax, &ay); sx += ax; sy += ay; }
    if (shear) { orc_shear_alpha(x, y, shear[0], shear[1], &ax, &ay); sx += ax; sy += ay; }
    for (int64_t j = 0; j < M; ++j) {
        orc_tnfw_alpha(x, y, tnfw[j], tnfw[M + j], tnfw[2 * M + j], tnfw[3 * M + j], tnfw[4 * M + j], &ax, &ay);
        sx += ax; sy += ay;
    }
    *bx = x - sx;
    *by = y - sy;
}

void orc_ray_shoot(int64_t n, const double *theta_x, const double *theta_y,
                   const double *sie, const double *shear, int64_t M, const double *tnfw,
                   double *beta_x, double *beta_y) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i)
        ray_beta(theta_x[i], theta_y[i], sie, shear, M, tnfw, &beta_x[i], &beta_y[i]);
}

/* ------------------------------------------------------------------ R: elliptical Sersic
 * p = {amp, R_sersic, n_sersic, e1, e2, cx, cy}.  R = sqrt(q x'^2 + y'^2/q), b_n = 1.9992 n - 0.3271,
 * I = amp exp(-b_n [ (R/R_sersic)^(1/n) - 1 ]). */
double orc_sersic(double x, double y, const double *p) {
    double phi, q;
    orc_ellipticity(p[3], p[4], &phi, &q);
    const double c = cos(phi), s = sin(phi);
    const double dx = x - p[5], dy = y - p[6];
    const double xr = c * dx + s * dy;
    const double yr = -s * dx + c * dy;
    const double R = sqrt(q * xr * xr + yr * yr / q);
    const double bn = 1.9992 * p[2] - 0.3271;
    return p[0] * exp(-bn * (pow(R / p[1], 1.0 / p[2]) - 1.0));
}

/* surface brightness (no area factor) summed over n_src components; src is [n_src][7] */
void orc_source_brightness(int64_t n, const double *beta_x, const double *beta_y,
                           int n_src, const double *src, double *flux) {
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double acc = 0.0;
        for (int k = 0; k < n_src; ++k) acc += orc_sersic(beta_x[i], beta_y[i], src + 7 * k);
        flux[i] = acc;
    }
}

/* ------------------------------------------------------------------ B: binning
 * image[j][i] = pixel_scale^2 / s^2 * sum over the s x s sub-rays of pixel (j,i). */
void orc_bin(int nx, int ny, int s, double pixel_scale, const double *flux, double *image) {
    const int NX = nx * s;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double acc = 0.0;
            for (int a = 0; a < s; ++a)
                for (int b = 0; b < s; ++b)
                    acc += flux[(size_t)(j * s + a) * NX + (i * s + b)];
            image[(size_t)j * nx + i] = pixel_scale * pixel_scale * acc / (double)(s * s);
        }
}

/* ------------------------------------------------------------------ P: PSF convolution
 * out[j][i] = sum_{u<ky} sum_{v<kx} K[u][v] img[j-(u-cy)][i-(v-cx)], cy = ky/2, cx = kx/2,
 * out-of-range terms dropped (zero padding, 'same' size, true convolution). */
void orc_convolve(int ny, int nx, const double *img, int ky, int kx, const double *K, double *out) {
    const int cy = ky / 2, cx = kx / 2;
#pragma omp parallel for schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double acc = 0.0;
            for (int u = 0; u < ky; ++u) {
                const int jj = j - (u - cy);
                if (jj < 0 || jj >= ny) continue;
                for (int v = 0; v < kx; ++v) {
                    const int ii = i - (v - cx);
                    if (ii < 0 || ii >= nx) continue;
                    acc += K[(size_t)u * kx + v] * img[(size_t)jj * nx + ii];
                }
            }
            out[(size_t)j * nx + i] = acc;
        }
}

/* ------------------------------------------------------------------ composed steps
 * Pre-PSF image rows [j0, j1): steps G, lens equation, R, B for those pixel rows only
 * (the row window exists so that the largest config can be sampled; j0=0, j1=ny is the whole image).
 * image_rows is [(j1-j0)][nx]. */
void orc_prepsf_rows(int nx, int ny, double pixel_scale, double gcx, double gcy, int s,
                     const double *sie, const double *shear, int64_t M, const double *tnfw,
                     int n_src, const double *src, int j0, int j1, double *image_rows) {
    const int NX = nx * s, NY = ny * s;
    const double h = pixel_scale / (double)s;
    const int64_t npix = (int64_t)(j1 - j0) * nx;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t pidx = 0; pidx < npix; ++pidx) {
        const int j = j0 + (int)(pidx / nx), i = (int)(pidx % nx);
        double acc = 0.0;
        for (int a = 0; a < s; ++a)
            for (int b = 0; b < s; ++b) {
                const int J = j * s + a, I = i * s + b;
                const double tx = gcx + ((double)I - 0.5 * (double)(NX - 1)) * h;
                const double ty = gcy + ((double)J - 0.5 * (double)(NY - 1)) * h;
                double bx, by;
                ray_beta(tx, ty, sie, shear, M, tnfw, &bx, &by);
                for (int k = 0; k < n_src; ++k) acc += orc_sersic(bx, by, src + 7 * k);
            }
        image_rows[pidx] = pixel_scale * pixel_scale * acc / (double)(s * s);
    }
}

/* whole pipeline: pre_psf [ny][nx] (scratch, also returned) and out [ny][nx] */
void orc_simulate_image(int nx, int ny, double pixel_scale, double gcx, double gcy, int s,
                        const double *sie, const double *shear, int64_t M, const double *tnfw,
                        int n_src, const double *src, int ky, int kx, const double *K,
                        double *pre_psf, double *out) {
    orc_prepsf_rows(nx, ny, pixel_scale, gcx, gcy, s, sie, shear, M, tnfw, n_src, src, 0, ny, pre_psf);
    orc_convolve(ny, nx, pre_psf, ky, kx, K, out);
}

/* B independent systems sharing one grid: sie [B][5], shear [B][2], tnfw [B][5][M], src [B][n_src][7], K [B][ky][kx] */
void orc_simulate_batch(int64_t B, int nx, int ny, double pixel_scale, double gcx, double gcy, int s,
                        const double *sie, const double *shear, int64_t M, const double *tnfw,
                        int n_src, const double *src, int ky, int kx, const double *K, double *out) {
    double *pre = (double *)malloc(sizeof(double) * (size_t)nx * ny);
    for (int64_t b = 0; b < B; ++b) {
        orc_simulate_image(nx, ny, pixel_scale, gcx, gcy, s, sie + 5 * b, shear + 2 * b, M, tnfw + 5 * M * b,
                           n_src, src + (size_t)7 * n_src * b, ky, kx, K + (size_t)ky * kx * b,
                           pre, out + (size_t)nx * ny * b);
    }
    free(pre);
}

/* ------------------------------------------------------------------ chi^2 of B model images against one data image
 * NEXT-3 (the particle-swarm benchmark: every particle is one simulated image
 * compared with the same data).  The paper prints no likelihood formula; reading Q24: Gaussian pixel noise,
 *   chi2[b] = sum_{j,i} ( (model[b][j][i] - data[j][i]) / sigma[j][i] )^2 ,   log L = -chi2 / 2,
 * sigma = the per-pixel noise rms map (> 0).  Plain double loop in row-major order. */
void orc_chi2_batch(int64_t B, int64_t n_pix, const double *models, const double *data, const double *sigma, double *chi2) {
    for (int64_t b = 0; b < B; ++b) {
        double acc = 0.0;
        for (int64_t p = 0; p < n_pix; ++p) {
            const double r = (models[b * n_pix + p] - data[p]) / sigma[p];
            acc += r * r;
        }
        chi2[b] = acc;
    }
}

