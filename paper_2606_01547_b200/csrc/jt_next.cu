// jt_next.cu -- the SURVEY.md section 8(f) rows beside the hot path:
//   NEXT-3  jt_chi2_batch: chi^2 of B model images against one data image (the particle-swarm
//           benchmark's inner loop; the fused form lives in jt_batch.cu as jt_simulate_batch_chi2)
//   NEXT-2  jt_lensing_maps: analytic Jacobian of the lens equation -- convergence, shear, magnification of SIE +
//           shear + TNFW (PAPER.md:35, :135 get derivatives by autodiff; here they are written out, reading Q25)
//   NEXT-1  jt_ray_shoot_profiles / jt_light_profiles: typed deflector and light lists with further profiles of
//           PAPER.md:63-87 and :95-108 (CONVERGENCE, SIS, NFW, HERNQUIST, PJAFFE; GAUSSIAN(_ELLIPSE), MULTI_GAUSSIAN)
// These kernels are correct-first: one ray per thread, the list streamed through shared memory, all arithmetic in
// double in both dtype modes (storage in the call's dtype).  They are measured (bench.py --next) but not tier-tuned
// like the hot path's subhalo sum.  Formulas: DESIGN.md readings Q24-Q30; nothing is shared with oracle/.
#include "jt_internal.h"

namespace jt {

constexpr int kNextThreads = 256;

// ---------------------------------------------------------------------------------------------- NEXT-3: chi^2
// One CTA per image; a thread sums its pixels in index order, then warp shuffles and one pass over the 8 warp sums in
// warp order: a fixed summation tree, the same result on every run.
__device__ __forceinline__ double block_sum_256(double v, double* red) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += red[w];
    return s;                                                 // valid in thread 0
}

template <typename T>
__global__ void __launch_bounds__(kNextThreads) k_chi2(int64_t n_pix, const T* __restrict__ models, const T* __restrict__ data,
                                                       const T* __restrict__ sigma, double* __restrict__ chi2) {
    __shared__ double red[kNextThreads / 32];
    const T* m = models + (size_t)blockIdx.x * n_pix;
    double acc = 0.0;
    for (int64_t p = threadIdx.x; p < n_pix; p += kNextThreads) {
        const double r = ((double)m[p] - (double)__ldg(&data[p])) / (double)__ldg(&sigma[p]);
        acc = fma(r, r, acc);
    }
    const double s = block_sum_256(acc, red);
    if (threadIdx.x == 0) chi2[blockIdx.x] = s;
}

jt_status launch_chi2(jt_dtype dtype, int64_t B, int64_t n_pix, const void* models, const void* data, const void* sigma,
                      double* chi2, cudaStream_t st) {
    if (B > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if (dtype == JT_F32)
        k_chi2<float><<<(unsigned)B, kNextThreads, 0, st>>>(n_pix, (const float*)models, (const float*)data, (const float*)sigma, chi2);
    else
        k_chi2<double><<<(unsigned)B, kNextThreads, 0, st>>>(n_pix, (const double*)models, (const double*)data, (const double*)sigma, chi2);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

// ---------------------------------------------------------------------------------------------- shared profile math (double)
// F(X) = arccosh(1/X)/sqrt(1-X^2) (X<1), 1, arccos(1/X)/sqrt(X^2-1) (X>1) in the cancellation-free forms of reading Q9a
__device__ __forceinline__ double nfw_F(double X) {
    if (X < 1.0) { const double s = sqrt((1.0 - X) * (1.0 + X)); return (log1p(s) - log(X)) / s; }
    if (X > 1.0) return 2.0 * atan(sqrt((X - 1.0) / (X + 1.0))) * rsqrt((X - 1.0) * (X + 1.0));
    return 1.0;
}
// (1 - F)/(X^2 - 1); Taylor series sum (-u)^k/(2k+3) around X = 1 (u = X^2 - 1), where the quotient cancels
__device__ __forceinline__ double nfw_G(double X) {
    const double u = fma(X, X, -1.0);
    if (fabs(u) < 0.05) {
        double acc = 1.0 / 25.0;
#pragma unroll
        for (int k = 10; k >= 0; --k) acc = fma(-u, acc, 1.0 / (double)(2 * k + 3));
        return acc;
    }
    return (1.0 - nfw_F(X)) / u;
}
// TNFW (definition T) in double from raw parameters: deflection per unit offset f (alpha = f (dx, dy)) and convergence.
struct TnfwRaw { double cx, cy, Rs, aRs, rt; };
__device__ __forceinline__ void tnfw_f_kappa(const TnfwRaw& s, double dx, double dy, double* f, double* kap) {
    const double R2 = dx * dx + dy * dy;
    if (R2 == 0.0) { *f = 0.0; *kap = 0.0; return; }
    const double X2 = R2 / (s.Rs * s.Rs), X = sqrt(X2);
    const double tau = s.rt / s.Rs, t = tau * tau;
    const double F = nfw_F(X);
    const double S = sqrt(t + X2);
    const double L = log(X / (S + tau));
    const double pre = s.aRs / (1.0 - JT_LN2_D) * t / ((t + 1.0) * (t + 1.0));
    double g;
    if (X2 < 1e-6) {                                           // two-term small-X series of the brace (definition T)
        const double l = log(2.0 / X), lt = log(tau), it = 1.0 / t;
        const double c2 = (t + 1.0) * (t + 1.0) * 0.5 * it * l - (t * t - 1.0) * 0.25 * it - (t - 1.0) * 0.5 * it * lt - JT_PI_D / (2.0 * tau);
        const double c4 = (0.375 * t + 0.625 + 0.125 * it - 0.125 * it * it) * l - 7.0 * t / 32.0 - 9.0 / 32.0 - it / 32.0 +
                          it * it / 32.0 + lt * 0.125 * (it - it * it) + JT_PI_D / (8.0 * tau * t);
        g = X2 * (c2 + X2 * c4);
    } else {
        g = (t + 1.0 + 2.0 * (X2 - 1.0)) * F + tau * JT_PI_D + (t - 1.0) * log(tau) + S * (-JT_PI_D + (t - 1.0) / tau * L);
    }
    *f = pre * g / (X * sqrt(R2));                             // alpha / R, alpha = pre g / X
    *kap = pre / (2.0 * s.Rs) * ((t + 1.0) * nfw_G(X) + 2.0 * F - JT_PI_D / S + (t - 1.0) / (tau * S) * L);
}

// SIE Hessian (reading Q25): |gamma| = kappa, direction along the position angle in the lens frame, spin-2 back-rotation
__device__ __forceinline__ void sie_kg(const MacroLens& m, double x, double y, double* k, double* g1, double* g2) {
    const double dx = x - m.cx, dy = y - m.cy;
    const double xr = m.c * dx + m.s * dy, yr = -m.s * dx + m.c * dy;
    const double r2 = xr * xr + yr * yr;
    if (r2 == 0.0) return;
    const double theta_E = m.b / sqrt(m.q);
    const double kap = 0.5 * theta_E / sqrt(m.q * xr * xr + yr * yr / m.q);
    const double c2 = (xr * xr - yr * yr) / r2, s2 = 2.0 * xr * yr / r2;
    const double C2 = m.c * m.c - m.s * m.s, S2 = 2.0 * m.s * m.c;
    const double g1r = -kap * c2, g2r = -kap * s2;
    *k += kap;
    *g1 += g1r * C2 - g2r * S2;
    *g2 += g1r * S2 + g2r * C2;
}

// ---------------------------------------------------------------------------------------------- NEXT-2: kappa, gamma, mu
template <typename T>
__global__ void __launch_bounds__(kNextThreads) k_lensing_maps(int64_t n, const T* __restrict__ tx, const T* __restrict__ ty,
                                                               const __grid_constant__ MacroLens m, int64_t M,
                                                               const T* __restrict__ t0, const T* __restrict__ t1,
                                                               const T* __restrict__ t2, const T* __restrict__ t3,
                                                               const T* __restrict__ t4, T* __restrict__ kappa,
                                                               T* __restrict__ gamma1, T* __restrict__ gamma2, T* __restrict__ mu) {
    __shared__ TnfwRaw recs[kNextThreads];
    const int64_t i = (int64_t)blockIdx.x * kNextThreads + threadIdx.x;
    const bool live = i < n;
    const double x = live ? (double)tx[i] : 0.0, y = live ? (double)ty[i] : 0.0;
    double k = 0.0, g1 = 0.0, g2 = 0.0;
    if (m.has_sie) sie_kg(m, x, y, &k, &g1, &g2);
    if (m.has_shear) { g1 += m.g1; g2 += m.g2; }
    for (int64_t base = 0; base < M; base += kNextThreads) {
        const int count = (int)min((int64_t)kNextThreads, M - base);
        __syncthreads();
        if ((int)threadIdx.x < count) {
            const int64_t j = base + threadIdx.x;
            recs[threadIdx.x] = {(double)t0[j], (double)t1[j], (double)t2[j], (double)t3[j], (double)t4[j]};
        }
        __syncthreads();
        for (int c = 0; c < count; ++c) {
            const TnfwRaw s = recs[c];
            const double dx = x - s.cx, dy = y - s.cy, R2 = dx * dx + dy * dy;
            if (R2 == 0.0) continue;
            double f, kap;
            tnfw_f_kappa(s, dx, dy, &f, &kap);
            const double gt = f - kap;                          // alpha / R - kappa
            k += kap;
            g1 -= gt * (dx * dx - dy * dy) / R2;
            g2 -= gt * 2.0 * dx * dy / R2;
        }
    }
    if (!live) return;
    if (kappa) kappa[i] = (T)k;
    if (gamma1) gamma1[i] = (T)g1;
    if (gamma2) gamma2[i] = (T)g2;
    if (mu) mu[i] = (T)(1.0 / ((1.0 - k) * (1.0 - k) - g1 * g1 - g2 * g2));
}

jt_status launch_lensing_maps(jt_dtype dtype, int64_t n, const void* tx, const void* ty, const jt_lens* lens, void* kappa,
                              void* gamma1, void* gamma2, void* mu, cudaStream_t st) {
    const MacroLens m = make_macro(lens);
    const int64_t blocks = (n + kNextThreads - 1) / kNextThreads;
    if (blocks > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if (dtype == JT_F32)
        k_lensing_maps<float><<<(unsigned)blocks, kNextThreads, 0, st>>>(
            n, (const float*)tx, (const float*)ty, m, lens->n_tnfw, (const float*)lens->tnfw_cx, (const float*)lens->tnfw_cy,
            (const float*)lens->tnfw_Rs, (const float*)lens->tnfw_alpha_Rs, (const float*)lens->tnfw_r_trunc, (float*)kappa,
            (float*)gamma1, (float*)gamma2, (float*)mu);
    else
        k_lensing_maps<double><<<(unsigned)blocks, kNextThreads, 0, st>>>(
            n, (const double*)tx, (const double*)ty, m, lens->n_tnfw, (const double*)lens->tnfw_cx, (const double*)lens->tnfw_cy,
            (const double*)lens->tnfw_Rs, (const double*)lens->tnfw_alpha_Rs, (const double*)lens->tnfw_r_trunc, (double*)kappa,
            (double*)gamma1, (double*)gamma2, (double*)mu);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

// ---------------------------------------------------------------------------------------------- NEXT-1: typed deflectors
// deflection of one typed record at (x, y), added to (ax, ay); parameters as listed in include/jt.h (jt_profile)
__device__ __forceinline__ void profile_alpha(const jt_profile& d, double x, double y, double& ax, double& ay) {
    const double* p = d.p;
    switch (d.type) {
        case JT_DEFL_CONVERGENCE: ax += p[0] * (x - p[1]); ay += p[0] * (y - p[2]); return;
        case JT_DEFL_SHEAR: ax += p[0] * x + p[1] * y; ay += p[1] * x - p[0] * y; return;
        case JT_DEFL_SIE: {
            const MacroLens m = derive_macro(1, p[0], p[1], p[2], p[3], p[4], 0, 0.0, 0.0);
            double mx, my;
            macro_alpha(m, x, y, mx, my);
            ax += mx; ay += my;
            return;
        }
        case JT_DEFL_NIE: {                                    // reading Q31: definition S with a core s_scale
            double c, sn, q;
            ellipticity(p[1], p[2], &c, &sn, &q);
            const double dx = x - p[4], dy = y - p[5];
            const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
            const double isq = fast_rsqrt(q), b = p[0] * isq, sk = p[3] * isq, f2 = 1.0 - q * q;
            const double psi = sqrt(q * q * (sk * sk + xr * xr) + yr * yr);
            if (psi + sk == 0.0) return;
            const double ux = xr / (psi + sk), uy = yr / (psi + q * q * sk);
            const double axr = b * q * ux * atan_over(f2 * ux * ux), ayr = b * q * uy * atanh_over(f2 * uy * uy);
            ax += c * axr - sn * ayr;
            ay += sn * axr + c * ayr;
            return;
        }
        case JT_DEFL_CSE: {                                    // reading Q37 (Oguri 2021): kappa = A/(2 (s^2 + x'^2 + y'^2/q^2)^(3/2))
            double c, sn, q;
            ellipticity(p[2], p[3], &c, &sn, &q);
            const double dx = x - p[4], dy = y - p[5], s = p[1];
            const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
            const double psi = sqrt(q * q * (s * s + xr * xr) + yr * yr);
            const double pre = p[0] * q / (s * psi * ((psi + s) * (psi + s) + (1.0 - q * q) * xr * xr));
            const double axr = pre * xr * (psi + q * q * s), ayr = pre * yr * (psi + s);
            ax += c * axr - sn * ayr;
            ay += sn * axr + c * ayr;
            return;
        }
        case JT_DEFL_PJAFFE_ELLIPSE_POTENTIAL: {               // reading Q38: psi(x', y') = psi_PJ(sqrt(q x'^2 + y'^2/q))
            double c, sn, q;
            ellipticity(p[3], p[4], &c, &sn, &q);
            const double dx = x - p[5], dy = y - p[6];
            const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
            const double R2 = q * xr * xr + yr * yr / q;
            if (R2 == 0.0) return;
            const double R = sqrt(R2), Ra = p[1], Rs = p[2];
            const double a = 2.0 * p[0] * Ra * Rs / (Rs - Ra) * ((sqrt(Ra * Ra + R2) - Ra) - (sqrt(Rs * Rs + R2) - Rs)) / R;
            const double axr = a * q * xr / R, ayr = a * yr / (q * R);
            ax += c * axr - sn * ayr;
            ay += sn * axr + c * ayr;
            return;
        }
        case JT_DEFL_MULTIPOLE: {                              // reading Q36: psi = r a_m/(1 - m^2) cos(m (phi - phi_m)), m >= 2
            const double dx = x - p[3], dy = y - p[4], m = p[0];
            if (dx == 0.0 && dy == 0.0) return;
            const double phi = atan2(dy, dx), amp = p[1] / (1.0 - m * m);
            double sm, cm, sp, cp;
            sincos(m * (phi - p[2]), &sm, &cm);
            sincos(phi, &sp, &cp);
            const double ar = amp * cm, aphi = -m * amp * sm;
            ax += ar * cp - aphi * sp;
            ay += ar * sp + aphi * cp;
            return;
        }
        case JT_DEFL_EPL: {                                    // reading Q32: Tessore & Metcalf (2015) series
            double c, sn, q;
            ellipticity(p[2], p[3], &c, &sn, &q);
            const double dx = x - p[4], dy = y - p[5];
            const double xr = c * dx + sn * dy, yr = -sn * dx + c * dy;
            const double t = p[1] - 1.0, b = p[0] * sqrt(q);
            const double R2 = q * q * xr * xr + yr * yr;
            if (R2 == 0.0) return;
            const double R = sqrt(R2), cph = q * xr / R, sph = yr / R;
            const double c2 = cph * cph - sph * sph, s2 = 2.0 * cph * sph, f = (1.0 - q) / (1.0 + q);
            double are = cph, aim = sph, sre = cph, sim = sph;
            for (int n = 1; n <= 400; ++n) {
                const double g = -f * (2.0 * n - (2.0 - t)) / (2.0 * n + (2.0 - t));
                const double nre = g * (c2 * are - s2 * aim), nim = g * (c2 * aim + s2 * are);
                are = nre; aim = nim;
                sre += are; sim += aim;
                if (are * are + aim * aim < 1e-34 * (sre * sre + sim * sim)) break;
            }
            const double pre = 2.0 * b / (1.0 + q) * pow(b / R, t - 1.0);
            ax += pre * (c * sre - sn * sim);
            ay += pre * (sn * sre + c * sim);
            return;
        }
        case JT_DEFL_TNFW: {
            const TnfwRaw s = {p[3], p[4], p[0], p[1], p[2]};
            double f, kap;
            tnfw_f_kappa(s, x - s.cx, y - s.cy, &f, &kap);
            ax += f * (x - s.cx); ay += f * (y - s.cy);
            return;
        }
        default: break;
    }
    double cx, cy;
    if (d.type == JT_DEFL_SIS) { cx = p[1]; cy = p[2]; }
    else if (d.type == JT_DEFL_PJAFFE) { cx = p[3]; cy = p[4]; }
    else { cx = p[2]; cy = p[3]; }
    const double dx = x - cx, dy = y - cy, R2 = dx * dx + dy * dy;
    if (R2 == 0.0) return;
    const double R = sqrt(R2);
    double a = 0.0;                                            // deflection magnitude
    if (d.type == JT_DEFL_SIS) {
        a = p[0];
    } else if (d.type == JT_DEFL_NFW) {
        const double X = R / p[0];
        a = p[1] / (1.0 - JT_LN2_D) * (log(0.5 * X) + nfw_F(X)) / X;
    } else if (d.type == JT_DEFL_HERNQUIST) {
        const double X = R / p[0];
        a = 2.0 * p[1] * p[0] * X * nfw_G(X);
    } else if (d.type == JT_DEFL_PJAFFE) {
        const double Ra = p[1], Rs = p[2];
        a = 2.0 * p[0] * Ra * Rs / (Rs - Ra) * ((sqrt(Ra * Ra + R2) - Ra) - (sqrt(Rs * Rs + R2) - Rs)) / R;
    }
    ax += a * dx / R;
    ay += a * dy / R;
}

template <typename T>
__global__ void __launch_bounds__(kNextThreads) k_ray_shoot_profiles(int64_t n, const T* __restrict__ tx, const T* __restrict__ ty,
                                                                     int64_t n_def, const jt_profile* __restrict__ defs,
                                                                     T* __restrict__ bx, T* __restrict__ by) {
    __shared__ jt_profile recs[64];
    const int64_t i = (int64_t)blockIdx.x * kNextThreads + threadIdx.x;
    const bool live = i < n;
    const double x = live ? (double)tx[i] : 0.0, y = live ? (double)ty[i] : 0.0;
    double ax = 0.0, ay = 0.0;
    for (int64_t base = 0; base < n_def; base += 64) {
        const int count = (int)min((int64_t)64, n_def - base);
        __syncthreads();
        for (int w = threadIdx.x; w < count * (int)(sizeof(jt_profile) / 8); w += kNextThreads)
            reinterpret_cast<double*>(recs)[w] = reinterpret_cast<const double*>(defs + base)[w];
        __syncthreads();
        for (int c = 0; c < count; ++c) profile_alpha(recs[c], x, y, ax, ay);
    }
    if (live) { bx[i] = (T)(x - ax); by[i] = (T)(y - ay); }
}

jt_status launch_ray_shoot_profiles(jt_dtype dtype, int64_t n, const void* tx, const void* ty, int64_t n_def,
                                    const jt_profile* defs, void* bx, void* by, cudaStream_t st) {
    const int64_t blocks = (n + kNextThreads - 1) / kNextThreads;
    if (blocks > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if (dtype == JT_F32)
        k_ray_shoot_profiles<float><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const float*)tx, (const float*)ty, n_def, defs,
                                                                               (float*)bx, (float*)by);
    else
        k_ray_shoot_profiles<double><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const double*)tx, (const double*)ty, n_def, defs,
                                                                                (double*)bx, (double*)by);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

// ---------------------------------------------------------------------------------------------- NEXT-1: typed light
__device__ __forceinline__ double profile_light(const jt_profile& d, double bx, double by) {
    const double* p = d.p;
    double c, s, q;
    if (d.type == JT_LIGHT_SERSIC_ELLIPSE) {
        ellipticity(p[3], p[4], &c, &s, &q);
        const double dx = bx - p[5], dy = by - p[6];
        const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
        const double a = (q * xr * xr + yr * yr / q) / (p[1] * p[1]);
        const double bn = 1.9992 * p[2] - 0.3271;             // reading Q10
        const double pw = a > 0.0 ? exp(0.5 / p[2] * log(a)) : 0.0;
        return p[0] * exp(-bn * (pw - 1.0));
    }
    if (d.type != JT_LIGHT_GAUSSIAN_ELLIPSE) return 0.0;      // unknown types contribute nothing (jt.h)
    ellipticity(p[2], p[3], &c, &s, &q);
    const double dx = bx - p[4], dy = by - p[5];
    const double xr = c * dx + s * dy, yr = -s * dx + c * dy;
    const double i2s = 0.5 / (p[1] * p[1]);
    return p[0] * i2s / JT_PI_D * exp(-(q * xr * xr + yr * yr / q) * i2s);
}

template <typename T>
__global__ void __launch_bounds__(kNextThreads) k_light_profiles(int64_t n, const T* __restrict__ bx, const T* __restrict__ by,
                                                                 int64_t n_comp, const jt_profile* __restrict__ comps,
                                                                 T* __restrict__ flux) {
    __shared__ jt_profile recs[64];
    const int64_t i = (int64_t)blockIdx.x * kNextThreads + threadIdx.x;
    const bool live = i < n;
    const double x = live ? (double)bx[i] : 0.0, y = live ? (double)by[i] : 0.0;
    double acc = 0.0;
    for (int64_t base = 0; base < n_comp; base += 64) {
        const int count = (int)min((int64_t)64, n_comp - base);
        __syncthreads();
        for (int w = threadIdx.x; w < count * (int)(sizeof(jt_profile) / 8); w += kNextThreads)
            reinterpret_cast<double*>(recs)[w] = reinterpret_cast<const double*>(comps + base)[w];
        __syncthreads();
        for (int c = 0; c < count; ++c) acc += profile_light(recs[c], x, y);
    }
    if (live) flux[i] = (T)acc;
}

jt_status launch_light_profiles(jt_dtype dtype, int64_t n, const void* bx, const void* by, int64_t n_comp,
                                const jt_profile* comps, void* flux, cudaStream_t st) {
    const int64_t blocks = (n + kNextThreads - 1) / kNextThreads;
    if (blocks > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if (dtype == JT_F32)
        k_light_profiles<float><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const float*)bx, (const float*)by, n_comp, comps, (float*)flux);
    else
        k_light_profiles<double><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const double*)bx, (const double*)by, n_comp, comps, (double*)flux);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

// ---------------------------------------------------------------------------------------------- NEXT-1: CORE_SERSIC, SHAPELETS
struct CoreSersic { double amp, iRs, n, Rb, gam, al, c, s, q, cx, cy, bn; };

template <typename T>
__global__ void __launch_bounds__(kNextThreads) k_core_sersic(int64_t n, const T* __restrict__ bx, const T* __restrict__ by,
                                                              const __grid_constant__ CoreSersic P, T* __restrict__ flux) {
    const int64_t i = (int64_t)blockIdx.x * kNextThreads + threadIdx.x;
    if (i >= n) return;
    const double dx = (double)bx[i] - P.cx, dy = (double)by[i] - P.cy;
    const double xr = P.c * dx + P.s * dy, yr = -P.s * dx + P.c * dy;
    const double R = sqrt(P.q * xr * xr + yr * yr / P.q);
    const double core = R > 0.0 ? pow(1.0 + pow(P.Rb / R, P.al), P.gam / P.al) : (P.gam > 0.0 ? INFINITY : 1.0);
    const double arg = pow((pow(R, P.al) + pow(P.Rb, P.al)) * pow(P.iRs, P.al), 1.0 / (P.al * P.n));
    flux[i] = (T)(P.amp * core * exp(-P.bn * (arg - 1.0)));
}

jt_status launch_core_sersic(jt_dtype dtype, int64_t n, const void* bx, const void* by, const double* p, void* flux, cudaStream_t st) {
    CoreSersic P;
    P.amp = p[0]; P.iRs = 1.0 / p[1]; P.n = p[2]; P.Rb = p[3]; P.gam = p[4]; P.al = p[5];
    ellipticity(p[6], p[7], &P.c, &P.s, &P.q);
    P.cx = p[8]; P.cy = p[9];
    P.bn = 1.9992 * p[2] - 0.3271;                             // reading Q10
    const int64_t blocks = (n + kNextThreads - 1) / kNextThreads;
    if (blocks > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if (dtype == JT_F32) k_core_sersic<float><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const float*)bx, (const float*)by, P, (float*)flux);
    else k_core_sersic<double><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const double*)bx, (const double*)by, P, (double*)flux);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

// Shapelets (reading Q34): the coefficient triangle sits in shared memory, pre-multiplied by the recurrence's
// normalisation; a thread runs the two 1-D recurrences in registers (n_max <= JT_MAX_SHAPELET_ORDER, unrolled) and
// contracts them with the triangle: (n_max+1)(n_max+2)/2 multiply-adds per ray.  A dense contraction only in name --
// one 66-vector per ray against basis values that exist nowhere but in that ray's registers -- so no tensor cores.
template <typename T>
__global__ void __launch_bounds__(kNextThreads) k_shapelets(int64_t n, const T* __restrict__ bx, const T* __restrict__ by, int n_max,
                                                            double ibeta, double cx, double cy, const T* __restrict__ coef,
                                                            T* __restrict__ flux) {
    __shared__ double s_c[(JT_MAX_SHAPELET_ORDER + 1) * (JT_MAX_SHAPELET_ORDER + 2) / 2];
    __shared__ double s_a[JT_MAX_SHAPELET_ORDER + 1], s_b[JT_MAX_SHAPELET_ORDER + 1];
    const int nk = (n_max + 1) * (n_max + 2) / 2;
    for (int k = threadIdx.x; k < nk; k += kNextThreads) s_c[k] = (double)coef[k];
    for (int m = threadIdx.x; m <= n_max; m += kNextThreads) {
        s_a[m] = m > 0 ? sqrt(2.0 / m) : 0.0;                  // B_m = a_m u B_(m-1) - b_m B_(m-2)
        s_b[m] = m > 0 ? sqrt((m - 1.0) / m) : 0.0;
    }
    __syncthreads();
    const int64_t i = (int64_t)blockIdx.x * kNextThreads + threadIdx.x;
    if (i >= n) return;
    const double u = ((double)bx[i] - cx) * ibeta, v = ((double)by[i] - cy) * ibeta;
    double Bx[JT_MAX_SHAPELET_ORDER + 1], By[JT_MAX_SHAPELET_ORDER + 1];
    const double g0 = 0.75112554446494248285870300477623;     // pi^(-1/4)
    Bx[0] = g0 * exp(-0.5 * u * u);
    By[0] = g0 * exp(-0.5 * v * v);
#pragma unroll
    for (int m = 1; m <= JT_MAX_SHAPELET_ORDER; ++m) {
        Bx[m] = m <= n_max ? s_a[m] * u * Bx[m - 1] - (m > 1 ? s_b[m] * Bx[m - 2] : 0.0) : 0.0;
        By[m] = m <= n_max ? s_a[m] * v * By[m - 1] - (m > 1 ? s_b[m] * By[m - 2] : 0.0) : 0.0;
    }
    double acc = 0.0;
#pragma unroll
    for (int N = 0; N <= JT_MAX_SHAPELET_ORDER; ++N) {
        if (N <= n_max) {
#pragma unroll
            for (int n2 = 0; n2 <= N; ++n2) acc = fma(s_c[N * (N + 1) / 2 + n2], Bx[N - n2] * By[n2], acc);
        }
    }
    flux[i] = (T)(acc * ibeta);
}

jt_status launch_shapelets(jt_dtype dtype, int64_t n, const void* bx, const void* by, int n_max, double beta, double cx, double cy,
                           const void* coef, void* flux, cudaStream_t st) {
    const int64_t blocks = (n + kNextThreads - 1) / kNextThreads;
    if (blocks > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if (dtype == JT_F32)
        k_shapelets<float><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const float*)bx, (const float*)by, n_max, 1.0 / beta, cx, cy,
                                                                      (const float*)coef, (float*)flux);
    else
        k_shapelets<double><<<(unsigned)blocks, kNextThreads, 0, st>>>(n, (const double*)bx, (const double*)by, n_max, 1.0 / beta, cx, cy,
                                                                       (const double*)coef, (double*)flux);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

// ---------------------------------------------------------------------------------------------- NEXT-4: s x s binning
// out[j][i] = sum of the s x s block of the ray-resolution image (summed in double, fixed order)
template <typename T>
__global__ void __launch_bounds__(kNextThreads) k_bin_sum(int ny, int nx, int s, const T* __restrict__ fine, T* __restrict__ out) {
    const int64_t p = (int64_t)blockIdx.x * kNextThreads + threadIdx.x;
    if (p >= (int64_t)ny * nx) return;
    const int j = (int)(p / nx), i = (int)(p - (int64_t)j * nx);
    const int64_t NX = (int64_t)nx * s;
    double acc = 0.0;
    for (int a = 0; a < s; ++a)
        for (int b = 0; b < s; ++b) acc += (double)fine[((int64_t)j * s + a) * NX + ((int64_t)i * s + b)];
    out[p] = (T)acc;
}

jt_status launch_bin_sum(jt_dtype dtype, int ny, int nx, int s, const void* fine, void* out, cudaStream_t st) {
    const int64_t blocks = ((int64_t)ny * nx + kNextThreads - 1) / kNextThreads;
    if (blocks > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if (dtype == JT_F32) k_bin_sum<float><<<(unsigned)blocks, kNextThreads, 0, st>>>(ny, nx, s, (const float*)fine, (float*)out);
    else k_bin_sum<double><<<(unsigned)blocks, kNextThreads, 0, st>>>(ny, nx, s, (const double*)fine, (double*)out);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

}  // namespace jt
