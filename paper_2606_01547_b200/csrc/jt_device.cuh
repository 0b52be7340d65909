// jt_device.cuh -- device arithmetic of the lensing hot path (sm_100a).
//
// Definitions implemented (readings in DESIGN.md; the paper, PAPER.md:55/:80/:85/:87/:103, prints names only):
//   E ellipticity, S SIE deflection, H external shear, T truncated-NFW deflection, R elliptical Sersic.
// Shares nothing with oracle/: the formulas are re-derived in the forms the GPU wants
// (rsqrt-based, polynomial atan/atanh, cancellation-free far field), see DESIGN.md "Kernel arithmetic".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "jt_poly.h"

namespace jt {

#define JT_PI_D 3.14159265358979323846264338327950288
#define JT_LN2_D 0.693147180559945309417232121458176568

// ------------------------------------------------------------------------------------------------
// small numeric helpers
// ------------------------------------------------------------------------------------------------
template <typename T, int N>
__device__ __forceinline__ T horner(const T (&c)[N], T z) {
    T p = c[0];
#pragma unroll
    for (int i = 1; i < N; ++i) p = fma(p, z, c[i]);
    return p;
}

// atan(sqrt z)/sqrt z on [0,1/9]  (far field: z = 1/(X^2-1))
__device__ __forceinline__ float atan_far(float z) { const float c[] = {JT_ATAN_FAR_F32_COEFS}; return horner(c, z); }
__device__ __forceinline__ double atan_far(double z) { const double c[] = {JT_ATAN_FAR_F64_COEFS}; return horner(c, z); }
// atan(sqrt z)/sqrt z on [0,1]
__device__ __forceinline__ float atan_full(float z) { const float c[] = {JT_ATAN_FULL_F32_COEFS}; return horner(c, z); }
__device__ __forceinline__ double atan_full(double z) { const double c[] = {JT_ATAN_FULL_F64_COEFS}; return horner(c, z); }
// atanh(sqrt z)/sqrt z on [0,1/4]
__device__ __forceinline__ float atanh_q(float z) { const float c[] = {JT_ATANH_Q_F32_COEFS}; return horner(c, z); }
__device__ __forceinline__ double atanh_q(double z) { const double c[] = {JT_ATANH_Q_F64_COEFS}; return horner(c, z); }

// Reciprocal square root / reciprocal: one MUFU seed (~20-22 bits) + one third-order correction.
__device__ __forceinline__ float fast_rsqrt(float x) {                                     // bare MUFU.RSQ
    float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
}
// keeps a value in its register: stops the compiler re-deriving a float from the double it was rounded from
__device__ __forceinline__ void pin(float& v) { asm volatile("" : "+f"(v)); }
__device__ __forceinline__ void pin(double& v) { asm volatile("" : "+d"(v)); }
__device__ __forceinline__ float fast_rcp(float x) { return __frcp_rn(x); }
__device__ __forceinline__ float approx_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ double fast_rsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));          // MUFU.RSQ64H, ~20 bits
    const double e = fma(-x, y * y, 1.0);                             // e = 1 - x y^2  (~2^-19)
    return fma(y, e * fma(0.375, e, 0.5), y);                         // y (1 + e/2 + 3e^2/8): error O(e^3)
}
__device__ __forceinline__ double fast_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));            // MUFU.RCP64H, ~20 bits
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);                                   // y (1 + e + e^2): error O(e^3)
}
__device__ __forceinline__ double approx_rcp(double x) { return fast_rcp(x); }

__device__ __forceinline__ float t_sqrt(float x) { return sqrtf(x); }
__device__ __forceinline__ double t_sqrt(double x) { return sqrt(x); }
__device__ __forceinline__ float t_log(float x) { return logf(x); }
__device__ __forceinline__ double t_log(double x) { return log(x); }

// ------------------------------------------------------------------------------------------------
// T: truncated NFW.  Per-subhalo record, derived once (in double) when a tile is staged.
//   alpha = amp * brace(X^2) / R^2 * (dx, dy),   X^2 = R^2 * iRs2,   amp = alpha_Rs/(1-ln2) * Rs * t/(t+1)^2,
//   brace = (t-1+2X^2) F(X) + c1 + S (c2 L - pi),  t = tau^2, c1 = tau pi + (t-1) ln tau, c2 = (t-1)/tau,
//   S = sqrt(t+X^2), L = ln(X/(S+tau)).
// ------------------------------------------------------------------------------------------------
// Far-far field: for X >= 9 max(1, tau) (double; 6.5 max(1, tau) in float) the brace is summed from its expansion in
// 1/X, derived with sympy from the closed form (every coefficient carries the factor (t+1)^2; the 1/X term vanishes):
//   brace = b0 + b2 / X^2 + b3 / X^3 + ... ,   b0 = (t-1) ln tau - t + pi tau - 1 (the total-mass limit),
//   b2 = -(t+1)^2/3, b3 = pi (t+1)^2/8, b4 = 2 (t+1)^2 (t-3)/15, b5 = -pi (t+1)^2 (t-2)/16, ...
// Truncated after 1/X^13 (double) / 1/X^8 (float) the relative error is <= 1e-13 / 3e-8 beyond those radii (reading
// Q9b in DESIGN.md: verified against the closed form at 50 digits for tau = 0.3 ... 1000).  With v = 1/R (NOT 1/X: the
// powers of Rs are folded into the coefficients, a_k = amp b_k Rs^k) the deflection is alpha = f (dx, dy),
//   f = v^2 (a_0 + v^2 (a_2 + a_3 v + ... + a_K v^(K-2))):  one MUFU and K + 1 multiply-adds per evaluation.
// The farther the ray, the shorter the sum: three levels (K, radius in units of max(1, tau) Rs), each within the same
// error bound (double 1e-13: 2.2e-14 / 6.0e-14 / 5e-14 worst case at tau = 1 on the radius; float 3e-8 = half an ulp:
// 2.7e-8 / 2.2e-8 / 2.1e-8):
template <typename T> struct FarFar;
template <> struct FarFar<double> {
    static constexpr int K = 13, K1 = 9, K2 = 7;
    static constexpr double kRadius = 9.0, kRadius1 = 20.0, kRadius2 = 44.0;
};
template <> struct FarFar<float> {
    static constexpr int K = 8, K1 = 5, K2 = 4;
    static constexpr double kRadius = 6.5, kRadius1 = 18.0, kRadius2 = 32.0;
};

// Field order = access order: the far-far loop reads the first (K + 3) values only (centre, a_0, a_2 ... a_K); the
// classification pass reads cx, cy, thr2, iRs2, thr; the far / mid / generic forms read the rest.
template <typename T>
struct alignas(sizeof(T) * 4) SubRec {
    T cx, cy, a0, thr2;        // centre; a_0; far-far threshold on X^2 (huge when the series is switched off for this record)
    T ak[(FarFar<T>::K - 1 + 3) / 4 * 4];      // a_2 ... a_K, zero-padded to a multiple of 4
    T iRs2, thr, t, a_tm1;     // 1/Rs^2; far-field threshold on X^2 (= max(10, 3t)); tau^2; amp (t-1)
    T a_c1, a_pi, c_a, c_b;    // amp c1, amp pi, amp (t-1) pi/2, amp (t+1)
    T c_c, amp, tm1, c1;       // 2 amp; amplitude; tau^2 - 1, c1 (generic near-field forms)
};

// b_k / (t+1)^2 for k = 2 ... 13 as polynomials in t (sympy series of the closed form)
__host__ __device__ inline double farfar_coef(int k, double t) {
    const double pi = JT_PI_D;
    switch (k) {
        case 2: return -1.0 / 3.0;
        case 3: return pi / 8.0;
        case 4: return 2.0 / 15.0 * (t - 3.0);
        case 5: return -pi / 16.0 * (t - 2.0);
        case 6: return -8.0 / 105.0 * ((t - 3.0) * t + 5.0);
        case 7: return 5.0 * pi / 128.0 * ((t - 2.0) * t + 3.0);
        case 8: return 16.0 / 315.0 * (((t - 3.0) * t + 5.0) * t - 7.0);
        case 9: return -7.0 * pi / 256.0 * (((t - 2.0) * t + 3.0) * t - 4.0);
        case 10: return -128.0 / 3465.0 * ((((t - 3.0) * t + 5.0) * t - 7.0) * t + 9.0);
        case 11: return 21.0 * pi / 1024.0 * ((((t - 2.0) * t + 3.0) * t - 4.0) * t + 5.0);
        case 12: return 256.0 / 9009.0 * (((((t - 3.0) * t + 5.0) * t - 7.0) * t + 9.0) * t - 11.0);
        case 13: return -33.0 * pi / 2048.0 * (((((t - 2.0) * t + 3.0) * t - 4.0) * t + 5.0) * t - 6.0);
        default: return 0.0;
    }
}

template <typename T>
__device__ __forceinline__ SubRec<T> make_rec(double cx, double cy, double Rs, double aRs, double rt) {
    const double tau = rt / Rs, t = tau * tau;
    const double lt = log(tau);
    const double c1 = tau * JT_PI_D + (t - 1.0) * lt;
    const double amp = aRs / (1.0 - JT_LN2_D) * Rs * t / ((t + 1.0) * (t + 1.0));
    const double iRs2 = 1.0 / (Rs * Rs);
    SubRec<T> r;
    r.cx = (T)cx;
    r.cy = (T)cy;
    r.iRs2 = (T)iRs2;
    r.thr = (T)fmax(10.0, 3.0 * t);
    r.t = (T)t;
    r.a_tm1 = (T)(amp * (t - 1.0));
    r.a_c1 = (T)(amp * c1);
    r.a_pi = (T)(amp * JT_PI_D);
    r.c_a = (T)(amp * (t - 1.0) * (JT_PI_D / 2));
    r.c_b = (T)(amp * (t + 1.0));
    r.c_c = (T)(2.0 * amp);
    r.amp = (T)amp;
    r.tm1 = (T)(t - 1.0);
    r.c1 = (T)c1;
    const double rad = FarFar<T>::kRadius * fmax(1.0, tau);
    r.thr2 = (T)(rad * rad);
    r.a0 = (T)(amp * ((t - 1.0) * lt - t + JT_PI_D * tau - 1.0));
    // a_k = amp b_k Rs^k.  A coefficient that leaves T's normal range in either direction (extreme tau, tiny Rs)
    // switches the series off for this record: it then takes the far form, which has no such limit.
    const double big = sizeof(T) == 4 ? 1e30 : 1e250, tiny = sizeof(T) == 4 ? 1e-30 : 1e-280;
    bool ok = isfinite((double)r.a0);
    double f = amp * (t + 1.0) * (t + 1.0) * Rs;
#pragma unroll
    for (int k = 2; k <= FarFar<T>::K; ++k) {
        f *= Rs;
        const double a = f * farfar_coef(k, t);
        ok = ok && isfinite(a) && fabs(a) < big && (a == 0.0 || fabs(a) > tiny);
        r.ak[k - 2] = (T)a;
    }
#pragma unroll
    for (int k = FarFar<T>::K - 1; k < (int)(sizeof(r.ak) / sizeof(T)); ++k) r.ak[k] = (T)0;
    if (!ok) {
        r.thr2 = (T)(sizeof(T) == 4 ? 3.0e38 : 1.0e300);
        r.a0 = (T)0;
#pragma unroll
        for (int k = 0; k < FarFar<T>::K - 1; ++k) r.ak[k] = (T)0;
    }
    return r;
}

// Far-far field (see FarFar above), series summed to 1/R^K.  Returns f with alpha = f * (dx, dy).
template <typename T, int K = FarFar<T>::K>
__device__ __forceinline__ T tnfw_farfar(T R2, const SubRec<T>& s) {
    const T v = fast_rsqrt(R2);
    const T v2 = v * v;
    T p = s.ak[K - 2];
#pragma unroll
    for (int k = K - 3; k >= 0; --k) p = fma(p, v, s.ak[k]);
    return v2 * fma(p, v2, s.a0);
}

// Far field, X^2 >= max(10, 3t): no logarithm, no cancellation growing with X.
//   w = 1/sqrt(X^2-1), z = w^2 <= 1/9, y = t/(X^2+t) <= 1/4,  P = atan(w)/w, Q = atanh(sqrt y)/sqrt y
//   F = (pi/2 - w P) w;   S c2 L = -(t-1) Q;   2 X^2 F - pi S = pi (w X^2 - S) - 2 (1+z) P      (w + u = w X^2)
//   amp brace = a_tm1 (F - Q) + a_c1 + a_pi (w X^2 - S) - 2 amp (1+z) P
//             = (c_a w + a_c1) - P (c_b z + c_c) - a_tm1 Q + a_pi (w X^2 - S)      (F and the (1+z) P term merged:
//               c_a = amp (t-1) pi/2, c_b = amp (t-1) + 2 amp, c_c = 2 amp; two instructions fewer)
// Returns f with alpha = f * (dx, dy).
template <typename T>
__device__ __forceinline__ T tnfw_far(T R2, const SubRec<T>& s) {
    const T X2 = R2 * s.iRs2;
    const T u2 = X2 - (T)1;
    const T S2 = X2 + s.t;
    const T w = fast_rsqrt(u2);
    const T rS = fast_rsqrt(S2);
    const T iR2 = approx_rcp(R2);
    const T S = S2 * rS, z = w * w, y = (s.t * rS) * rS;
    const T P = atan_far(z);
    const T Q = atanh_q(y);
    T b = fma(-P, fma(s.c_b, z, s.c_c), fma(s.c_a, w, s.a_c1));
    b = fma(-s.a_tm1, Q, b);
    b = fma(s.a_pi, fma(w, X2, -S), b);
    return b * iR2;
}

// Two rays at once in float: the two Horner chains (10 of the 30 FP32 instructions of an evaluation) run as sm_100
// packed FMAs (fma.rn.f32x2 -> FFMA2, the coefficient as a broadcast operand), which halves their issue slots -- the
// float far loop is bound by the issue port, not by the FP32 pipe.
__device__ __forceinline__ unsigned long long pack2(float lo, float hi) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpack2(unsigned long long v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long fma2c(unsigned long long p, unsigned long long z, float c) {
    unsigned long long d;
    asm("{\n\t.reg .b64 cc;\n\tmov.b64 cc, {%3, %3};\n\tfma.rn.f32x2 %0, %1, %2, cc;\n\t}" : "=l"(d) : "l"(p), "l"(z), "f"(c));
    return d;
}
template <int N>
__device__ __forceinline__ unsigned long long horner2(const float (&c)[N], unsigned long long z) {
    unsigned long long p = pack2(c[0], c[0]);
#pragma unroll
    for (int i = 1; i < N; ++i) p = fma2c(p, z, c[i]);
    return p;
}
typedef unsigned long long f32x2;                         // two floats in one 64-bit register (lo, hi)
__device__ __forceinline__ f32x2 bc2(float x) { return pack2(x, x); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
// far-far field on two rays at once (float): R2 = (R2a, R2b) packed
template <int K>
__device__ __forceinline__ f32x2 tnfw_farfar2(f32x2 R2, const SubRec<float>& s) {
    float ra, rb;
    unpack2(R2, ra, rb);
    const f32x2 v = pack2(fast_rsqrt(ra), fast_rsqrt(rb));
    const f32x2 v2 = mul2(v, v);
    f32x2 p = bc2(s.ak[K - 2]);
#pragma unroll
    for (int k = K - 3; k >= 0; --k) p = fma2(p, v, bc2(s.ak[k]));
    return mul2(v2, fma2(p, v2, bc2(s.a0)));
}

// The whole far-field form on two rays at once (same algebra as tnfw_far<float>; MUFU on the halves).
__device__ __forceinline__ void tnfw_far_pair(float R2a, float R2b, const SubRec<float>& s, float& fa, float& fb) {
    const f32x2 R2 = pack2(R2a, R2b);
    const f32x2 X2 = mul2(R2, bc2(s.iRs2));
    const f32x2 u2 = add2(X2, bc2(-1.f));
    const f32x2 S2 = add2(X2, bc2(s.t));
    float u2a, u2b, S2a, S2b;
    unpack2(u2, u2a, u2b);
    unpack2(S2, S2a, S2b);
    const f32x2 w = pack2(fast_rsqrt(u2a), fast_rsqrt(u2b));
    const f32x2 rS = pack2(fast_rsqrt(S2a), fast_rsqrt(S2b));
    const f32x2 iR2 = pack2(approx_rcp(R2a), approx_rcp(R2b));
    const f32x2 z = mul2(w, w);
    const f32x2 y = mul2(mul2(bc2(s.t), rS), rS);
    const float cp[] = {JT_ATAN_FAR_F32_COEFS};
    const float cq[] = {JT_ATANH_Q_F32_COEFS};
    const f32x2 P = horner2(cp, z);
    const f32x2 Q = horner2(cq, y);
    // amp brace = (c_a w + a_c1) - P (c_b z + c_c) - a_tm1 Q + a_pi (w X2 - S2 rS)
    const f32x2 g = fma2(bc2(-s.c_b), z, bc2(-s.c_c));                 // -(c_b z + c_c)
    f32x2 b = fma2(P, g, fma2(bc2(s.c_a), w, bc2(s.a_c1)));
    b = fma2(bc2(-s.a_tm1), Q, b);
    b = fma2(bc2(s.a_pi), mul2(w, X2), b);
    b = fma2(bc2(-s.a_pi), mul2(S2, rS), b);
    unpack2(mul2(b, iR2), fa, fb);
}

// ln x for normal positive x.  float: one MUFU.LG2.  double: x = 2^e m, m in (sqrt(1/2), sqrt 2],
// ln m = 2 atanh(s), s = (m-1)/(m+1), |s| <= 0.1716: odd series to s^19 (remainder 2.3e-17); no libdevice slow path.
__device__ __forceinline__ float ln_pos(float x) { return __log2f(x) * 0.693147180559945f; }
__device__ __forceinline__ double ln_pos(double x) {
    int hi = __double2hiint(x);
    const int lo = __double2loint(x);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;
    if (hi > 0x3ff6a09e) { hi -= 0x00100000; e += 1; }
    const double m = __hiloint2double(hi, lo);
    const double q = (m - 1.0) * fast_rcp(m + 1.0);
    const double q2 = q * q;
    double p = 1.0 / 19.0;
    p = fma(p, q2, 1.0 / 17.0);
    p = fma(p, q2, 1.0 / 15.0);
    p = fma(p, q2, 1.0 / 13.0);
    p = fma(p, q2, 1.0 / 11.0);
    p = fma(p, q2, 1.0 / 9.0);
    p = fma(p, q2, 1.0 / 7.0);
    p = fma(p, q2, 1.0 / 5.0);
    p = fma(p, q2, 1.0 / 3.0);
    const double lm = fma(q * q2, p + p, q + q);
    return fma((double)e, JT_LN2_D, lm);
}

// Mid field, X^2 >= 2: the far-field algebra with the full-range atan polynomial (w = 1/sqrt(X^2-1) <= 1) and
//   Q = atanh(tau/S)/(tau/S) = (S/tau) ln((S+tau)/X)  from one logarithm (S^2 - tau^2 = X^2, so no cancellation).
// Returns f with alpha = f * (dx, dy).
template <typename T>
__device__ __forceinline__ T tnfw_midfast(T R2, const SubRec<T>& s) {
    const T X2 = R2 * s.iRs2;
    const T u2 = X2 - (T)1, S2 = X2 + s.t;
    const T w = fast_rsqrt(u2);
    const T rS = fast_rsqrt(S2);
    const T rt = fast_rsqrt(s.t);
    const T iR2 = approx_rcp(R2);
    const T iX2 = approx_rcp(X2);
    const T S = S2 * rS, tau = s.t * rt, z = w * w;
    const T P = atan_full(z);
    const T d = S + tau;
    const T Q = (S * rt) * ((T)0.5 * ln_pos((d * d) * iX2));
    T b = fma(-P, fma(s.c_b, z, s.c_c), fma(s.c_a, w, s.a_c1));
    b = fma(-s.a_tm1, Q, b);
    b = fma(s.a_pi, fma(w, X2, -S), b);
    return b * iR2;
}

// Closed form for any X^2 > 0 (float: use only for X^2 >= 1/4; double: X^2 >= 1e-6).
template <typename T>
__device__ __noinline__ T tnfw_mid(T R2, T iRs2, T t, T c1, T amp, T tm1) {
    const T X2 = R2 * iRs2;
    const T S = t_sqrt(t + X2);
    const T tau = t_sqrt(t);
    const T d = S + tau;
    const T L = (T)0.5 * t_log(X2 / (d * d));
    T F, G2;                                         // G2 = 2 X^2 F - pi S
    if (X2 > (T)1) {
        const T u2 = X2 - (T)1;
        if (u2 >= (T)1) {
            const T w = (T)1 / t_sqrt(u2), z = w * w;
            const T P = atan_full(z);
            F = fma(-w, P, (T)(JT_PI_D / 2)) * w;
            G2 = fma((T)JT_PI_D, (w + u2 * w) - S, (T)-2 * fma(z, P, P));
        } else {
            F = atan_full(u2);
            G2 = fma((T)2 * X2, F, -(T)JT_PI_D * S);
        }
    } else {
        const T u2 = (T)1 - X2;
        if (u2 <= (T)0.25) {
            F = atanh_q(u2);
        } else {
            const T u = t_sqrt(u2);
            F = (t_log((T)1 + u) - (T)0.5 * t_log(X2)) / u;
        }
        G2 = fma((T)2 * X2, F, -(T)JT_PI_D * S);
    }
    const T b = fma(tm1, F, c1) + fma((tm1 / tau) * S, L, G2);
    return amp * b / R2;
}

// Two-term small-X series of the brace (X < 1e-3 in double), l = ln(2/X), t = tau^2.
static __device__ __noinline__ double tnfw_series(double R2, double iRs2, double t, double amp) {
    const double X2 = R2 * iRs2;
    const double tau = sqrt(t), lt = log(tau), l = 0.5 * log(4.0 / X2);
    const double it = 1.0 / t;
    const double c2 = (t + 1.0) * (t + 1.0) * 0.5 * it * l - (t * t - 1.0) * 0.25 * it - (t - 1.0) * 0.5 * it * lt
                    - JT_PI_D / (2.0 * tau);
    const double c4 = (0.375 * t + 0.625 + 0.125 * it - 0.125 * it * it) * l - 7.0 * t / 32.0 - 9.0 / 32.0
                    - it / 32.0 + it * it / 32.0 + lt * 0.125 * (it - it * it) + JT_PI_D / (8.0 * tau * t);
    const double b = X2 * (c2 + X2 * c4);
    return amp * b / R2;
}

// Any R^2 in double from a double record (used by the f64 kernels' generic path and by the f32 near path).
__device__ __forceinline__ double tnfw_any(double R2, const SubRec<double>& s) {
    if (R2 == 0.0) return 0.0;
    const double X2 = R2 * s.iRs2;
    if (X2 < 1e-6) return tnfw_series(R2, s.iRs2, s.t, s.amp);
    return tnfw_mid<double>(R2, s.iRs2, s.t, s.c1, s.amp, s.tm1);
}

// ------------------------------------------------------------------------------------------------
// S + H: smooth lens, evaluated per ray in double (both modes).  Host precomputes E: (cos phi, sin phi, q).
//   b = theta_E sqrt q, f = sqrt(1-q^2), psi = sqrt(q^2 x'^2 + y'^2)
//   a'x = b (x'/psi) A(f x'/psi), a'y = b (y'/psi) Bh(f y'/psi), A = atan(z)/z, Bh = atanh(z)/z.
// ------------------------------------------------------------------------------------------------
struct MacroLens {
    int has_sie, has_shear;
    double c, s, q, b, f, cx, cy;
    double g1, g2;
};

// definition E: (e1,e2) -> (cos phi, sin phi, q), |e| clamped to 0.9999
__host__ __device__ inline void ellipticity(double e1, double e2, double* c, double* s, double* q) {
    double m = sqrt(e1 * e1 + e2 * e2);
    if (m > 0.9999) m = 0.9999;
    const double phi = 0.5 * atan2(e2, e1);
    *c = cos(phi);
    *s = sin(phi);
    *q = (1.0 - m) / (1.0 + m);
}

__host__ __device__ inline MacroLens derive_macro(int has_sie, double theta_E, double e1, double e2, double cx, double cy,
                                                  int has_shear, double g1, double g2) {
    MacroLens m = {};
    m.has_sie = has_sie ? 1 : 0;
    m.has_shear = has_shear ? 1 : 0;
    if (m.has_sie) {
        ellipticity(e1, e2, &m.c, &m.s, &m.q);
        m.b = theta_E * sqrt(m.q);
        m.f = sqrt(1.0 - m.q * m.q);
        m.cx = cx;
        m.cy = cy;
    }
    if (m.has_shear) { m.g1 = g1; m.g2 = g2; }
    return m;
}

__device__ __forceinline__ double atanh_over(double z2) {      // atanh(z)/z as a function of z^2 in [0,1)
    if (z2 <= 0.25) return atanh_q(z2);
    const double iz = fast_rsqrt(z2), z = z2 * iz;             // no libdevice sqrt / log / division slow paths
    return 0.5 * ln_pos((1.0 + z) * fast_rcp(1.0 - z)) * iz;
}

__device__ __forceinline__ double atan_over(double z2) {       // atan(z)/z as a function of z^2 >= 0
    if (z2 <= 1.0) return atan_full(z2);
    const double iz = fast_rsqrt(z2), iz2 = iz * iz;           // atan z = pi/2 - atan(1/z)
    return fma(JT_PI_D / 2, iz, -atan_full(iz2) * iz2);
}

__device__ __forceinline__ void macro_alpha(const MacroLens& m, double x, double y, double& ax, double& ay) {
    ax = 0.0; ay = 0.0;
    if (m.has_sie) {
        const double dx = x - m.cx, dy = y - m.cy;
        const double xr = m.c * dx + m.s * dy, yr = -m.s * dx + m.c * dy;
        const double psi2 = m.q * m.q * xr * xr + yr * yr;
        if (psi2 > 0.0) {
            const double ipsi = fast_rsqrt(psi2);
            const double cx_ = xr * ipsi, cy_ = yr * ipsi;        // x'/psi, y'/psi
            const double zx = m.f * cx_, zy = m.f * cy_;
            const double A = atan_over(zx * zx);                  // |zx| <= f/q, above 1 when q < 0.707
            const double Bh = atanh_over(zy * zy);
            const double axr = m.b * cx_ * A, ayr = m.b * cy_ * Bh;
            ax = m.c * axr - m.s * ayr;
            ay = m.s * axr + m.c * ayr;
        }
    }
    if (m.has_shear) {
        ax += m.g1 * x + m.g2 * y;
        ay += m.g2 * x - m.g1 * y;
    }
}

// ------------------------------------------------------------------------------------------------
// R: elliptical Sersic.  Host precomputes per component: cos phi, sin phi, q, 1/q, centre, amp, b_n,
// p = 1/(2 n), 1/R_sersic^2.   I = amp exp(-b_n ((R^2/Rs^2)^p - 1)),  R^2 = q x'^2 + y'^2/q.
// ------------------------------------------------------------------------------------------------
#define JT_MAX_SRC 16
struct SrcSet {
    int n;
    double c[JT_MAX_SRC], s[JT_MAX_SRC], q[JT_MAX_SRC], iq[JT_MAX_SRC], cx[JT_MAX_SRC], cy[JT_MAX_SRC];
    double amp[JT_MAX_SRC], bn[JT_MAX_SRC], p[JT_MAX_SRC], iRs2[JT_MAX_SRC];
};

__host__ __device__ inline void derive_source(SrcSet& S, int k, double amp, double R_sersic, double n_sersic, double e1,
                                              double e2, double cx, double cy) {
    ellipticity(e1, e2, &S.c[k], &S.s[k], &S.q[k]);
    S.iq[k] = 1.0 / S.q[k];
    S.cx[k] = cx;
    S.cy[k] = cy;
    S.amp[k] = amp;
    S.bn[k] = 1.9992 * n_sersic - 0.3271;                 // reading Q10
    S.p[k] = 0.5 / n_sersic;
    S.iRs2[k] = 1.0 / (R_sersic * R_sersic);
}

template <typename T>
__device__ __forceinline__ double sersic_sum(const SrcSet& S, double bx, double by);

template <>
__device__ __forceinline__ double sersic_sum<double>(const SrcSet& S, double bx, double by) {
    double acc = 0.0;
    for (int k = 0; k < S.n; ++k) {
        const double dx = bx - S.cx[k], dy = by - S.cy[k];
        const double xr = S.c[k] * dx + S.s[k] * dy, yr = -S.s[k] * dx + S.c[k] * dy;
        const double a = (S.q[k] * xr * xr + S.iq[k] * yr * yr) * S.iRs2[k];
        const double pw = (a > 0.0) ? exp(S.p[k] * log(a)) : 0.0;
        acc += S.amp[k] * exp(-S.bn[k] * (pw - 1.0));
    }
    return acc;
}

// float mode: the subtraction beta - centre stays double (it cancels), the profile itself is float
// with MUFU lg2/ex2 (error analysis in DESIGN.md "Precision").
template <>
__device__ __forceinline__ double sersic_sum<float>(const SrcSet& S, double bx, double by) {
    float acc = 0.f;
    for (int k = 0; k < S.n; ++k) {
        const float dx = (float)(bx - S.cx[k]), dy = (float)(by - S.cy[k]);
        const float c = (float)S.c[k], s = (float)S.s[k];
        const float xr = c * dx + s * dy, yr = -s * dx + c * dy;
        const float a = ((float)S.q[k] * xr * xr + (float)S.iq[k] * yr * yr) * (float)S.iRs2[k];
        const float pw = (a > 0.f) ? exp2f((float)S.p[k] * __log2f(a)) : 0.f;
        acc += (float)S.amp[k] * exp2f((float)(-S.bn[k] * 1.4426950408889634) * (pw - 1.f));
    }
    return (double)acc;
}

}  // namespace jt
