// jt_fft.cu -- step 5b: PSF convolution by hand-written shared-memory FFTs (definition P; PAPER.md:110-114
// "FFT convolution").  Reaches the direct-convolution result up to rounding.  cuFFT is not used (tests only).
//
// out = crop( IFFT2( FFT2(img) . FFT2(ker) ) ), both zero-padded to Py x Px, the smallest 2^a 3^b 5^c sizes
// >= n + K - 1 (Px even): C4 pads 600 x 600, not 1024 x 1024.
//
// Real input, so only the Px/2 + 1 non-redundant columns of the row spectra exist anywhere:
//   k_fft_rows_fwd : two REAL rows of the same array ride one complex transform, z = row_a + i row_b ->
//                    A_k = (Z_k + conj Z_{P-k})/2, B_k = (Z_k - conj Z_{P-k})/(2i); image rows -> plane SA [ny][Ph],
//                    kernel rows -> plane SB [ky][Ph]  (Ph = Px/2 + 1; rows of zeros are never transformed)
//   k_fft_cols     : a CTA owns a few spectrum columns: column FFTs of SA and SB (zero-padded to Py), pointwise
//                    product with the 1/(Px Py) scale, inverse column FFT, all in shared memory; stores only the ny
//                    rows the crop keeps -> plane SC [ny][Ph]
//   k_fft_rows_inv : two output rows ride one inverse complex transform (Z_k = C_a,k + i C_b,k, Hermitian-extended),
//                    real part -> row a, imaginary part -> row b, cropped at kx/2
// Three launches on the caller's stream; the two later ones are programmatic dependent launches whose twiddle set-up
// overlaps the previous kernel's tail.  The planes (C4: 5.3 MB) live in the caller's workspace and stay in L2.
//
// The transforms are Stockham autosort FFTs (natural order in and out, ping-pong between two shared-memory buffers,
// no bit reversal), mixed radix 4 / 2 / 3 / 5 with the butterflies in registers; a thread reads its R inputs at
// stride N/R (conflict-free) and one table twiddle per output.  All arithmetic is double in BOTH dtype modes (float
// converts on load and store only): the FP64 pipe is nowhere near the limit here, L2 traffic and launch latency are.
#include "jt_internal.h"

namespace jt {

using Cd = double2;
constexpr int kFftMaxThreads = 512;            // CTA size is chosen per plan
constexpr int kFftMaxP = 2048;                 // two ping-pong buffers + the twiddle table of one transform fit 227 KB
constexpr int kFftMaxPasses = 12;
constexpr size_t kFftMaxSmem = 220 * 1024;

__device__ __forceinline__ Cd cadd(Cd a, Cd b) { return {a.x + b.x, a.y + b.y}; }
__device__ __forceinline__ Cd csub(Cd a, Cd b) { return {a.x - b.x, a.y - b.y}; }
__device__ __forceinline__ Cd cmul(Cd a, Cd b) { return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x}; }
__device__ __forceinline__ Cd cmul_conj(Cd a, Cd b) { return {a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y}; }  // a conj(b)
// multiply by SIGN * i  (forward transforms use exp(-i...): SIGN = -1)
template <int SIGN> __device__ __forceinline__ Cd mul_i(Cd a) { return SIGN < 0 ? Cd{a.y, -a.x} : Cd{-a.y, a.x}; }

// length-R DFT in registers, c_k = sum_j a_j exp(SIGN 2 pi i j k / R)
template <int R, int SIGN> struct Dft;
template <int SIGN> struct Dft<2, SIGN> {
    static __device__ __forceinline__ void run(Cd (&a)[2]) {
        const Cd t = a[0];
        a[0] = cadd(t, a[1]);
        a[1] = csub(t, a[1]);
    }
};
template <int SIGN> struct Dft<4, SIGN> {
    static __device__ __forceinline__ void run(Cd (&a)[4]) {
        const Cd t0 = cadd(a[0], a[2]), t1 = csub(a[0], a[2]), t2 = cadd(a[1], a[3]), t3 = mul_i<SIGN>(csub(a[1], a[3]));
        a[0] = cadd(t0, t2);
        a[1] = cadd(t1, t3);
        a[2] = csub(t0, t2);
        a[3] = csub(t1, t3);
    }
};
template <int SIGN> struct Dft<3, SIGN> {
    static __device__ __forceinline__ void run(Cd (&a)[3]) {
        const double s3 = SIGN * 0.86602540378443864676372317075294;      // sin(2 pi / 3)
        const Cd s = cadd(a[1], a[2]), d = csub(a[1], a[2]);
        const Cd m = {a[0].x - 0.5 * s.x, a[0].y - 0.5 * s.y};
        const Cd n = {-s3 * d.y, s3 * d.x};                               // i sin d
        a[0] = cadd(a[0], s);
        a[1] = cadd(m, n);
        a[2] = csub(m, n);
    }
};
template <int SIGN> struct Dft<5, SIGN> {
    static __device__ __forceinline__ void run(Cd (&a)[5]) {
        const double c1 = 0.30901699437494742410229341718282, c2 = -0.80901699437494742410229341718282;   // cos(2 pi/5), cos(4 pi/5)
        const double s1 = SIGN * 0.95105651629515357211643933337938, s2 = SIGN * 0.58778525229247312916870595463907;
        const Cd p1 = cadd(a[1], a[4]), d1 = csub(a[1], a[4]), p2 = cadd(a[2], a[3]), d2 = csub(a[2], a[3]);
        const Cd m1 = {a[0].x + c1 * p1.x + c2 * p2.x, a[0].y + c1 * p1.y + c2 * p2.y};
        const Cd m2 = {a[0].x + c2 * p1.x + c1 * p2.x, a[0].y + c2 * p1.y + c1 * p2.y};
        const Cd u1 = {s1 * d1.x + s2 * d2.x, s1 * d1.y + s2 * d2.y};     // sin1 d1 + sin2 d2
        const Cd u2 = {s2 * d1.x - s1 * d2.x, s2 * d1.y - s1 * d2.y};     // sin2 d1 - sin1 d2
        const Cd n1 = {-u1.y, u1.x}, n2 = {-u2.y, u2.x};                  // times i
        a[0] = {a[0].x + p1.x + p2.x, a[0].y + p1.y + p2.y};
        a[1] = cadd(m1, n1);
        a[4] = csub(m1, n1);
        a[2] = cadd(m2, n2);
        a[3] = csub(m2, n2);
    }
};

// tw[j] = exp(-2 pi i j / N), j < N.  sincospi in double for j <= N/2 only; the upper half by conjugation.
// Ends with a barrier.
__device__ __forceinline__ void make_twiddles(Cd* tw, int N, int tid, int nthr) {
    const int half = N / 2;
    for (int j = tid; j <= half; j += nthr) {
        double s, c;
        sincospi(-2.0 * (double)j / (double)N, &s, &c);
        tw[j] = {c, s};
        if (j > 0 && N - j > half) tw[N - j] = {c, -s};
    }
    __syncthreads();
}

// One Stockham pass of radix R over `nbatch` transforms of length N (x -> y, transform b at offset b * pitch):
// current sub-length n (N = n s), butterfly t = p s + q reads x[t + j N/R], writes y[q + s (R p + k)] * w_n^{p k}.
template <int R, int SIGN>
__device__ __forceinline__ void stockham_pass(const Cd* __restrict__ x, Cd* __restrict__ y, const Cd* __restrict__ tw, int N,
                                              int s, int nbatch, int pitch, int tid, int nthr) {
    const int nb = N / R;
    const int total = nbatch * nb;
    for (int u = tid; u < total; u += nthr) {
        const int b = u / nb, t = u - b * nb;
        const int p = t / s, q = t - p * s;
        const Cd* xb = x + (size_t)b * pitch + t;
        Cd a[R];
#pragma unroll
        for (int j = 0; j < R; ++j) a[j] = xb[j * nb];
        Dft<R, SIGN>::run(a);
        const int ps = p * s;                                  // twiddle index step: w_n^{p k} = tw[p s k], p s k < N
        Cd* yb = y + (size_t)b * pitch + q + s * R * p;
        yb[0] = a[0];
#pragma unroll
        for (int k = 1; k < R; ++k) yb[s * k] = SIGN < 0 ? cmul(a[k], tw[ps * k]) : cmul_conj(a[k], tw[ps * k]);
    }
}

struct Radices { int n; int r[kFftMaxPasses]; };

// nbatch transforms of length N; input in x, scratch y; returns the buffer that holds the result.
template <int SIGN>
__device__ __forceinline__ Cd* stockham(Cd* x, Cd* y, const Cd* tw, int N, const Radices& rad, int nbatch, int pitch, int tid,
                                        int nthr) {
    int s = 1;
    for (int i = 0; i < rad.n; ++i) {
        const int R = rad.r[i];
        switch (R) {
            case 4: stockham_pass<4, SIGN>(x, y, tw, N, s, nbatch, pitch, tid, nthr); break;
            case 2: stockham_pass<2, SIGN>(x, y, tw, N, s, nbatch, pitch, tid, nthr); break;
            case 3: stockham_pass<3, SIGN>(x, y, tw, N, s, nbatch, pitch, tid, nthr); break;
            default: stockham_pass<5, SIGN>(x, y, tw, N, s, nbatch, pitch, tid, nthr); break;
        }
        __syncthreads();
        s *= R;
        Cd* t = x; x = y; y = t;
    }
    return x;
}

struct FftArgs {
    int ny, nx, ky, kx;
    int Px, Py, Ph;                  // padded sizes, Ph = Px/2 + 1 stored spectrum columns
    int nb;                          // row pairs per CTA (row kernels)
    int tc;                          // spectrum columns per CTA (column kernel)
    int n_cta_img;                   // rows_fwd: CTAs that transform image row pairs (the rest take kernel rows)
    Radices rx, ry;
    double scale;                    // 1 / (Px Py)
    int B;                           // images sharing the one kernel
    Cd *SA, *SB, *SC;                // planes [B][ny][Ph], [ky][Ph], [B][ny][Ph]
    Cd *SBF;                         // B > 1: the kernel's full 2-D spectrum [Py][Ph], scaled, transformed once
};

// ---- rows forward: pairs of real rows -> half spectra ----
template <typename T>
__global__ void __launch_bounds__(kFftMaxThreads) k_fft_rows_fwd(const __grid_constant__ FftArgs a, const T* __restrict__ img,
                                                              const T* __restrict__ ker) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.Px, tid = threadIdx.x, nthr = blockDim.x;
    Cd* x = reinterpret_cast<Cd*>(smem_raw);
    Cd* y = x + (size_t)a.nb * P;
    Cd* tw = y + (size_t)a.nb * P;
    cudaTriggerProgrammaticLaunchCompletion();                 // lets k_fft_cols start its twiddle set-up once every CTA here runs
    make_twiddles(tw, P, tid, nthr);
    const int n_img_ctas = a.n_cta_img * a.B;
    const bool is_img = (int)blockIdx.x < n_img_ctas;
    const int b_img = is_img ? (int)blockIdx.x / a.n_cta_img : 0;
    const T* src = is_img ? img + (size_t)b_img * a.ny * a.nx : ker;
    const int rows = is_img ? a.ny : a.ky, width = is_img ? a.nx : a.kx;
    Cd* plane = is_img ? a.SA + (size_t)b_img * a.ny * a.Ph : a.SB;
    const int pair0 = (is_img ? (int)blockIdx.x - b_img * a.n_cta_img : (int)blockIdx.x - n_img_ctas) * a.nb;
    for (int idx = tid; idx < a.nb * P; idx += nthr) {
        const int b = idx / P, i = idx - b * P;
        const int r0 = 2 * (pair0 + b), r1 = r0 + 1;
        Cd v = {0.0, 0.0};
        if (i < width) {
            if (r0 < rows) v.x = (double)__ldg(&src[(size_t)r0 * width + i]);
            if (r1 < rows) v.y = (double)__ldg(&src[(size_t)r1 * width + i]);
        }
        x[idx] = v;
    }
    __syncthreads();
    const Cd* X = stockham<-1>(x, y, tw, P, a.rx, a.nb, P, tid, nthr);
    for (int idx = tid; idx < a.nb * a.Ph; idx += nthr) {
        const int b = idx / a.Ph, k = idx - b * a.Ph;
        const int r0 = 2 * (pair0 + b), r1 = r0 + 1;
        if (r0 >= rows) continue;
        const Cd z = X[b * P + k], zn = X[b * P + (k == 0 ? 0 : P - k)];
        plane[(size_t)r0 * a.Ph + k] = {0.5 * (z.x + zn.x), 0.5 * (z.y - zn.y)};                 // (Z_k + conj Z_{P-k}) / 2
        if (r1 < rows) plane[(size_t)r1 * a.Ph + k] = {0.5 * (z.y + zn.y), -0.5 * (z.x - zn.x)}; // (Z_k - conj Z_{P-k}) / (2i)
    }
}

// ---- columns: forward FFTs of tc image and tc kernel spectrum columns, product, inverse FFT, crop ----
// KER_READY (batches): the kernel's columns were transformed once by k_fft_cols_ker; the product reads SBF.
template <bool KER_READY>
__global__ void __launch_bounds__(kFftMaxThreads) k_fft_cols(const __grid_constant__ FftArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.Py, tc = a.tc, tid = threadIdx.x, nthr = blockDim.x;
    constexpr int NSET = KER_READY ? 1 : 2;
    Cd* x = reinterpret_cast<Cd*>(smem_raw);                   // [NSET tc][P]: image columns, then kernel columns
    Cd* y = x + (size_t)NSET * tc * P;
    Cd* tw = y + (size_t)NSET * tc * P;
    make_twiddles(tw, P, tid, nthr);
    cudaGridDependencySynchronize();                           // the planes of the previous kernel are complete
    cudaTriggerProgrammaticLaunchCompletion();
    const int k0 = blockIdx.x * tc;
    const int ncol = min(tc, a.Ph - k0);
    const Cd* SA = a.SA + (size_t)blockIdx.y * a.ny * a.Ph;
    Cd* SC = a.SC + (size_t)blockIdx.y * a.ny * a.Ph;
    for (int idx = tid; idx < P * tc; idx += nthr) {
        const int r = idx / tc, c = idx - r * tc;
        Cd va = {0.0, 0.0}, vb = {0.0, 0.0};
        if (c < ncol) {
            if (r < a.ny) va = __ldcg(&SA[(size_t)r * a.Ph + k0 + c]);
            if (!KER_READY && r < a.ky) vb = __ldcg(&a.SB[(size_t)r * a.Ph + k0 + c]);
        }
        x[c * P + r] = va;
        if (!KER_READY) x[(tc + c) * P + r] = vb;
    }
    __syncthreads();
    Cd* X = stockham<-1>(x, y, tw, P, a.ry, NSET * tc, P, tid, nthr);
    Cd* Y = (X == x) ? y : x;
    for (int idx = tid; idx < tc * P; idx += nthr) {
        Cd c;
        if (KER_READY) {
            const int col = idx / P, r = idx - col * P;
            const Cd kf = col < ncol ? __ldcg(&a.SBF[(size_t)r * a.Ph + k0 + col]) : Cd{0.0, 0.0};
            c = cmul(X[idx], kf);
        } else {
            c = cmul(X[idx], X[tc * P + idx]);
            c.x *= a.scale;
            c.y *= a.scale;
        }
        X[idx] = c;
    }
    __syncthreads();
    const Cd* C = stockham<+1>(X, Y, tw, P, a.ry, tc, P, tid, nthr);
    const int row0 = a.ky / 2;
    for (int idx = tid; idx < a.ny * tc; idx += nthr) {
        const int j = idx / tc, c = idx - j * tc;
        if (c < ncol) SC[(size_t)j * a.Ph + k0 + c] = C[c * P + row0 + j];
    }
}

// ---- batches: column FFTs of the kernel's row spectra, once -> SBF [Py][Ph] with the 1 / (Px Py) scale ----
__global__ void __launch_bounds__(kFftMaxThreads) k_fft_cols_ker(const __grid_constant__ FftArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.Py, tc = a.tc, tid = threadIdx.x, nthr = blockDim.x;
    Cd* x = reinterpret_cast<Cd*>(smem_raw);
    Cd* y = x + (size_t)tc * P;
    Cd* tw = y + (size_t)tc * P;
    make_twiddles(tw, P, tid, nthr);
    cudaGridDependencySynchronize();                           // plane SB of k_fft_rows_fwd is complete
    cudaTriggerProgrammaticLaunchCompletion();
    const int k0 = blockIdx.x * tc;
    const int ncol = min(tc, a.Ph - k0);
    for (int idx = tid; idx < P * tc; idx += nthr) {
        const int r = idx / tc, c = idx - r * tc;
        Cd vb = {0.0, 0.0};
        if (c < ncol && r < a.ky) vb = __ldcg(&a.SB[(size_t)r * a.Ph + k0 + c]);
        x[c * P + r] = vb;
    }
    __syncthreads();
    const Cd* X = stockham<-1>(x, y, tw, P, a.ry, tc, P, tid, nthr);
    for (int idx = tid; idx < P * tc; idx += nthr) {
        const int r = idx / tc, c = idx - r * tc;
        if (c < ncol) {
            Cd v = X[c * P + r];
            v.x *= a.scale;
            v.y *= a.scale;
            a.SBF[(size_t)r * a.Ph + k0 + c] = v;
        }
    }
}

// ---- rows inverse: two output rows per inverse complex transform ----
template <typename T>
__global__ void __launch_bounds__(kFftMaxThreads) k_fft_rows_inv(const __grid_constant__ FftArgs a, T* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int P = a.Px, tid = threadIdx.x, nthr = blockDim.x;
    Cd* x = reinterpret_cast<Cd*>(smem_raw);
    Cd* y = x + (size_t)a.nb * P;
    Cd* tw = y + (size_t)a.nb * P;
    make_twiddles(tw, P, tid, nthr);
    cudaGridDependencySynchronize();                           // plane SC of k_fft_cols is complete
    const int pair0 = blockIdx.x * a.nb;
    const Cd* SC = a.SC + (size_t)blockIdx.y * a.ny * a.Ph;
    out += (size_t)blockIdx.y * a.ny * a.nx;
    for (int idx = tid; idx < a.nb * P; idx += nthr) {
        const int b = idx / P, k = idx - b * P;
        const int r0 = 2 * (pair0 + b), r1 = r0 + 1;
        Cd v = {0.0, 0.0};
        if (r0 < a.ny) {
            const bool mirror = k >= a.Ph;                     // C_k = conj C_{P-k} for k > P/2
            const int kk = mirror ? P - k : k;
            Cd ca = __ldcg(&SC[(size_t)r0 * a.Ph + kk]);
            Cd cb = {0.0, 0.0};
            if (r1 < a.ny) cb = __ldcg(&SC[(size_t)r1 * a.Ph + kk]);
            if (mirror) { ca.y = -ca.y; cb.y = -cb.y; }
            v = {ca.x - cb.y, ca.y + cb.x};                    // C_a + i C_b
        }
        x[idx] = v;
    }
    __syncthreads();
    const Cd* X = stockham<+1>(x, y, tw, P, a.rx, a.nb, P, tid, nthr);
    const int col0 = a.kx / 2;
    for (int idx = tid; idx < a.nb * a.nx; idx += nthr) {
        const int b = idx / a.nx, i = idx - b * a.nx;
        const int r0 = 2 * (pair0 + b), r1 = r0 + 1;
        if (r0 >= a.ny) continue;
        const Cd v = X[b * P + col0 + i];
        out[(size_t)r0 * a.nx + i] = (T)v.x;
        if (r1 < a.ny) out[(size_t)r1 * a.nx + i] = (T)v.y;
    }
}

// ------------------------------------------------------------------------------------------------ host side
// smallest 2^a 3^b 5^c >= v (even when `even`)
static int next_smooth(int v, bool even) {
    for (int p = v < 2 ? 2 : v;; ++p) {
        if (even && (p & 1)) continue;
        int q = p;
        while (q % 2 == 0) q /= 2;
        while (q % 3 == 0) q /= 3;
        while (q % 5 == 0) q /= 5;
        if (q == 1) return p;
    }
}

static bool factor(int P, Radices* out) {
    out->n = 0;
    int q = P;
    auto push = [&](int r) { if (out->n < kFftMaxPasses) out->r[out->n++] = r; };
    while (q % 4 == 0) { push(4); q /= 4; }
    if (q % 2 == 0) { push(2); q /= 2; }
    while (q % 3 == 0) { push(3); q /= 3; }
    while (q % 5 == 0) { push(5); q /= 5; }
    return q == 1 && out->n < kFftMaxPasses;
}

struct FftPlan {
    FftArgs a;
    size_t smem_rows, smem_cols;
    size_t plane_a, plane_b, plane_c;          // bytes, 256-aligned
    int grid_rows_fwd, grid_cols, grid_rows_inv, thr_rows, thr_cols;
    bool ok;
};

static FftPlan plan_fft(int ny, int nx, int ky, int kx, int64_t B = 1) {
    FftPlan p = {};
    p.ok = false;
    if ((int64_t)ny + ky - 1 > kFftMaxP || (int64_t)nx + kx - 1 > kFftMaxP) return p;
    FftArgs& a = p.a;
    a.ny = ny; a.nx = nx; a.ky = ky; a.kx = kx;
    a.Px = next_smooth(nx + kx - 1, true);
    a.Py = next_smooth(ny + ky - 1, false);
    if (a.Px > kFftMaxP || a.Py > kFftMaxP) return p;
    a.Ph = a.Px / 2 + 1;
    if (!factor(a.Px, &a.rx) || !factor(a.Py, &a.ry)) return p;
    a.scale = 1.0 / ((double)a.Px * (double)a.Py);
    const size_t csz = sizeof(Cd);
    // row kernels: enough butterflies per CTA for 256 threads, enough CTAs for 148 SMs
    const int pairs_img = (ny + 1) / 2, pairs_ker = (ky + 1) / 2;
    int nb = 1;
    const int64_t pairs_all = (int64_t)pairs_img * B + pairs_ker;
    // one image: short transforms share a CTA; a batch: as many row pairs per CTA as keep 4 CTAs per SM busy
    while (nb < 8 && (B > 1 || nb * a.Px < 1024) && pairs_all / (2 * nb) >= (B > 1 ? 4 : 2) * kNumSMs) nb *= 2;
    a.nb = nb;
    p.smem_rows = ((size_t)2 * nb * a.Px + a.Px) * csz;
    a.n_cta_img = (pairs_img + nb - 1) / nb;
    p.grid_rows_fwd = a.n_cta_img + (pairs_ker + nb - 1) / nb;
    p.grid_rows_inv = a.n_cta_img;
    // column kernel: 2 columns per CTA (one 32-byte sector per plane row); 4 when the transform is short
    int tc = 2;
    while (tc < 8 && (B > 1 || tc * a.Py < 512) && (int64_t)((a.Ph + 2 * tc - 1) / (2 * tc)) * B >= (B > 1 ? 4 : 1) * kNumSMs) tc *= 2;
    while (tc > 1 && ((size_t)4 * tc * a.Py + a.Py) * csz > (B > 1 ? kFftMaxSmem / 2 : kFftMaxSmem)) tc /= 2;
    a.tc = tc;
    p.smem_cols = ((size_t)(B > 1 ? 2 : 4) * tc * a.Py + a.Py) * csz;     // batches: the kernel's columns are not in the CTA
    p.grid_cols = (a.Ph + tc - 1) / tc;
    if (p.smem_rows > kFftMaxSmem || p.smem_cols > kFftMaxSmem) return p;
    // CTA sizes: about one radix-4 butterfly per thread and pass, capped where more warps only lengthen the barriers
    // (measured on B200: rows 256, columns 384-512 are best from 60^2 to 1000^2)
    auto pick_threads = [](int butterflies, int cap) { int t = (butterflies + 31) / 32 * 32; return t < 128 ? 128 : (t > cap ? cap : t); };
    p.thr_rows = pick_threads(nb * a.Px / 4, 256);
    p.thr_cols = pick_threads((B > 1 ? 1 : 2) * tc * a.Py / 4, 512);
    p.plane_a = align_up((size_t)ny * a.Ph * csz, 256);
    p.plane_b = align_up((size_t)ky * a.Ph * csz, 256);
    p.plane_c = align_up((size_t)ny * a.Ph * csz, 256);
    p.ok = true;
    return p;
}

bool conv_fft_supported(jt_dtype, int ny, int nx, int ky, int kx) { return plan_fft(ny, nx, ky, kx).ok; }
void conv_fft_describe(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx, jt_conv_plan* out) {
    const FftPlan p = plan_fft(ny, nx, ky, kx, B);
    out->method = JT_CONV_FFT;
    out->path = JT_PATH_CONV_FFT;
    out->pad_y = p.a.Py; out->pad_x = p.a.Px;
    out->est_us = conv_fft_estimate_us(d, B, ny, nx, ky, kx);
}

// A batch is transformed in groups of G images (all of it when its planes fit kFftGroupBytes of workspace).
constexpr size_t kFftGroupBytes = (size_t)2 << 30;
static int64_t fft_group(const FftPlan& p, int64_t B) {
    const size_t per = p.plane_a + p.plane_c;
    int64_t G = (int64_t)(kFftGroupBytes / (per ? per : 1));
    if (G < 1) G = 1;
    if (G > 65535) G = 65535;                       // gridDim.y
    return B < G ? B : G;
}
static size_t fft_plane_bf(const FftPlan& p, int64_t B) { return B > 1 ? align_up((size_t)p.a.Py * p.a.Ph * sizeof(Cd), 256) : 0; }

// Time model behind JT_CONV_AUTO, calibrated on B200 with bench.py --conv-sweep: dependent
// launches plus the planes' trips through L2 (one image) or HBM (a batch: the kernel's spectrum is formed once).
double conv_fft_estimate_us(jt_dtype, int64_t B, int ny, int nx, int ky, int kx) {
    const FftPlan p = plan_fft(ny, nx, ky, kx, B);
    if (!p.ok) return 1e30;
    const double mb = (double)(p.plane_a + p.plane_b + p.plane_c) * 2.0 / 1048576.0;
    if (B <= 1) return 9.0 + 1.2 * mb;
    const double mb_img = (double)(p.plane_a + p.plane_c) * 2.0 / 1048576.0;
    return 14.0 + 1.2 * mb + (double)(B - 1) * 1.3 * mb_img;   // measured: 0.77 TB/s of plane traffic (FP64 butterflies in shared memory)
}

size_t fft_conv_workspace_bytes(jt_dtype, int64_t B, int ny, int nx, int ky, int kx) {
    const FftPlan p = plan_fft(ny, nx, ky, kx, B);
    if (!p.ok) return 0;
    const int64_t G = fft_group(p, B);
    return (size_t)G * (p.plane_a + p.plane_c) + p.plane_b + fft_plane_bf(p, B);
}

template <typename K, typename... Args>
static jt_status launch_fft_kernel(K kern, dim3 grid, int threads, size_t smem, bool dependent, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = dependent ? 1 : 0;
    JT_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, args...));
    JT_LAUNCH_CHECK();
    return JT_OK;
}

// workspace: [SA: G images][SC: G images][SB][SBF (batches)]
template <typename T>
static jt_status conv_fft_t(FftPlan& p, int64_t B, const T* img, const T* ker, void* workspace, T* out, cudaStream_t st) {
    FftArgs& a = p.a;
    const int64_t G = fft_group(p, B);
    a.SA = (Cd*)workspace;
    a.SC = (Cd*)((char*)workspace + (size_t)G * p.plane_a);
    a.SB = (Cd*)((char*)workspace + (size_t)G * (p.plane_a + p.plane_c));
    a.SBF = (Cd*)((char*)a.SB + p.plane_b);
    auto k1 = k_fft_rows_fwd<T>;
    auto k2 = k_fft_cols<false>;
    auto k2r = k_fft_cols<true>;
    auto k2k = k_fft_cols_ker;
    auto k3 = k_fft_rows_inv<T>;
    static PerDeviceOnce attr;                     // once per instantiation and device: allow the full dynamic shared memory
    if (attr.needed()) {
        JT_CUDA_TRY(cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFftMaxSmem));
        JT_CUDA_TRY(cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFftMaxSmem));
        JT_CUDA_TRY(cudaFuncSetAttribute(k2r, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFftMaxSmem));
        JT_CUDA_TRY(cudaFuncSetAttribute(k2k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFftMaxSmem));
        JT_CUDA_TRY(cudaFuncSetAttribute(k3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kFftMaxSmem));
        attr.mark();
    }
    const int ker_ctas = p.grid_rows_fwd - a.n_cta_img;
    const size_t img_elems = (size_t)a.ny * a.nx;
    for (int64_t b0 = 0; b0 < B; b0 += G) {
        const int g = (int)(B - b0 < G ? B - b0 : G);
        a.B = g;
        // the kernel's rows ride the first group's row pass (its CTAs come after the images'); later groups reuse SB / SBF
        const int rows_grid = a.n_cta_img * g + (b0 == 0 ? ker_ctas : 0);
        jt_status s = launch_fft_kernel(k1, dim3((unsigned)rows_grid), p.thr_rows, p.smem_rows, false, st, a, img + b0 * img_elems, ker);
        if (s != JT_OK) return s;
        if (B > 1) {
            if (b0 == 0) {
                s = launch_fft_kernel(k2k, dim3((unsigned)p.grid_cols), p.thr_cols, p.smem_cols, true, st, a);
                if (s != JT_OK) return s;
            }
            s = launch_fft_kernel(k2r, dim3((unsigned)p.grid_cols, (unsigned)g), p.thr_cols, p.smem_cols, true, st, a);
        } else {
            s = launch_fft_kernel(k2, dim3((unsigned)p.grid_cols, 1u), p.thr_cols, p.smem_cols, true, st, a);
        }
        if (s != JT_OK) return s;
        s = launch_fft_kernel(k3, dim3((unsigned)p.grid_rows_inv, (unsigned)g), p.thr_rows, p.smem_rows, true, st, a, out + b0 * img_elems);
        if (s != JT_OK) return s;
    }
    return JT_OK;
}

jt_status launch_conv_fft(jt_dtype dtype, int64_t B, int ny, int nx, const void* img, int ky, int kx, const void* ker,
                          void* workspace, void* out, cudaStream_t st) {
    FftPlan p = plan_fft(ny, nx, ky, kx, B);
    if (!p.ok) return JT_ERR_UNSUPPORTED;
    return dtype == JT_F32 ? conv_fft_t<float>(p, B, (const float*)img, (const float*)ker, workspace, (float*)out, st)
                           : conv_fft_t<double>(p, B, (const double*)img, (const double*)ker, workspace, (double*)out, st);
}

}  // namespace jt
