// jt_fft.cu -- step 5b: PSF convolution by hand-written shared-memory FFTs (definition P; PAPER.md:110-114
// "FFT convolution").  Reaches the direct-convolution result up to rounding.  cuFFT is not used (tests only).
//
// Both inputs are real, so ONE complex transform carries both: z = img + i ker (zero-padded to Py x Px, powers of
// two >= n + K - 1), Z = FFT2(z);  A = FFT2(img) = (Z(k) + conj Z(-k))/2,  B = FFT2(ker) = (Z(k) - conj Z(-k))/(2i);
// C = A B is Hermitian, out = Re IFFT2(C) cropped at (ky/2, kx/2).
//
// Forward transforms are decimation-in-frequency (natural order in, bit-reversed positions out; two radix-2 stages
// fused per shared-memory pass), inverse
// transforms decimation-in-time with conjugate twiddles (bit-reversed positions in, natural order out), so no
// permutation pass exists anywhere: position p of an axis holds frequency brev(p), and the pointwise step pairs
// position (py, px) with (brev(-brev py), brev(-brev px)).
//
// Four launches on the caller's stream, one complex plane [Py][Px] in the caller's workspace (L2-resident):
//   k_fft_sums     : sum|img|, sum|ker| partial sums (scale balance of the packed transform, see below)
//   k_fft_rows_fwd : pack img + i ker, row FFTs; only the max(ny, ky) non-zero rows are computed and stored
//   k_fft_cols     : a CTA owns a group of adjacent position-columns and the group holding their -kx partners:
//                    column FFTs, pointwise product (both members of a +-k pair at once), inverse column FFTs,
//                    all in shared memory; stores only the ny rows the crop keeps
//   k_fft_rows_inv : inverse row FFTs of those rows, crop, real part -> out
#include "jt_internal.h"

namespace jt {

// Packing the two real inputs into one complex transform couples their spectra: B is recovered with an absolute
// error of eps |A|, i.e. eps sum|img| / sum|ker| relative.  Two measures keep that at rounding level:
//   (1) the kernel is packed as lambda ker with lambda = the power of two nearest sum|img| / sum|ker| (k_fft_sums
//       writes per-CTA partial sums, every later CTA adds them in the same order: deterministic, no atomics);
//   (2) the transforms run in double in BOTH dtype modes (JT_F32 converts on load and store only).
// The path is bound by launch latency and L2 traffic, not by the FP64 pipe.
using Cd = double2;
constexpr int kFftSumCtas = 64;        // partial sums: [2][kFftSumCtas] doubles behind the plane

constexpr int kFftRowThreads = 256;
constexpr int kFftColThreads = 512;
constexpr size_t kFftMaxSmem = 220 * 1024;

__host__ __device__ inline int ilog2(int v) { int l = 0; while ((1 << l) < v) ++l; return l; }
static int next_pow2(int v, int lo) { int p = lo; while (p < v) p <<= 1; return p; }

__device__ __forceinline__ Cd cmul(Cd a, Cd b) { return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x}; }
__device__ __forceinline__ Cd cmul_conj(Cd a, Cd b) { return {a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y}; }  // a conj(b)

__device__ __forceinline__ int brev_bits(int v, int bits) { return (int)(__brev((unsigned)v) >> (32 - bits)); }

// tw[m] = exp(-2 pi i m / n), m < n/2, from sincospi in double (m/n is exact for a power of two)
__device__ __forceinline__ void make_twiddles(Cd* tw, int n, int tid, int nthr) {
    for (int m = tid; m < n / 2; m += nthr) {
        double s, c;
        sincospi(-2.0 * (double)m / (double)n, &s, &c);
        tw[m] = {c, s};
    }
}

// nb transforms of length n = 2^logn at s + b * pitch.  Forward, decimation in frequency.  Two radix-2 stages are
// fused per pass (a thread carries four points through both in registers: half the shared-memory traffic and half the
// barriers of a stage-by-stage sweep, identical arithmetic); an odd logn ends with one plain radix-2 stage.
__device__ __forceinline__ void fft_dif(Cd* s, const Cd* tw, int logn, int nb, int pitch, int tid, int nthr) {
    int lh = logn - 1;
    for (; lh >= 1; lh -= 2) {                       // stages with half-sizes h = 2^lh and q = h/2
        const int h = 1 << lh, q = h >> 1;
        const int quarter = 1 << (logn - 2);
        const int total = nb * quarter;
        for (int u = tid; u < total; u += nthr) {
            const int tr = u >> (logn - 2), uu = u & (quarter - 1);
            const int k = uu & (q - 1), g = uu >> (lh - 1);
            const int i0 = tr * pitch + (g << (lh + 1)) + k, i1 = i0 + q, i2 = i0 + h, i3 = i2 + q;
            const Cd x0 = s[i0], x1 = s[i1], x2 = s[i2], x3 = s[i3];
            const Cd wa = tw[k << (logn - 1 - lh)], wb = tw[(k + q) << (logn - 1 - lh)], wc = tw[k << (logn - lh)];
            const Cd a0 = {x0.x + x2.x, x0.y + x2.y};
            const Cd a2 = cmul({x0.x - x2.x, x0.y - x2.y}, wa);
            const Cd a1 = {x1.x + x3.x, x1.y + x3.y};
            const Cd a3 = cmul({x1.x - x3.x, x1.y - x3.y}, wb);
            s[i0] = {a0.x + a1.x, a0.y + a1.y};
            s[i1] = cmul({a0.x - a1.x, a0.y - a1.y}, wc);
            s[i2] = {a2.x + a3.x, a2.y + a3.y};
            s[i3] = cmul({a2.x - a3.x, a2.y - a3.y}, wc);
        }
        __syncthreads();
    }
    if (lh == 0) {                                   // last stage, h = 1, twiddle 1
        const int half = 1 << (logn - 1);
        const int total = nb * half;
        for (int b = tid; b < total; b += nthr) {
            const int tr = b >> (logn - 1), bb = b & (half - 1);
            const int i = tr * pitch + (bb << 1), j = i + 1;
            const Cd a = s[i], c = s[j];
            s[i] = {a.x + c.x, a.y + c.y};
            s[j] = cmul({a.x - c.x, a.y - c.y}, tw[0]);
        }
        __syncthreads();
    }
}

// Inverse of fft_dif stage by stage (unnormalised: fft_dit_inv(fft_dif(x)) = n x), the stages fused in pairs likewise.
__device__ __forceinline__ void fft_dit_inv(Cd* s, const Cd* tw, int logn, int nb, int pitch, int tid, int nthr) {
    int lh = 0;
    if (logn & 1) {                                  // undo fft_dif's last stage first (h = 1)
        const int half = 1 << (logn - 1);
        const int total = nb * half;
        for (int b = tid; b < total; b += nthr) {
            const int tr = b >> (logn - 1), bb = b & (half - 1);
            const int i = tr * pitch + (bb << 1), j = i + 1;
            const Cd a = s[i];
            const Cd c = cmul_conj(s[j], tw[0]);
            s[i] = {a.x + c.x, a.y + c.y};
            s[j] = {a.x - c.x, a.y - c.y};
        }
        __syncthreads();
        lh = 1;
    }
    for (; lh + 1 < logn; lh += 2) {                 // stages with half-sizes h = 2^lh and 2h
        const int h = 1 << lh;
        const int quarter = 1 << (logn - 2);
        const int total = nb * quarter;
        for (int u = tid; u < total; u += nthr) {
            const int tr = u >> (logn - 2), uu = u & (quarter - 1);
            const int k = uu & (h - 1), g = uu >> lh;
            const int i0 = tr * pitch + (g << (lh + 2)) + k, i1 = i0 + h, i2 = i1 + h, i3 = i2 + h;
            const Cd x0 = s[i0], x2 = s[i2];
            const Cd w1 = tw[k << (logn - 1 - lh)];
            const Cd c1 = cmul_conj(s[i1], w1), c3 = cmul_conj(s[i3], w1);
            const Cd b0 = {x0.x + c1.x, x0.y + c1.y}, b1 = {x0.x - c1.x, x0.y - c1.y};
            const Cd b2 = {x2.x + c3.x, x2.y + c3.y}, b3 = {x2.x - c3.x, x2.y - c3.y};
            const Cd d2 = cmul_conj(b2, tw[k << (logn - 2 - lh)]);
            const Cd d3 = cmul_conj(b3, tw[(k + h) << (logn - 2 - lh)]);
            s[i0] = {b0.x + d2.x, b0.y + d2.y};
            s[i2] = {b0.x - d2.x, b0.y - d2.y};
            s[i1] = {b1.x + d3.x, b1.y + d3.y};
            s[i3] = {b1.x - d3.x, b1.y - d3.y};
        }
        __syncthreads();
    }
}

// partial[c] = sum |img| over CTA c's slice, partial[kFftSumCtas + c] = the same for ker
template <typename T>
__global__ void __launch_bounds__(256) k_fft_sums(int64_t n_img, const T* __restrict__ img, int64_t n_ker,
                                                  const T* __restrict__ ker, double* __restrict__ partial) {
    __shared__ double red[2][8];
    double a = 0.0, b = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n_img; i += (int64_t)gridDim.x * 256) a += fabs((double)__ldg(&img[i]));
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n_ker; i += (int64_t)gridDim.x * 256) b += fabs((double)__ldg(&ker[i]));
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = a; red[1][threadIdx.x >> 5] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double sa = 0.0, sb = 0.0;
        for (int w = 0; w < 8; ++w) { sa += red[0][w]; sb += red[1][w]; }
        partial[blockIdx.x] = sa;
        partial[kFftSumCtas + blockIdx.x] = sb;
    }
}

// lambda = 2^round(log2(sum|img| / sum|ker|)), 1 when either sum is zero or not finite
__device__ __forceinline__ double fft_lambda(const double* __restrict__ partial, int n_part) {
    double sa = 0.0, sb = 0.0;
    for (int c = 0; c < n_part; ++c) { sa += partial[c]; sb += partial[kFftSumCtas + c]; }
    if (!(sa > 0.0) || !(sb > 0.0) || !isfinite(sa) || !isfinite(sb)) return 1.0;
    int ea, eb;
    frexp(sa, &ea);
    frexp(sb, &eb);
    int d = ea - eb;
    d = d > 1000 ? 1000 : (d < -1000 ? -1000 : d);
    return ldexp(1.0, d);
}

template <typename T>
__global__ void __launch_bounds__(kFftRowThreads) k_fft_rows_fwd(int ny, int nx, const T* __restrict__ img, int ky, int kx,
                                                                 const T* __restrict__ ker, int logPx, int rows_nz, int nb,
                                                                 const double* __restrict__ partial, int n_part,
                                                                 Cd* __restrict__ plane) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int Px = 1 << logPx;
    Cd* s = reinterpret_cast<Cd*>(smem_raw);
    Cd* tw = s + (size_t)nb * Px;
    const int tid = threadIdx.x;
    make_twiddles(tw, Px, tid, kFftRowThreads);
    const double lambda = fft_lambda(partial, n_part);
    const int r0 = blockIdx.x * nb;
    for (int idx = tid; idx < nb * Px; idx += kFftRowThreads) {
        const int r = r0 + (idx >> logPx), x = idx & (Px - 1);
        const T re = (r < ny && x < nx) ? __ldg(&img[(size_t)r * nx + x]) : (T)0;
        const T im = (r < ky && x < kx) ? __ldg(&ker[(size_t)r * kx + x]) : (T)0;
        s[idx] = {(double)re, lambda * (double)im};
    }
    __syncthreads();
    fft_dif(s, tw, logPx, nb, Px, tid, kFftRowThreads);
    for (int idx = tid; idx < nb * Px; idx += kFftRowThreads) {
        const int r = r0 + (idx >> logPx);
        if (r < rows_nz) plane[(size_t)r * Px + (idx & (Px - 1))] = s[idx];
    }
}

// tb = log2(columns per group).  CTA kc in [0, Px/(2 TC)] owns the position group whose bit-reversed index is kc and
// the group holding its -kx partners (the same group when kc = 0 or kc = Px/(2 TC)).
__global__ void __launch_bounds__(kFftColThreads) k_fft_cols(int logPx, int logPy, int tb, int rows_nz, int row_out0,
                                                             int n_rows_out, double scale, const double* __restrict__ partial,
                                                             int n_part, Cd* __restrict__ plane) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int Px = 1 << logPx, Py = 1 << logPy, TC = 1 << tb;
    const int pitch = Py + 1;                      // odd pitch: the TC columns of one row land in different banks
    const int gbits = logPx - tb;                  // bits of a group index
    const int kc = blockIdx.x;
    const int n_groups = 1 << gbits;
    const int kcp = (n_groups - kc) & (n_groups - 1);
    const bool self = (kcp == kc);
    const int cA = gbits > 0 ? brev_bits(kc, gbits) : 0;
    const int cB = gbits > 0 ? brev_bits(kcp, gbits) : 0;
    const int ncol = self ? TC : 2 * TC;
    const int lcol = self ? tb : tb + 1;
    Cd* s = reinterpret_cast<Cd*>(smem_raw);
    Cd* tw = s + (size_t)2 * TC * pitch;
    const int tid = threadIdx.x;
    make_twiddles(tw, Py, tid, kFftColThreads);
    scale /= fft_lambda(partial, n_part);          // exact: lambda is a power of two

    for (int idx = tid; idx < (Py << lcol); idx += kFftColThreads) {
        const int r = idx >> lcol, lc = idx & (ncol - 1);
        const int px = (lc < TC ? cA : cB) * TC + (lc & (TC - 1));
        Cd v = {0.0, 0.0};
        if (r < rows_nz) v = plane[(size_t)r * Px + px];
        s[lc * pitch + r] = v;
    }
    __syncthreads();
    fft_dif(s, tw, logPy, ncol, pitch, tid, kFftColThreads);

    // pointwise product; the thread that owns the smaller linear index of a (+k, -k) pair writes both members
    for (int idx = tid; idx < (Py << lcol); idx += kFftColThreads) {
        const int lc = idx >> logPy, py = idx & (Py - 1);
        const int px = (lc < TC ? cA : cB) * TC + (lc & (TC - 1));
        const int pxp = brev_bits((Px - brev_bits(px, logPx)) & (Px - 1), logPx);
        const int pyp = brev_bits((Py - brev_bits(py, logPy)) & (Py - 1), logPy);
        const int lcp = ((pxp >> tb) == cA ? 0 : TC) + (pxp & (TC - 1));
        const int id = lc * pitch + py, idp = lcp * pitch + pyp;
        if (id <= idp) {
            const Cd z = s[id], zp = s[idp];
            const Cd A = {0.5 * (z.x + zp.x), 0.5 * (z.y - zp.y)};      // (Z + conj Z')/2
            const Cd Bk = {0.5 * (z.y + zp.y), -0.5 * (z.x - zp.x)};    // (Z - conj Z')/(2i)
            Cd c = cmul(A, Bk);
            c.x *= scale; c.y *= scale;
            s[id] = c;
            s[idp] = {c.x, -c.y};
        }
    }
    __syncthreads();
    fft_dit_inv(s, tw, logPy, ncol, pitch, tid, kFftColThreads);

    for (int idx = tid; idx < (n_rows_out << lcol); idx += kFftColThreads) {
        const int r = row_out0 + (idx >> lcol), lc = idx & (ncol - 1);
        const int px = (lc < TC ? cA : cB) * TC + (lc & (TC - 1));
        plane[(size_t)r * Px + px] = s[lc * pitch + r];
    }
}

template <typename T>
__global__ void __launch_bounds__(kFftRowThreads) k_fft_rows_inv(int ny, int nx, int logPx, int row_out0, int col_out0,
                                                                 int nb, const Cd* __restrict__ plane, T* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int Px = 1 << logPx;
    Cd* s = reinterpret_cast<Cd*>(smem_raw);
    Cd* tw = s + (size_t)nb * Px;
    const int tid = threadIdx.x;
    make_twiddles(tw, Px, tid, kFftRowThreads);
    const int j0 = blockIdx.x * nb;
    for (int idx = tid; idx < nb * Px; idx += kFftRowThreads) {
        const int j = j0 + (idx >> logPx);
        Cd v = {0.0, 0.0};
        if (j < ny) v = plane[(size_t)(row_out0 + j) * Px + (idx & (Px - 1))];
        s[idx] = v;
    }
    __syncthreads();
    fft_dit_inv(s, tw, logPx, nb, Px, tid, kFftRowThreads);
    for (int idx = tid; idx < nb * nx; idx += kFftRowThreads) {
        const int b = idx / nx, i = idx - b * nx;
        const int j = j0 + b;
        if (j < ny) out[(size_t)j * nx + i] = (T)s[b * Px + col_out0 + i].x;
    }
}

struct FftPlan {
    int Px, Py, logPx, logPy, tb, nb;
    size_t smem_rows, smem_cols, plane_bytes;
    bool ok;
};

static FftPlan plan_fft(jt_dtype d, int ny, int nx, int ky, int kx) {
    FftPlan p = {};
    const size_t csz = sizeof(Cd);
    (void)d;
    if ((int64_t)ny + ky - 1 > (1 << 14) || (int64_t)nx + kx - 1 > (1 << 14)) return p;
    p.Px = next_pow2(nx + kx - 1, 16);
    p.Py = next_pow2(ny + ky - 1, 16);
    p.logPx = ilog2(p.Px);
    p.logPy = ilog2(p.Py);
    p.nb = 1;
    while (p.nb < 8 && (size_t)(2 * p.nb) * p.Px <= 1024) p.nb *= 2;
    p.smem_rows = ((size_t)p.nb * p.Px + p.Px / 2) * csz;
    p.tb = -1;
    for (int tb = 2; tb >= 0; --tb) {
        const size_t sm = ((size_t)2 * (1 << tb) * (p.Py + 1) + p.Py / 2) * csz;
        if (sm <= kFftMaxSmem && p.Px >= 2 * (1 << tb)) { p.tb = tb; p.smem_cols = sm; break; }
    }
    p.plane_bytes = (size_t)p.Px * p.Py * csz;
    p.ok = p.tb >= 0 && p.smem_rows <= kFftMaxSmem;
    return p;
}

bool conv_fft_supported(jt_dtype d, int ny, int nx, int ky, int kx) { return plan_fft(d, ny, nx, ky, kx).ok; }

// Time model behind JT_CONV_AUTO (bench.py --conv-sweep on B200: P = 128: 17 us, 256: 21.5, 512: 34, 1024: 77, 2048: 305;
// beyond 1024 x 1024 the 16 B/point plane no longer sits comfortably in L2)
double conv_fft_estimate_us(jt_dtype d, int ny, int nx, int ky, int kx) {
    const FftPlan p = plan_fft(d, ny, nx, ky, kx);
    if (!p.ok) return 1e30;
    const double area = (double)p.Px * p.Py / 1048576.0;
    return 1.17 * (p.logPx + p.logPy) + 54.0 * area + (area > 1.0 ? 20.0 * (area - 1.0) : 0.0);
}

size_t fft_conv_workspace_bytes(jt_dtype d, int ny, int nx, int ky, int kx) {
    const FftPlan p = plan_fft(d, ny, nx, ky, kx);
    return p.ok ? align_up(p.plane_bytes, 256) + 2 * kFftSumCtas * sizeof(double) : 0;
}

template <typename T>
static jt_status conv_fft_t(const FftPlan& p, int ny, int nx, const T* img, int ky, int kx, const T* ker, void* workspace,
                            T* out, cudaStream_t st) {
    Cd* plane = (Cd*)workspace;
    double* partial = (double*)((char*)workspace + align_up(p.plane_bytes, 256));
    const int rows_nz = ny > ky ? ny : ky;
    const int64_t n_img = (int64_t)ny * nx, n_ker = (int64_t)ky * kx;
    int n_part = (int)((n_img + 4095) / 4096);
    n_part = n_part < 1 ? 1 : (n_part > kFftSumCtas ? kFftSumCtas : n_part);
    k_fft_sums<T><<<n_part, 256, 0, st>>>(n_img, img, n_ker, ker, partial);
    JT_LAUNCH_CHECK();
    auto k1 = k_fft_rows_fwd<T>;
    auto k2 = k_fft_cols;
    auto k3 = k_fft_rows_inv<T>;
    JT_CUDA_TRY(cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_rows));
    JT_CUDA_TRY(cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_cols));
    JT_CUDA_TRY(cudaFuncSetAttribute(k3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_rows));
    k1<<<(rows_nz + p.nb - 1) / p.nb, kFftRowThreads, p.smem_rows, st>>>(ny, nx, img, ky, kx, ker, p.logPx, rows_nz, p.nb, partial, n_part, plane);
    JT_LAUNCH_CHECK();
    const int n_cta = (p.Px >> (p.tb + 1)) + 1;
    const double scale = 1.0 / ((double)p.Px * (double)p.Py);
    k2<<<n_cta, kFftColThreads, p.smem_cols, st>>>(p.logPx, p.logPy, p.tb, rows_nz, ky / 2, ny, scale, partial, n_part, plane);
    JT_LAUNCH_CHECK();
    k3<<<(ny + p.nb - 1) / p.nb, kFftRowThreads, p.smem_rows, st>>>(ny, nx, p.logPx, ky / 2, kx / 2, p.nb, plane, out);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

jt_status launch_conv_fft(jt_dtype dtype, int ny, int nx, const void* img, int ky, int kx, const void* ker, void* workspace,
                          void* out, cudaStream_t st) {
    const FftPlan p = plan_fft(dtype, ny, nx, ky, kx);
    if (!p.ok) return JT_ERR_UNSUPPORTED;
    return dtype == JT_F32 ? conv_fft_t<float>(p, ny, nx, (const float*)img, ky, kx, (const float*)ker, workspace, (float*)out, st)
                           : conv_fft_t<double>(p, ny, nx, (const double*)img, ky, kx, (const double*)ker, workspace, (double*)out, st);
}

}  // namespace jt
