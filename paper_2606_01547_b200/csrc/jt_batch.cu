// jt_batch.cu -- jt_simulate_batch: B independent lens systems in ONE launch (PAPER.md:47 training-set
// generation; BASELINE.json configs[3]).
//
// One CTA of 256 threads per system runs the whole pipeline on chip:
//   per-system parameters -> derived once into shared memory (definition E, SubRec records of T, flipped PSF)
//   for every ray tile of the system's grid: subhalo sum over the staged records (registers), SIE + shear,
//       lens equation, Sersic, s x s warp-shuffle binning -> pre-PSF pixel into a zero-haloed shared image
//   direct convolution (definition P) out of that shared image with the register-window sweep of jt_conv.cuh
//   one coalesced HBM write of the final image.
// HBM traffic per system is its parameters in and its image out; nothing intermediate leaves the SM.
#include "jt_conv.cuh"
#include "jt_trace.cuh"

namespace jt {

constexpr int kBatchRecCap = 512;            // subhalo records resident per staging round (float; 256 in double)
template <typename T> struct BatchRecCap { static constexpr int value = sizeof(T) == 8 ? 256 : 512; };
constexpr int kBatchVar = 2;                 // subhalo_tile_sorted variant (jt_trace.cuh): the batch kernel's code must stay small
constexpr int kBatchTW = 64;                 // convolution pass: 64 columns (32 lanes x 2) x 8 warps * OY rows
template <typename T> struct BatchOY { static constexpr int value = sizeof(T) == 4 ? 8 : 4; };   // as in jt_conv.cu

template <typename T>
struct BatchArgs {
    int nx, ny, s, NX, NY;
    double hh, cx, cy, area_over_s2;
    int cols_per_warp, wtiles_x, n_wt, n_tiles;
    int M, n_src, ky, kx, kyp;
    int pw, ph, img_elems;                   // padded shared image: pw columns, ph rows; elements rounded up to 16 B
    int rec_cap;
    int dacc_off;                            // byte offset of the DAcc columns (float mode), 16-byte aligned
    const T *sie, *shear, *tnfw, *sersic, *psf;
    T* out;                                  // [B][ny][nx] or nullptr (chi^2 only)
    const T *data, *sigma;                   // chi^2 mode (jt_simulate_batch_chi2): [ny][nx] each, else nullptr
    double* chi2;                            // [B]
};

template <typename T, int R, int VAR>
__global__ void __launch_bounds__(kBatchThreads, sizeof(T) == 4 ? 2 : 1) k_batch(const __grid_constant__ BatchArgs<T> a) {
    extern __shared__ __align__(32) unsigned char smem_raw[];      // SubRec<double> is 32-byte aligned
    __shared__ MacroLens s_m;
    __shared__ SrcSet s_src;
    __shared__ int s_next;                         // next warp tile to hand out
    __shared__ unsigned short s_queue[kBatchThreads / 32][2 * kBatchRecCap];

    SubRec<T>* recs = reinterpret_cast<SubRec<T>*>(smem_raw);
    T* img = reinterpret_cast<T*>(smem_raw + (size_t)a.rec_cap * sizeof(SubRec<T>));
    T* Kc = img + a.img_elems;
    double2* dacc = reinterpret_cast<double2*>(smem_raw + a.dacc_off);       // float mode only

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t b = blockIdx.x;
    const bool conv = a.ky > 0;
    const int hy = a.ky / 2, hx = a.kx / 2;

    // ---- per-system derived parameters ----
    if (tid == 0) {
        const T* p = a.sie + b * 5;
        const T* g = a.shear + b * 2;
        s_m = derive_macro(1, (double)p[0], (double)p[1], (double)p[2], (double)p[3], (double)p[4], 1, (double)g[0],
                           (double)g[1]);
    }
    if (tid == 32) { s_src.n = a.n_src; s_next = 0; }
    if (tid >= 32 && tid < 32 + a.n_src) {
        const int k = tid - 32;
        const T* q = a.sersic + (b * a.n_src + k) * 7;
        derive_source(s_src, k, (double)q[0], (double)q[1], (double)q[2], (double)q[3], (double)q[4], (double)q[5],
                      (double)q[6]);
    }
    if (conv) {
        for (int i = tid; i < a.pw * a.ph; i += kBatchThreads) img[i] = (T)0;
        stage_taps<T>(Kc, a.psf + b * (int64_t)a.ky * a.kx, a.ky, a.kx, a.kyp, 0, (a.kx + 1) / 2, tid, kBatchThreads);
    }
    const RawTn<T> raw = {{a.tnfw + (b * 5 + 0) * a.M, a.tnfw + (b * 5 + 1) * a.M, a.tnfw + (b * 5 + 2) * a.M,
                           a.tnfw + (b * 5 + 3) * a.M, a.tnfw + (b * 5 + 4) * a.M}};
    const bool resident = a.M <= a.rec_cap;        // the whole subhalo list is staged once
    if (resident) {
        for (int k = tid; k < a.M; k += kBatchThreads)
            recs[k] = make_rec<T>((double)raw.p[0][k], (double)raw.p[1][k], (double)raw.p[2][k], (double)raw.p[3][k],
                                  (double)raw.p[4][k]);
    }
    __syncthreads();

    // ---- ray tiles: steps 1-4 ----
    T* gout = a.out ? a.out + b * (int64_t)a.ny * a.nx : nullptr;
    double chi = 0.0;                              // this thread's share of chi^2 (NEXT-3), summed per block at the end
    const T* cdata = a.data;
    const T* csigma = a.sigma;
    const int onx = a.nx;
    auto emit = [&chi, gout, cdata, csigma, onx](int j, int i, T v) {       // a finished pixel of the final image
        const int64_t p = (int64_t)j * onx + i;
        if (gout) gout[p] = v;
        if (cdata) {
            const double r = ((double)v - (double)__ldg(&cdata[p])) / (double)__ldg(&csigma[p]);
            chi = fma(r, r, chi);
        }
    };
    // Warp tiles are handed out dynamically (a shared counter): a warp whose tiles hold subhalo cores takes fewer of
    // them, so the warps reach the barrier in front of the convolution together.  A pixel's value does not depend on
    // which warp forms it; only the chi^2 of the no-PSF path sums per thread in tile order, so that path deals statically.
    const bool dynamic = !resident ? false : (conv || a.chi2 == nullptr);
    for (int tile = 0;; ++tile) {
        int wt = tile * (kBatchThreads / 32) + warp;
        if (dynamic) {
            if (lane == 0) wt = atomicAdd(&s_next, 1);
            wt = __shfl_sync(0xffffffffu, wt, 0);
            if (wt >= a.n_wt) break;
        } else if (tile >= a.n_tiles) {
            break;
        }
        RayGeom g = {a.hh, a.cx, a.cy, a.NX, a.NY, a.NX, a.NY};     // idle warp: clamped coordinates, no stores
        if (wt < a.n_wt) {
            g.I = (wt % a.wtiles_x) * a.cols_per_warp + lane;
            g.J0 = (wt / a.wtiles_x) * R;
        }
        T xs[R], ys[R];
        T x = (T)g.xd();
        pin(x);
#pragma unroll
        for (int r = 0; r < R; ++r) { xs[r] = x; ys[r] = (T)g.yd(r); pin(ys[r]); }
        DAcc<T, R, kBatchThreads> acc;
        acc.init(dacc + tid);
        TierCount tiers = {};
        WarpBox<T> box;
        box.xlo = __shfl_sync(0xffffffffu, xs[0], 0);
        box.xhi = __shfl_sync(0xffffffffu, xs[0], 31);      // columns ascend with the lane (clamped at the grid edge)
        box.ylo = ys[0];
        box.yhi = ys[R - 1];

        if (resident) {
            subhalo_tile_sorted<T, R, kBatchThreads, VAR>(recs, a.M, kBatchRecCap, 0, raw, g, box, xs, ys, acc, s_queue[warp], tiers);
        } else {
            for (int base = 0; base < a.M; base += a.rec_cap) {
                const int count = min(a.rec_cap, a.M - base);
                __syncthreads();
                for (int k = tid; k < count; k += kBatchThreads)
                    recs[k] = make_rec<T>((double)raw.p[0][base + k], (double)raw.p[1][base + k],
                                          (double)raw.p[2][base + k], (double)raw.p[3][base + k],
                                          (double)raw.p[4][base + k]);
                __syncthreads();
                subhalo_tile_sorted<T, R, kBatchThreads, VAR>(recs, count, kBatchRecCap, base, raw, g, box, xs, ys, acc, s_queue[warp], tiers);
            }
        }
        double axd[R], ayd[R];
        acc.result(axd, ayd);
        if (conv) {
            const int pw = a.pw;
            grid_epilogue<T, R>(s_m, s_src, g, a.s, a.cols_per_warp, a.area_over_s2, lane, axd, ayd,
                                [img, pw, hy, hx](int j, int i, double v) { img[(j + hy) * pw + (i + hx)] = (T)v; });
        } else {
            grid_epilogue<T, R>(s_m, s_src, g, a.s, a.cols_per_warp, a.area_over_s2, lane, axd, ayd,
                                [&emit](int j, int i, double v) { emit(j, i, (T)v); });
        }
    }
    if (conv) {
    __syncthreads();

    // ---- step 5a out of shared memory: passes of 64 columns x 64 rows, OY x 2 outputs per thread ----
    constexpr int kBatchOY = BatchOY<T>::value;
    constexpr int TH = (kBatchThreads / 32) * kBatchOY;
    const int npairs = (a.kx + 1) / 2;
    for (int j0 = 0; j0 < a.ny; j0 += TH) {
        for (int i0 = 0; i0 < a.nx; i0 += kBatchTW) {
            ConvAcc<T, kBatchOY> acc;
            acc.zero();
            acc.template sweep<false>(img + (size_t)(j0 + warp * kBatchOY) * a.pw + i0 + 2 * lane, a.pw, Kc, a.kyp, npairs);
            const int i = i0 + 2 * lane;
#pragma unroll
            for (int r = 0; r < kBatchOY; ++r) {
                const int j = j0 + warp * kBatchOY + r;
                if (j < a.ny) {
                    if (i < a.nx) emit(j, i, acc.col0(r));
                    if (i + 1 < a.nx) emit(j, i + 1, acc.col1(r));
                }
            }
        }
    }
    }
    if (a.chi2 != nullptr) {                       // fixed summation tree: lanes, then the 8 warps in order
        __shared__ double s_red[kBatchThreads / 32];
        for (int o = 16; o > 0; o >>= 1) chi += __shfl_xor_sync(0xffffffffu, chi, o);
        if (lane == 0) s_red[warp] = chi;
        __syncthreads();
        if (tid == 0) {
            double tot = 0.0;
            for (int w = 0; w < kBatchThreads / 32; ++w) tot += s_red[w];
            a.chi2[b] = tot;
        }
    }
}

constexpr size_t kBatchMaxSmem = 227 * 1024 - 4096 - 16384;      // static MacroLens + SrcSet live beside the dynamic part

template <typename T>
static size_t batch_smem_front(const BatchArgs<T>& a) {
    return align_up((size_t)a.rec_cap * sizeof(SubRec<T>) + ((size_t)a.img_elems + (size_t)4 * ((a.kx + 1) / 2) * a.kyp) * sizeof(T), 16);
}

#define JT_BATCH_CASE(RR)                                                                              \
    case RR: {                                                                                         \
        auto kern = k_batch<T, RR, kBatchVar>;                                                         \
        static PerDeviceOnce attr;   /* once per instantiation and device: allow the full dynamic shared memory */ \
        if (attr.needed()) {                                                                           \
            JT_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kBatchMaxSmem)); \
            attr.mark();                                                                               \
        }                                                                                              \
        kern<<<(unsigned)B, kBatchThreads, smem, st>>>(a);                                             \
        break;                                                                                         \
    }

template <typename T>
static jt_status batch_t(jt_dtype dtype, int64_t B, const jt_grid* g, const jt_batch_params* p, void* out,
                         const void* data, const void* sigma, double* chi2, cudaStream_t st) {
    if (B > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    const TracePlan plan = plan_trace_grid(dtype, g, 1 << 20);      // warp-tile geometry with the register-blocked ray count
    BatchArgs<T> a = {};
    const int s = g->supersample;
    a.nx = g->nx; a.ny = g->ny; a.s = s; a.NX = g->nx * s; a.NY = g->ny * s;
    a.hh = 0.5 * (g->pixel_scale / (double)s);
    a.cx = g->cx;
    a.cy = g->cy;
    a.area_over_s2 = g->pixel_scale * g->pixel_scale / ((double)s * (double)s);
    a.cols_per_warp = plan.cols_per_warp;
    a.wtiles_x = plan.tiles_x; a.n_wt = (int)plan.n_wt;
    a.n_tiles = (int)((plan.n_wt + kBatchThreads / 32 - 1) / (kBatchThreads / 32));
    a.M = p->n_tnfw; a.n_src = p->n_src;
    const bool conv = p->ky > 0;
    a.ky = conv ? p->ky : 0; a.kx = conv ? p->kx : 0;
    constexpr int kBatchOY = BatchOY<T>::value;
    a.kyp = (a.ky + kBatchOY - 1) / kBatchOY * kBatchOY;
    constexpr int TH = (kBatchThreads / 32) * kBatchOY;
    const int64_t pw64 = conv ? ((int64_t)g->nx + kBatchTW - 1) / kBatchTW * kBatchTW + a.kx - 1 : 0;   // even: pair loads stay aligned
    const int64_t ph64 = conv ? ((int64_t)g->ny + TH - 1) / TH * TH + a.kyp - 1 : 0;
    if (pw64 * ph64 * (int64_t)sizeof(T) > (int64_t)kBatchMaxSmem) return JT_ERR_UNSUPPORTED;   // before any int arithmetic on it
    a.pw = (int)pw64;
    a.ph = (int)ph64;
    a.img_elems = (a.pw * a.ph + 3) / 4 * 4;
    a.rec_cap = a.M < BatchRecCap<T>::value ? (a.M > 0 ? a.M : 1) : BatchRecCap<T>::value;
    a.sie = (const T*)p->sie; a.shear = (const T*)p->shear; a.tnfw = (const T*)p->tnfw;
    a.sersic = (const T*)p->sersic; a.psf = (const T*)p->psf;
    a.out = (T*)out;
    a.data = (const T*)data; a.sigma = (const T*)sigma; a.chi2 = chi2;
    a.dacc_off = (int)batch_smem_front(a);
    const size_t smem = (size_t)a.dacc_off + (sizeof(T) == 4 ? (size_t)plan.R * kBatchThreads * sizeof(double2) : 0);
    if (smem > kBatchMaxSmem) return JT_ERR_UNSUPPORTED;
    switch (plan.R) {
        JT_BATCH_CASE(5) JT_BATCH_CASE(6) JT_BATCH_CASE(7) JT_BATCH_CASE(8) JT_BATCH_CASE(9) JT_BATCH_CASE(10)
        JT_BATCH_CASE(11) JT_BATCH_CASE(12) JT_BATCH_CASE(13) JT_BATCH_CASE(14) JT_BATCH_CASE(15) JT_BATCH_CASE(16)
        default: return JT_ERR_UNSUPPORTED;
    }
    JT_LAUNCH_CHECK();
    return JT_OK;
}

jt_status launch_batch(jt_dtype dtype, int64_t B, const jt_grid* g, const jt_batch_params* p, void* out,
                       const void* data, const void* sigma, double* chi2, cudaStream_t st) {
    return dtype == JT_F32 ? batch_t<float>(dtype, B, g, p, out, data, sigma, chi2, st)
                           : batch_t<double>(dtype, B, g, p, out, data, sigma, chi2, st);
}

}  // namespace jt
