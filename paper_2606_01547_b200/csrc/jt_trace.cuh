// jt_trace.cuh -- the ray-tracing kernel: steps 1-4 of the hot path.
//
//   GRID mode  (jt_simulate_image): observer grid G generated in registers -> subhalo sum (definition T)
//              -> SIE + shear (S, H) -> lens equation -> Sersic (R) -> s x s binning with warp shuffles (B)
//              -> pre-PSF image.  Traced coordinates never leave the chip (PAPER.md:55 steps 1+2 fused).
//   RAYS mode  (jt_ray_shoot): same subhalo sum + SIE + shear on caller-supplied ray positions -> beta.
//
// N-body-style structure (PAPER.md:47 is where the time goes): 256 threads, each owning R rays whose deflection
// accumulators live in registers (float: per-tile float sums + double running sums in shared memory); a warp owns a
// "warp tile" of cols_per_warp x R rays, warp tiles are dealt to CTAs eight at a time.  The subhalo list streams
// through shared memory in tiles of derived records (SubRec, built in double by the staging threads; the CTA's whole
// chunk when it fits).  Per record the warp votes on the form of definition T:
//   far-far  X >= 9 max(1, tau):  the 1/X series of the brace (1 MUFU + K+1 multiply-adds), two records per iteration
//   far      X^2 >= max(10, 3 tau^2): logarithm-free closed form (3 MUFU + two polynomials)
//   mid      X^2 >= 2: the same with one logarithm
//   else     queued per warp and handled per ray by the out-of-line subhalo_cold after the hot loop
// float runs the far-far and far forms on two rays at once with packed f32x2 instructions (FFMA2 / FMUL2 / FADD2).
// When there are too few ray tiles to fill 148 SMs the subhalo list is split into chunks (wave-aware choice in
// jt_trace.cu); every (tile, chunk) CTA writes double partial sums to the workspace and the last CTA to arrive for
// a tile adds them in chunk order (deterministic) and runs the epilogue.
#pragma once
#include "jt_internal.h"

namespace jt {

template <typename T>
struct TraceArgs {
    // grid mode geometry (definition G)
    int nx, ny, s, NX, NY;
    double hh, cx, cy, area_over_s2;      // half ray spacing, grid centre
    int cols_per_warp, wtiles_x;
    int64_t n_wt;                         // warp tiles of the grid, dealt to CTAs eight at a time
    // ray mode
    int64_t n_rays;
    const T *tx, *ty;
    T *bx, *by;
    // lens
    MacroLens m;
    int64_t M;
    const T* tn[5];
    int n_chunks;
    int tile_recs;                         // subhalo records staged per shared-memory round
    int64_t chunk_len, n_tiles;
    double2* partial;
    unsigned int* counter;
    unsigned long long* tier_counts;       // 4 counters or nullptr (profiling off)
    // grid mode output
    T* out;
    SrcSet src;
};

// raw (caller) subhalo arrays of one system: cx, cy, Rs, alpha_Rs, r_trunc
template <typename T>
struct RawTn { const T* p[5]; };

constexpr double kMidX2 = 2.0;          // below this X^2 a ray takes the generic (logarithm, series) form

// geometry of definition G for one thread: column I, first row J0 of its R vertically adjacent rays.
// theta_x(I) = cx + (I - (NX-1)/2) h is evaluated as (2I - (NX-1)) * (h/2) + cx: the integer factor and h/2 are
// exact, so a centred grid with an odd ray count puts its middle ray exactly on 0 (the SIE centre, alpha = 0).
struct RayGeom {
    double hh, cx, cy;          // half ray spacing, grid centre
    int NX, NY, I, J0;
    __device__ __forceinline__ double xd() const { return fma((double)(2 * min(I, NX - 1) - (NX - 1)), hh, cx); }
    __device__ __forceinline__ double yd(int r) const { return fma((double)(2 * min(J0 + r, NY - 1) - (NY - 1)), hh, cy); }
};

// near/mid evaluation for the float kernel: coordinates re-derived in double so that dx, dy are exact
// where they matter; closed form in float for X^2 >= 1/4, double from the raw parameters below that.
template <typename T>
__device__ __noinline__ double2 tnfw_slow_f32(double xd, double yd, float cx, float cy, float iRs2, float t, float c1,
                                              float amp, float tm1, int64_t j, const RawTn<T>* raw) {
    const double dx = xd - (double)cx, dy = yd - (double)cy;
    const double R2 = dx * dx + dy * dy;
    double f;
    if (R2 * (double)iRs2 >= 0.25) {
        f = (double)tnfw_mid<float>((float)R2, iRs2, t, c1, amp, tm1);
    } else {
        const SubRec<double> s = make_rec<double>((double)raw->p[0][j], (double)raw->p[1][j], (double)raw->p[2][j],
                                                  (double)raw->p[3][j], (double)raw->p[4][j]);
        f = tnfw_any(R2, s);
    }
    return make_double2(f * dx, f * dy);
}

// Deflection accumulators of one thread's R rays.  double mode: 2R registers, summed directly.  float mode: the hot
// loop carries only float per-tile sums (tx, ty); the double running sums live in a column of shared memory
// (p[r * kTraceThreads]) that is touched once per staged tile, which keeps the float kernel at 128 registers
// (2 CTAs per SM) without spilling the ray coordinates.
// (warp, record) pairs handled by each form: far-far series, far, mid, queued for the per-ray cold path
struct TierCount { unsigned int n[4]; };

template <typename T, int R> struct DAcc;
template <int R> struct DAcc<double, R> {
    double tx[R], ty[R];
    __device__ __forceinline__ void init(double2*) {
#pragma unroll
        for (int r = 0; r < R; ++r) { tx[r] = 0.0; ty[r] = 0.0; }
    }
    __device__ __forceinline__ void begin_tile() {}
    __device__ __forceinline__ void end_tile() {}
    __device__ __forceinline__ void add_double(int r, double x, double y) { tx[r] += x; ty[r] += y; }
    __device__ __forceinline__ void result(double (&x)[R], double (&y)[R]) const {
#pragma unroll
        for (int r = 0; r < R; ++r) { x[r] = tx[r]; y[r] = ty[r]; }
    }
};
template <int R> struct DAcc<float, R> {
    float tx[R], ty[R];
    double2* p;
    __device__ __forceinline__ void init(double2* base) {
        p = base;
#pragma unroll
        for (int r = 0; r < R; ++r) p[r * kTraceThreads] = make_double2(0.0, 0.0);
    }
    __device__ __forceinline__ void begin_tile() {
#pragma unroll
        for (int r = 0; r < R; ++r) { tx[r] = 0.f; ty[r] = 0.f; }
    }
    __device__ __forceinline__ void end_tile() {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double2 v = p[r * kTraceThreads];
            v.x += (double)tx[r]; v.y += (double)ty[r];
            p[r * kTraceThreads] = v;
        }
    }
    __device__ __forceinline__ void add_double(int r, double x, double y) {
        double2 v = p[r * kTraceThreads];
        v.x += x; v.y += y;
        p[r * kTraceThreads] = v;
    }
    __device__ __forceinline__ void result(double (&x)[R], double (&y)[R]) const {
#pragma unroll
        for (int r = 0; r < R; ++r) { const double2 v = p[r * kTraceThreads]; x[r] = v.x; y[r] = v.y; }
    }
};
template <typename T, int R>
__host__ __device__ constexpr size_t dacc_smem_bytes() { return sizeof(T) == 4 ? (size_t)R * kTraceThreads * sizeof(double2) : 0; }

// Cold path: one record against this thread's R rays when the warp is not uniformly far or mid.  Out of line, and
// all per-ray state comes in through memory, so that the hot loop's register allocation never sees it.  Each ray
// picks its own form: far / mid as in the hot loop, else the generic closed form (series below X = 1e-3) in double.
// dp: the thread's double accumulator column in shared memory (float mode; nullptr in double mode).
template <typename T, int R, bool GRID>
__device__ __noinline__ void subhalo_cold(const SubRec<T>* rec, int64_t j, const RawTn<T>* raw, const RayGeom* g,
                                          const T* xs, const T* ys, T* ax, T* ay, double2* dp) {
    const SubRec<T> s = *rec;
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        const T dx = (GRID ? xs[0] : xs[r]) - s.cx, dy = ys[r] - s.cy;
        const T R2 = fma(dy, dy, dx * dx);
        const T X2 = R2 * s.iRs2;
        if (X2 >= (T)kMidX2) {
            const T f = (X2 >= s.thr) ? tnfw_far<T>(R2, s) : tnfw_midfast<T>(R2, s);
            ax[r] = fma(f, dx, ax[r]);
            ay[r] = fma(f, dy, ay[r]);
        } else if constexpr (sizeof(T) == 8) {
            const T f = (T)tnfw_any((double)R2, *(const SubRec<double>*)&s);
            ax[r] = fma(f, dx, ax[r]);
            ay[r] = fma(f, dy, ay[r]);
        } else {
            double xd, yd;
            if constexpr (GRID) { xd = g->xd(); yd = g->yd(r); }
            else { xd = (double)xs[r]; yd = (double)ys[r]; }
            const double2 c = tnfw_slow_f32<T>(xd, yd, s.cx, s.cy, s.iRs2, s.t, s.c1, s.amp, s.tm1, j, raw);
            double2 v = dp[r * kTraceThreads];
            v.x += c.x; v.y += c.y;
            dp[r * kTraceThreads] = v;
        }
    }
}

// One staged tile of `count` subhalo records against this thread's R rays: adds the tile's deflection to acc.
// GRID: the R rays share one column (xs[0]) and ascend in y.  Records for which the warp is neither uniformly far
// nor uniformly mid are queued (wq: this warp's index queue in shared memory, >= count entries) and handled by
// subhalo_cold after the hot loop.
template <typename T, int R, bool GRID, bool DUAL = true>
__device__ __forceinline__ void subhalo_tile(const SubRec<T>* __restrict__ recs, int count, int64_t base,
                                             const RawTn<T>& raw, const RayGeom& g, const T (&xs)[R], const T (&ys)[R],
                                             DAcc<T, R>& acc, unsigned short* wq, TierCount& tiers) {
    T (&ax)[R] = acc.tx;
    T (&ay)[R] = acc.ty;
    acc.begin_tile();
    int qn = 0;

    int jj = 0;
#pragma unroll 1
    while (jj < count) {
        // Two records at once when the warp is far-far from both (93-97 % of the pairs in the single-image paper-shaped
        // workloads; DUAL is off in the batch kernel, where only ~80 % qualify and the failed checks cost more): twice the independent dependency chains per warp for the MUFU + Horner sequence.
        if (DUAL && jj + 1 < count) {
            const SubRec<T>& sA = recs[jj];
            const SubRec<T>& sB = recs[jj + 1];
            T dxA[R], dyA[R], R2A[R], dxB[R], dyB[R], R2B[R];
            T mA, mB;
            if constexpr (GRID) {
                const T dA = xs[0] - sA.cx, dB = xs[0] - sB.cx, d2A = dA * dA, d2B = dB * dB;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    dxA[r] = dA; dyA[r] = ys[r] - sA.cy; R2A[r] = fma(dyA[r], dyA[r], d2A);
                    dxB[r] = dB; dyB[r] = ys[r] - sB.cy; R2B[r] = fma(dyB[r], dyB[r], d2B);
                }
                const T eA = fmax(fmax(ys[0] - sA.cy, sA.cy - ys[R - 1]), (T)0);
                const T eB = fmax(fmax(ys[0] - sB.cy, sB.cy - ys[R - 1]), (T)0);
                mA = fma(eA, eA, d2A);
                mB = fma(eB, eB, d2B);
            } else {
                mA = (T)3.0e38; mB = (T)3.0e38;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    dxA[r] = xs[r] - sA.cx; dyA[r] = ys[r] - sA.cy; R2A[r] = fma(dyA[r], dyA[r], dxA[r] * dxA[r]);
                    dxB[r] = xs[r] - sB.cx; dyB[r] = ys[r] - sB.cy; R2B[r] = fma(dyB[r], dyB[r], dxB[r] * dxB[r]);
                    mA = fmin(mA, R2A[r]); mB = fmin(mB, R2B[r]);
                }
            }
            if (__all_sync(0xffffffffu, mA * sA.iRs2 >= sA.thr2 && mB * sB.iRs2 >= sB.thr2)) {
                tiers.n[0] += 2;
                if constexpr (sizeof(T) == 4 && R % 2 == 0) {
#pragma unroll
                    for (int r = 0; r < R; r += 2) {
                        float f0, f1, h0, h1;
                        tnfw_farfar_pair(R2A[r], R2A[r + 1], sA, f0, f1);
                        tnfw_farfar_pair(R2B[r], R2B[r + 1], sB, h0, h1);
                        ax[r] = fma(f0, dxA[r], ax[r]);
                        ay[r] = fma(f0, dyA[r], ay[r]);
                        ax[r + 1] = fma(f1, dxA[r + 1], ax[r + 1]);
                        ay[r + 1] = fma(f1, dyA[r + 1], ay[r + 1]);
                        ax[r] = fma(h0, dxB[r], ax[r]);
                        ay[r] = fma(h0, dyB[r], ay[r]);
                        ax[r + 1] = fma(h1, dxB[r + 1], ax[r + 1]);
                        ay[r + 1] = fma(h1, dyB[r + 1], ay[r + 1]);
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const T fA = tnfw_farfar<T>(R2A[r], sA);
                        const T fB = tnfw_farfar<T>(R2B[r], sB);
                        ax[r] = fma(fA, dxA[r], ax[r]);
                        ay[r] = fma(fA, dyA[r], ay[r]);
                        ax[r] = fma(fB, dxB[r], ax[r]);
                        ay[r] = fma(fB, dyB[r], ay[r]);
                    }
                }
                jj += 2;
                continue;
            }
        }
        // one record, any tier
        const SubRec<T> s = recs[jj];
        T dx[R], dy[R], R2[R];
        T R2min;
        if constexpr (GRID) {
            const T d = xs[0] - s.cx, d2 = d * d;
#pragma unroll
            for (int r = 0; r < R; ++r) { dx[r] = d; dy[r] = ys[r] - s.cy; R2[r] = fma(dy[r], dy[r], d2); }
            // rows ascend in y: the closest row bounds the whole column
            const T m = fmax(fmax(ys[0] - s.cy, s.cy - ys[R - 1]), (T)0);
            R2min = fma(m, m, d2);
        } else {
            R2min = (T)3.0e38;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                dx[r] = xs[r] - s.cx; dy[r] = ys[r] - s.cy;
                R2[r] = fma(dy[r], dy[r], dx[r] * dx[r]);
                R2min = fmin(R2min, R2[r]);
            }
        }
        const T X2min = R2min * s.iRs2;
        if (__all_sync(0xffffffffu, X2min >= s.thr2)) {
            ++tiers.n[0];
            if constexpr (sizeof(T) == 4 && R % 2 == 0) {
#pragma unroll
                for (int r = 0; r < R; r += 2) {
                    float f0, f1;
                    tnfw_farfar_pair(R2[r], R2[r + 1], s, f0, f1);
                    ax[r] = fma(f0, dx[r], ax[r]);
                    ay[r] = fma(f0, dy[r], ay[r]);
                    ax[r + 1] = fma(f1, dx[r + 1], ax[r + 1]);
                    ay[r + 1] = fma(f1, dy[r + 1], ay[r + 1]);
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const T f = tnfw_farfar<T>(R2[r], s);
                    ax[r] = fma(f, dx[r], ax[r]);
                    ay[r] = fma(f, dy[r], ay[r]);
                }
            }
        } else if (__all_sync(0xffffffffu, X2min >= s.thr)) {
            ++tiers.n[1];
            if constexpr (sizeof(T) == 4 && R % 2 == 0) {
#pragma unroll
                for (int r = 0; r < R; r += 2) {
                    float f0, f1;
                    tnfw_far_pair(R2[r], R2[r + 1], s, f0, f1);
                    ax[r] = fma(f0, dx[r], ax[r]);
                    ay[r] = fma(f0, dy[r], ay[r]);
                    ax[r + 1] = fma(f1, dx[r + 1], ax[r + 1]);
                    ay[r + 1] = fma(f1, dy[r + 1], ay[r + 1]);
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const T f = tnfw_far<T>(R2[r], s);
                    ax[r] = fma(f, dx[r], ax[r]);
                    ay[r] = fma(f, dy[r], ay[r]);
                }
            }
        } else if (__all_sync(0xffffffffu, X2min >= (T)kMidX2)) {
            ++tiers.n[2];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T f = tnfw_midfast<T>(R2[r], s);
                ax[r] = fma(f, dx[r], ax[r]);
                ay[r] = fma(f, dy[r], ay[r]);
            }
        } else {
            if ((threadIdx.x & 31) == 0) wq[qn] = (unsigned short)jj;
            ++qn;
            ++tiers.n[3];
        }
        ++jj;
    }
    if (qn > 0) {                                   // warp-uniform
        __syncwarp();
        T lx[R], ly[R], lax[R], lay[R];             // local-memory copies: the cold path indexes them dynamically
#pragma unroll
        for (int r = 0; r < R; ++r) { lx[r] = xs[r]; ly[r] = ys[r]; lax[r] = ax[r]; lay[r] = ay[r]; }
        double2* dp = nullptr;
        if constexpr (sizeof(T) == 4) dp = acc.p;
#pragma unroll 1
        for (int q = 0; q < qn; ++q) {
            const int jj = wq[q];
            subhalo_cold<T, R, GRID>(&recs[jj], base + jj, &raw, &g, lx, ly, lax, lay, dp);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) { ax[r] = lax[r]; ay[r] = lay[r]; }
        __syncwarp();
    }
    acc.end_tile();
}

// stage `count` derived records (built in double) from the raw arrays starting at `base`
template <typename T>
__device__ __forceinline__ void stage_tile(SubRec<T>* recs, const RawTn<T>& raw, int64_t base, int count, int tid,
                                           int nthreads) {
    for (int k = tid; k < count; k += nthreads) {
        const int64_t j = base + k;
        recs[k] = make_rec<T>((double)raw.p[0][j], (double)raw.p[1][j], (double)raw.p[2][j], (double)raw.p[3][j],
                              (double)raw.p[4][j]);
    }
}

// O(rays) epilogue of the grid path in double: SIE + shear, lens equation, Sersic sum, s x s binning (definition B:
// s adjacent lanes hold the s sub-columns of a pixel -> segmented shuffle sum; each thread's R rows are a whole
// number of pixels).  store(j_pixel, i_pixel, value) receives pixel_scale^2/s^2 * sum.
template <typename T, int R, typename Store>
__device__ __forceinline__ void grid_epilogue(const MacroLens& m, const SrcSet& src, const RayGeom& g, int s,
                                              int cols_per_warp, double area_over_s2, int lane, const double (&axd)[R],
                                              const double (&ayd)[R], Store store) {
    double sx[R], sy[R];                        // dynamically indexed below -> local memory, once per ray
#pragma unroll
    for (int r = 0; r < R; ++r) { sx[r] = axd[r]; sy[r] = ayd[r]; }
    const double xd = g.xd();
    const int seg = lane - lane % s;
    const bool writer = (lane % s == 0) && (lane < cols_per_warp) && (g.I < g.NX);
    const int ip = g.I / s;
    double acc = 0.0;
    int sub = 0;
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        const int J = g.J0 + r;
        const double yd = g.yd(r);
        double mx, my;
        macro_alpha(m, xd, yd, mx, my);
        const double bx = xd - mx - sx[r], by = yd - my - sy[r];
        acc += sersic_sum<T>(src, bx, by);
        if (++sub == s) {
            double tot = 0.0;
            for (int d = 0; d < s; ++d) tot += __shfl_sync(0xffffffffu, acc, seg + d);
            if (writer && J < g.NY) store(J / s, ip, tot * area_over_s2);
            acc = 0.0;
            sub = 0;
        }
    }
}

template <typename T, int R, bool GRID>
__global__ void __launch_bounds__(kTraceThreads, sizeof(T) == 4 ? 2 : 1) k_trace(const __grid_constant__ TraceArgs<T> a) {
    __shared__ int s_last;
    // dynamic shared memory: [float mode: DAcc columns, R * 256 double2][tile_recs records][8 warp queues of tile_recs]
    extern __shared__ __align__(32) unsigned char dacc_raw[];
    SubRec<T>* recs = reinterpret_cast<SubRec<T>*>(dacc_raw + dacc_smem_bytes<T, R>());
    unsigned short* s_queue = reinterpret_cast<unsigned short*>(recs + a.tile_recs);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t tile = (int64_t)blockIdx.x / a.n_chunks;
    const int chunk = (int)((int64_t)blockIdx.x % a.n_chunks);

    // ---- ray ownership ----
    RayGeom g = {a.hh, a.cx, a.cy, a.NX, a.NY, 0, 0};
    int64_t idx0 = 0;                // ray mode: first ray index (stride 256)
    T xs[R], ys[R];
    if constexpr (GRID) {
        const int64_t wt = tile * (kTraceThreads / 32) + warp;
        if (wt < a.n_wt) {
            g.I = (int)(wt % a.wtiles_x) * a.cols_per_warp + lane;
            g.J0 = (int)(wt / a.wtiles_x) * R;
        } else {                                   // idle warp of the last CTA: clamped coordinates, no stores
            g.I = a.NX;
            g.J0 = a.NY;
        }
        T x = (T)g.xd();
        pin(x);
#pragma unroll
        for (int r = 0; r < R; ++r) { xs[r] = x; ys[r] = (T)g.yd(r); pin(ys[r]); }
    } else {
        idx0 = tile * (int64_t)(R * kTraceThreads) + tid;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = min(idx0 + (int64_t)r * kTraceThreads, a.n_rays - 1);
            xs[r] = a.tx[i];
            ys[r] = a.ty[i];
        }
    }

    DAcc<T, R> acc;
    acc.init(reinterpret_cast<double2*>(dacc_raw) + tid);
    TierCount tiers = {{0u, 0u, 0u, 0u}};

    // ---- subhalo sum over this CTA's chunk ----
    const RawTn<T> raw = {{a.tn[0], a.tn[1], a.tn[2], a.tn[3], a.tn[4]}};
    const int64_t j_begin = (int64_t)chunk * a.chunk_len;
    const int64_t j_end = min(a.M, j_begin + a.chunk_len);
    for (int64_t base = j_begin; base < j_end; base += a.tile_recs) {
        const int count = (int)min((int64_t)a.tile_recs, j_end - base);
        __syncthreads();
        stage_tile<T>(recs, raw, base, count, tid, kTraceThreads);
        __syncthreads();
        subhalo_tile<T, R, GRID>(recs, count, base, raw, g, xs, ys, acc, s_queue + warp * a.tile_recs, tiers);
    }
    double axd[R], ayd[R];
    acc.result(axd, ayd);
    if (a.tier_counts != nullptr && lane == 0) {          // measurement aid (jt_profile_tiers): four atomics per warp
#pragma unroll
        for (int k = 0; k < 4; ++k) atomicAdd(&a.tier_counts[k], (unsigned long long)tiers.n[k]);
    }

    // ---- split subhalo list: publish partial sums; the last CTA of the tile reduces them in chunk order ----
    if (a.n_chunks > 1) {
        const int64_t slot0 = ((int64_t)chunk * a.n_tiles + tile) * R;
#pragma unroll
        for (int r = 0; r < R; ++r)
            __stcg(&a.partial[(slot0 + r) * kTraceThreads + tid], make_double2(axd[r], ayd[r]));
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const unsigned int old = atomicAdd(&a.counter[tile], 1u);
            s_last = (old == (unsigned int)(a.n_chunks - 1));
        }
        __syncthreads();
        if (!s_last) return;
        __threadfence();
#pragma unroll
        for (int r = 0; r < R; ++r) { axd[r] = 0.0; ayd[r] = 0.0; }
        for (int c = 0; c < a.n_chunks; ++c) {
            const int64_t s0 = ((int64_t)c * a.n_tiles + tile) * R;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double2 v = __ldcg(&a.partial[(s0 + r) * kTraceThreads + tid]);
                axd[r] += v.x; ayd[r] += v.y;
            }
        }
        if (tid == 0) a.counter[tile] = 0u;     // leave the counter clean for the next call
    }

    // ---- epilogue: O(rays) work in double ----
    if constexpr (GRID) {
        T* out = a.out;
        const int nx = a.nx;
        grid_epilogue<T, R>(a.m, a.src, g, a.s, a.cols_per_warp, a.area_over_s2, lane, axd, ayd,
                            [out, nx](int j, int i, double v) { out[(int64_t)j * nx + i] = (T)v; });
    } else {
        double sx[R], sy[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { sx[r] = axd[r]; sy[r] = ayd[r]; }
#pragma unroll 1
        for (int r = 0; r < R; ++r) {
            const int64_t i = idx0 + (int64_t)r * kTraceThreads;
            if (i < a.n_rays) {
                const double xd = (double)a.tx[i], yd = (double)a.ty[i];
                double mx, my;
                macro_alpha(a.m, xd, yd, mx, my);
                a.bx[i] = (T)(xd - mx - sx[r]);
                a.by[i] = (T)(yd - my - sy[r]);
            }
        }
    }
}

// host launcher for one (T, GRID) pair; instantiated in jt_trace_f32.cu / jt_trace_f64.cu
template <typename T, bool GRID>
jt_status launch_trace_t(const TraceArgs<T>& a, int R, cudaStream_t st);

#define JT_TRACE_CASE(RR)                                                                         \
    case RR: {                                                                                    \
        auto kern = k_trace<T, RR, GRID>;                                                         \
        const size_t dsm = dacc_smem_bytes<T, RR>() + (size_t)a.tile_recs * (sizeof(SubRec<T>) + (kTraceThreads / 32) * 2); \
        static bool attr_set = false;   /* once per instantiation: allow the full dynamic shared memory */ \
        if (!attr_set) {                                                                          \
            JT_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024)); \
            attr_set = true;                                                                      \
        }                                                                                         \
        kern<<<(unsigned)grid, kTraceThreads, dsm, st>>>(a);                                      \
        break;                                                                                    \
    }

template <typename T, bool GRID>
jt_status launch_trace_impl(const TraceArgs<T>& a, int R, cudaStream_t st) {
    const int64_t grid = a.n_tiles * a.n_chunks;
    if (grid <= 0) return JT_OK;
    if (grid > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    if constexpr (GRID) {
        switch (R) {
            JT_TRACE_CASE(5) JT_TRACE_CASE(6) JT_TRACE_CASE(7) JT_TRACE_CASE(8) JT_TRACE_CASE(9) JT_TRACE_CASE(10) JT_TRACE_CASE(11)
            JT_TRACE_CASE(12) JT_TRACE_CASE(13) JT_TRACE_CASE(14) JT_TRACE_CASE(15) JT_TRACE_CASE(16)
            default: return JT_ERR_UNSUPPORTED;
        }
    } else {
        switch (R) {
            JT_TRACE_CASE(8)
            default: return JT_ERR_UNSUPPORTED;
        }
    }
    JT_LAUNCH_CHECK();
    return JT_OK;
}

}  // namespace jt
