// jt_trace.cuh -- the ray-tracing kernel: steps 1-4 of the hot path.
//
//   GRID mode  (jt_simulate_image): observer grid G generated in registers -> subhalo sum (definition T)
//              -> SIE + shear (S, H) -> lens equation -> Sersic (R) -> s x s binning with warp shuffles (B)
//              -> pre-PSF image.  Traced coordinates never leave the chip (PAPER.md:55 steps 1+2 fused).
//   RAYS mode  (jt_ray_shoot): same subhalo sum + SIE + shear on caller-supplied ray positions -> beta.
//
// N-body-style structure (PAPER.md:47 is where the time goes): NT threads, each owning R rays whose deflection
// accumulators live in registers (float: per-tile float sums + double running sums in shared memory); a warp owns a
// "warp tile" of cols_per_warp x R rays, warp tiles are dealt to CTAs NT/32 at a time.
//
// The subhalo list arrives as derived records (SubRec, built once per call in double by k_make_recs, in the caller's
// workspace) and streams through a ring of kStages shared-memory tiles filled by 1-D TMA bulk copies
// (cp.async.bulk + mbarrier).  No CTA-wide barrier sits in the loop: a warp waits on the tile's "full" mbarrier, and
// the last warp to finish a tile (a shared-memory arrival counter) issues the copy that refills its slot, so warps
// drift up to kStages - 1 tiles apart and a slow warp (one with subhalos inside its rays) delays nobody.
//
// Per tile and warp, GRID mode first SORTS the records by the form of definition T the whole warp tile can take
// (lane-parallel over records, from the distance between the record's centre and the warp tile's bounding box):
//   far-far  X >= 9 max(1, tau):  the 1/R series of the brace (1 MUFU + K+1 multiply-adds), U records per iteration
//   far      X^2 >= max(10, 3 tau^2): logarithm-free closed form (3 MUFU + two polynomials)
//   near     the same with one logarithm on every ray with X^2 >= 2, the generic closed form (out of line, double)
//            on the others
// and then runs one branch-free loop per class over its index list.  RAYS mode (arbitrary ray positions: no useful
// bounding box) votes per record on the rays themselves.  float runs the far-far and far forms on two rays at once
// with packed f32x2 instructions (FFMA2 / FMUL2 / FADD2).
// When there are too few ray tiles to fill the SMs the subhalo list is split into chunks (wave-aware choice in
// jt_trace.cu); every (tile, chunk) CTA writes double partial sums to the workspace and, warp by warp, the last to
// arrive for a warp tile adds them in chunk order (deterministic) and runs that warp tile's epilogue.
#pragma once
#include "jt_internal.h"

namespace jt {

constexpr int kStages = 3;              // record tiles in flight per CTA

template <typename T>
struct TraceArgs {
    // grid mode geometry (definition G)
    int nx, ny, s, NX, NY;
    double hh, cx, cy, area_over_s2;      // half ray spacing, grid centre
    int cols_per_warp, wtiles_x;
    int64_t n_wt;                         // warp tiles of the grid, dealt to CTAs NT/32 at a time
    int wide, cols_per_cta, ctiles_x;     // s does not divide 32: a CTA owns floor(NT/s)*s adjacent columns x R rows and bins through shared memory
    // ray mode
    int64_t n_rays;
    const T *tx, *ty;
    T *bx, *by;
    // lens
    MacroLens m;
    int64_t M;
    const T* tn[5];                        // raw subhalo arrays (float mode re-derives near-field records in double)
    const SubRec<T>* recs;                 // [M] derived records (workspace, written by k_make_recs)
    int n_chunks;
    int tile_recs;                         // records per shared-memory tile (multiple of 32)
    int64_t chunk_len, n_tiles;
    double2* partial;
    unsigned int* counter;
    unsigned long long* tier_counts;       // kTiers counters or nullptr (profiling off)
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

// ---- mbarrier / bulk-copy primitives ----
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned phase) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(phase) : "memory");
}
// `bytes` (multiple of 16) from global `src` to shared `dst` (both 16-byte aligned); completion counted on `bar`
__device__ __forceinline__ void bulk_load(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

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

// (warp, record) pairs handled by each form: far-far series at its three lengths, far, mid, per-ray cold path
constexpr int kTiers = 6;
struct TierCount { unsigned int n[kTiers]; };

// Deflection accumulators of one thread's R rays.  double mode: 2R registers, summed directly.  float mode: the hot
// loops carry only float per-tile sums (tx, ty); the double running sums live in a column of shared memory
// (p[r * NT]) that is touched once per record tile, which keeps the float kernel at 128 registers (2 CTAs per SM).
template <typename T, int R, int NT> struct DAcc;
template <int R, int NT> struct DAcc<double, R, NT> {
    double tx[R], ty[R];
    __device__ __forceinline__ void init(double2*) {
#pragma unroll
        for (int r = 0; r < R; ++r) { tx[r] = 0.0; ty[r] = 0.0; }
    }
    __device__ __forceinline__ void begin_tile() {}
    __device__ __forceinline__ void end_tile() {}
    __device__ __forceinline__ double2* column() { return nullptr; }
    __device__ __forceinline__ void result(double (&x)[R], double (&y)[R]) const {
#pragma unroll
        for (int r = 0; r < R; ++r) { x[r] = tx[r]; y[r] = ty[r]; }
    }
};
template <int R, int NT> struct DAcc<float, R, NT> {
    float tx[R], ty[R];
    double2* p;
    __device__ __forceinline__ void init(double2* base) {
        p = base;
#pragma unroll
        for (int r = 0; r < R; ++r) p[r * NT] = make_double2(0.0, 0.0);
    }
    __device__ __forceinline__ void begin_tile() {
#pragma unroll
        for (int r = 0; r < R; ++r) { tx[r] = 0.f; ty[r] = 0.f; }
    }
    __device__ __forceinline__ void end_tile() {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double2 v = p[r * NT];
            v.x += (double)tx[r]; v.y += (double)ty[r];
            p[r * NT] = v;
        }
    }
    __device__ __forceinline__ double2* column() { return p; }
    __device__ __forceinline__ void result(double (&x)[R], double (&y)[R]) const {
#pragma unroll
        for (int r = 0; r < R; ++r) { const double2 v = p[r * NT]; x[r] = v.x; y[r] = v.y; }
    }
};
template <typename T, int R, int NT>
__host__ __device__ constexpr size_t dacc_smem_bytes() { return sizeof(T) == 4 ? (size_t)R * NT * sizeof(double2) : 0; }

// far / mid forms of one record on the thread's R rays (warp-uniform choice)
template <typename T, int R, bool GRID, bool FULL = true>
__device__ __forceinline__ void eval_far(const SubRec<T>& s, const T (&xs)[R], const T (&ys)[R], T (&ax)[R], T (&ay)[R]) {
    T dx[R], dy[R], R2[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        dx[r] = (GRID ? xs[0] : xs[r]) - s.cx;
        dy[r] = ys[r] - s.cy;
        R2[r] = fma(dy[r], dy[r], dx[r] * dx[r]);
    }
    if constexpr (sizeof(T) == 4 && R % 2 == 0) {
        auto pair = [&](int r) {
            float f0, f1;
            tnfw_far_pair(R2[r], R2[r + 1], s, f0, f1);
            ax[r] = fma(f0, dx[r], ax[r]);
            ay[r] = fma(f0, dy[r], ay[r]);
            ax[r + 1] = fma(f1, dx[r + 1], ax[r + 1]);
            ay[r + 1] = fma(f1, dy[r + 1], ay[r + 1]);
        };
        if constexpr (FULL) {
#pragma unroll
            for (int r = 0; r < R; r += 2) pair(r);
        } else {                                    // two pairs in flight: a quarter of the code (instruction-cache space)
#pragma unroll 2
            for (int r = 0; r < R; r += 2) pair(r);
        }
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const T f = tnfw_far<T>(R2[r], s);
            ax[r] = fma(f, dx[r], ax[r]);
            ay[r] = fma(f, dy[r], ay[r]);
        }
    }
}
// Anything nearer: the mid form (valid for X^2 >= 2) on every ray that qualifies, masked on the others, which are
// then evaluated one by one by the generic closed form (series below X = 1e-3) in double -- out of line, so that the
// hot loops' register allocation never sees it.  No local-memory copies: every array index is a compile-time constant.
// dp: the thread's double accumulator column in shared memory (float mode; nullptr in double mode).
template <typename T, int R, bool GRID, int NT>
__device__ __forceinline__ void eval_near(const SubRec<T>& s, int64_t j, const RawTn<T>& raw, const RayGeom& g, const T (&xs)[R],
                                          const T (&ys)[R], T (&ax)[R], T (&ay)[R], double2* dp) {
    unsigned slow = 0u;
    const T R2safe = (T)4 * ((T)1 / s.iRs2);        // X^2 = 4 for the masked rays: keeps their (discarded) arithmetic finite
#pragma unroll 2                                    // rare (a few % of the pairs): kept small for the instruction cache
    for (int r = 0; r < R; ++r) {
        const T dx = (GRID ? xs[0] : xs[r]) - s.cx, dy = ys[r] - s.cy;
        const T R2 = fma(dy, dy, dx * dx);
        const bool ok = R2 * s.iRs2 >= (T)kMidX2;
        const T f = tnfw_midfast<T>(ok ? R2 : R2safe, s);
        if (ok) {
            ax[r] = fma(f, dx, ax[r]);
            ay[r] = fma(f, dy, ay[r]);
        } else {
            slow |= 1u << r;
        }
    }
    if (__any_sync(0xffffffffu, slow != 0u)) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (slow & (1u << r)) {
                if constexpr (sizeof(T) == 8) {
                    const T dx = (GRID ? xs[0] : xs[r]) - s.cx, dy = ys[r] - s.cy;
                    const T f = (T)tnfw_any((double)fma(dy, dy, dx * dx), *(const SubRec<double>*)&s);
                    ax[r] = fma(f, dx, ax[r]);
                    ay[r] = fma(f, dy, ay[r]);
                } else {
                    double xd, yd;
                    if constexpr (GRID) { xd = g.xd(); yd = g.yd(r); }
                    else { xd = (double)xs[r]; yd = (double)ys[r]; }
                    const double2 c = tnfw_slow_f32<T>(xd, yd, s.cx, s.cy, s.iRs2, s.t, s.c1, s.amp, s.tm1, j, &raw);
                    double2 v = dp[r * NT];
                    v.x += c.x; v.y += c.y;
                    dp[r * NT] = v;
                }
            }
        }
    }
}

// ---- GRID mode: the far-far loops over this warp's index lists ----
// One record per iteration against the thread's R rays (R independent chains; the rays share one column, so dx and
// dx^2 are per record), Horner recurrence unrolled for the level's series length K.  One record per iteration and no
// remainder loops keep the three levels' loop bodies small: with two records per iteration (and their remainder
// loops) the hot code of all resident warps no longer fitted the 32 KB instruction cache, and ncu showed 30-40 % of
// the warp samples waiting for instructions; a rolled Horner loop (one body for all levels) was 25-40 % slower.
// The list is read at list[i * stride], i < n (stride = +1 or -1: two lists share one array from its two ends).
template <int R, int K>
__device__ __forceinline__ void farfar_list(const SubRec<double>* __restrict__ recs, const unsigned short* __restrict__ list, int stride,
                                            int n, double x, const double (&ys)[R], double (&ax)[R], double (&ay)[R]) {
    unsigned nxt = n > 0 ? list[0] : 0u;           // indices are fetched one iteration ahead
#pragma unroll 1
    for (int i = 0; i < n; ++i) {
        const SubRec<double>& s = recs[nxt];
        nxt = i + 1 < n ? list[(i + 1) * stride] : 0u;
        const double dx = x - s.cx, d2 = dx * dx;
        double dy[R], v[R], p[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            dy[r] = ys[r] - s.cy;
            v[r] = fast_rsqrt(fma(dy[r], dy[r], d2));
            p[r] = s.ak[K - 2];
        }
#pragma unroll
        for (int k = K - 3; k >= 0; --k)
#pragma unroll
            for (int r = 0; r < R; ++r) p[r] = fma(p[r], v[r], s.ak[k]);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const double v2 = v[r] * v[r];
            const double f = v2 * fma(p[r], v2, s.a0);
            ax[r] = fma(f, dx, ax[r]);
            ay[r] = fma(f, dy[r], ay[r]);
        }
    }
}

// float: everything packed (two rows per 64-bit register): FADD2 dy, FFMA2 R^2, 2 MUFU, FMUL2 v^2, K-2 FFMA2 Horner
// steps, FFMA2 + FMUL2, 2 FFMA2 into the accumulators = K + 5 packed instructions + 2 MUFU per two evaluations.
// ax2, ay2, y2: the thread's accumulators and rows as packed pairs.  U records per iteration: the float loop is bound
// by issue slots as much as by the FP32 pipe, so the per-record bookkeeping (index, addresses, dx) is shared by two
// records when the register budget allows (measured: C2-f32 0.96 ms with U = 2, 1.11 ms with U = 1); the float bodies
// are small enough for that (and their one-record remainder loops) to stay in the instruction cache.
template <int H, int K, int U>
__device__ __forceinline__ void farfar_list2(const SubRec<float>* __restrict__ recs, const unsigned short* __restrict__ list, int stride,
                                             int n, float x, const f32x2 (&y2)[H], f32x2 (&ax2)[H], f32x2 (&ay2)[H]) {
    int i = 0;
    unsigned nxt[U];
#pragma unroll
    for (int u = 0; u < U; ++u) nxt[u] = u < n ? list[u * stride] : 0u;
#pragma unroll 1
    for (; i + U <= n; i += U) {
        const SubRec<float>* s[U];
        f32x2 dx2[U], dy[U][H], f[U][H];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            s[u] = recs + nxt[u];
            nxt[u] = i + U + u < n ? list[(i + U + u) * stride] : 0u;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const float dx = x - s[u]->cx;
            const f32x2 d2 = bc2(dx * dx), ncy = bc2(-s[u]->cy);
            dx2[u] = bc2(dx);
#pragma unroll
            for (int h = 0; h < H; ++h) {
                dy[u][h] = add2(y2[h], ncy);
                f[u][h] = tnfw_farfar2<K>(fma2(dy[u][h], dy[u][h], d2), *s[u]);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int h = 0; h < H; ++h) {
                ax2[h] = fma2(f[u][h], dx2[u], ax2[h]);
                ay2[h] = fma2(f[u][h], dy[u][h], ay2[h]);
            }
    }
    if constexpr (U > 1) {
#pragma unroll 1
        for (; i < n; ++i) {
            const SubRec<float>& s = recs[list[i * stride]];
            const float dx = x - s.cx;
            const f32x2 d2 = bc2(dx * dx), ncy = bc2(-s.cy), dx2 = bc2(dx);
#pragma unroll
            for (int h = 0; h < H; ++h) {
                const f32x2 dy = add2(y2[h], ncy);
                const f32x2 f = tnfw_farfar2<K>(fma2(dy, dy, d2), s);
                ax2[h] = fma2(f, dx2, ax2[h]);
                ay2[h] = fma2(f, dy, ay2[h]);
            }
        }
    }
}
template <int R, int K>
__device__ __forceinline__ void farfar_list(const SubRec<float>* __restrict__ recs, const unsigned short* __restrict__ list, int stride,
                                            int n, float x, const float (&ys)[R], float (&ax)[R], float (&ay)[R]) {
#pragma unroll 1
    for (int i = 0; i < n; ++i) {                  // odd R only (even R goes through farfar_list2)
        const SubRec<float>& s = recs[list[i * stride]];
        const float dx = x - s.cx, d2 = dx * dx;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float dy = ys[r] - s.cy;
            const float f = tnfw_farfar<float, K>(fma(dy, dy, d2), s);
            ax[r] = fma(f, dx, ax[r]);
            ay[r] = fma(f, dy, ay[r]);
        }
    }
}

// the three levels, shortest series first
// VAR: bit 0: float far-far loops take two records per iteration; bit 1: far form fully unrolled over the rays;
// bit 2: one far-far level (the longest series for every far-far record).  Measured on B200:
// the single-image kernels run best with 3 (float) / 2 (double), the batch kernel -- whose code also holds the
// staging, the epilogue and the convolution, and whose 16 warps per SM are spread over all of it -- with 2: two
// records per iteration cost it 25 % (instruction cache), a software-pipelined one-record loop 11 %.
template <typename T, int R, int VAR>
__device__ __forceinline__ void farfar_levels(const SubRec<T>* __restrict__ recs, const unsigned short* l0, int n0, const unsigned short* l1,
                                              int n1, const unsigned short* l2, int n2, const T (&xs)[R], const T (&ys)[R],
                                              T (&ax)[R], T (&ay)[R]) {
    using FF = FarFar<T>;
    if constexpr (sizeof(T) == 4 && R % 2 == 0) {
        constexpr int H = R / 2;
        f32x2 y2[H], ax2[H], ay2[H];
#pragma unroll
        for (int h = 0; h < H; ++h) {
            y2[h] = pack2(ys[2 * h], ys[2 * h + 1]);
            ax2[h] = pack2(ax[2 * h], ax[2 * h + 1]);
            ay2[h] = pack2(ay[2 * h], ay[2 * h + 1]);
        }
        constexpr int U = (H <= 5 && (VAR & 1)) ? 2 : 1;
        farfar_list2<H, FF::K2, U>(recs, l2, 1, n2, xs[0], y2, ax2, ay2);
        farfar_list2<H, FF::K1, U>(recs, l1, -1, n1, xs[0], y2, ax2, ay2);
        farfar_list2<H, FF::K, U>(recs, l0, 1, n0, xs[0], y2, ax2, ay2);
#pragma unroll
        for (int h = 0; h < H; ++h) {
            unpack2(ax2[h], ax[2 * h], ax[2 * h + 1]);
            unpack2(ay2[h], ay[2 * h], ay[2 * h + 1]);
        }
    } else {
        farfar_list<R, FF::K2>(recs, l2, 1, n2, xs[0], ys, ax, ay);
        farfar_list<R, FF::K1>(recs, l1, -1, n1, xs[0], ys, ax, ay);
        farfar_list<R, FF::K>(recs, l0, 1, n0, xs[0], ys, ax, ay);
    }
}

// bounding box of a warp tile in the call's dtype (GRID mode: all lanes share the R rows)
template <typename T> struct WarpBox { T xlo, xhi, ylo, yhi; };

// One tile of `count` records against this thread's R rays, GRID mode.  Pass 1 (lane-parallel over records) sorts the
// record indices by class into `list` (this warp's, 2 * cap entries): first array: longest far-far series from the
// front, middle one from the back; second array: shortest series from the front, everything else from the back with
// the class in the top two bits.  Then one loop per class.
template <typename T, int R, int NT, int VAR>
__device__ __forceinline__ void subhalo_tile_sorted(const SubRec<T>* __restrict__ recs, int count, int cap, int64_t base,
                                                    const RawTn<T>& raw, const RayGeom& g, const WarpBox<T>& box, const T (&xs)[R],
                                                    const T (&ys)[R], DAcc<T, R, NT>& acc, unsigned short* list, TierCount& tiers) {
    using FF = FarFar<T>;
    constexpr T kL1 = (T)((FF::kRadius1 / FF::kRadius) * (FF::kRadius1 / FF::kRadius));
    constexpr T kL2 = (T)((FF::kRadius2 / FF::kRadius) * (FF::kRadius2 / FF::kRadius));
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    unsigned short* list2 = list + cap;
    int n0 = 0, n1 = 0, n2 = 0, n_ot = 0, n_near = 0, n_cold = 0;
#pragma unroll 1
    for (int b0 = 0; b0 < count; b0 += 32) {
        const int j = b0 + lane;
        int cls = -1;                               // 0, 1, 2: far-far levels; 3 far; 4 mid; 5 cold
        if (j < count) {
            const SubRec<T>& s = recs[j];
            const T ex = fmax(fmax(box.xlo - s.cx, s.cx - box.xhi), (T)0);
            const T ey = fmax(fmax(box.ylo - s.cy, s.cy - box.yhi), (T)0);
            const T X2 = fma(ey, ey, ex * ex) * s.iRs2;
            cls = X2 >= s.thr2 ? ((VAR & 4) ? 0 : (X2 >= s.thr2 * kL2 ? 2 : (X2 >= s.thr2 * kL1 ? 1 : 0)))
                               : (X2 >= s.thr ? 3 : (X2 >= (T)kMidX2 ? 4 : 5));
        }
        const unsigned m0 = __ballot_sync(0xffffffffu, cls == 0), m1 = __ballot_sync(0xffffffffu, cls == 1);
        const unsigned m2 = __ballot_sync(0xffffffffu, cls == 2), mo = __ballot_sync(0xffffffffu, cls >= 3);
        const unsigned mn = __ballot_sync(0xffffffffu, cls >= 4), mc = __ballot_sync(0xffffffffu, cls == 5);
        if (cls == 0) list[n0 + __popc(m0 & lt)] = (unsigned short)j;
        if (cls == 1) list[cap - 1 - (n1 + __popc(m1 & lt))] = (unsigned short)j;
        if (cls == 2) list2[n2 + __popc(m2 & lt)] = (unsigned short)j;
        if (cls >= 3) list2[cap - 1 - (n_ot + __popc(mo & lt))] = (unsigned short)(j | ((cls == 3 ? 1 : 2) << 14));
        n0 += __popc(m0);
        n1 += __popc(m1);
        n2 += __popc(m2);
        n_ot += __popc(mo);
        n_near += __popc(mn);
        n_cold += __popc(mc);
    }
    __syncwarp();
    tiers.n[0] += n0;
    tiers.n[1] += n1;
    tiers.n[2] += n2;
    tiers.n[4] += n_near - n_cold;
    tiers.n[5] += n_cold;

    acc.begin_tile();
    T (&ax)[R] = acc.tx;
    T (&ay)[R] = acc.ty;
    farfar_levels<T, R, VAR>(recs, list, n0, list + cap - 1, n1, list2, n2, xs, ys, ax, ay);
#pragma unroll 1
    for (int q = 0; q < n_ot; ++q) {
        const unsigned e = list2[cap - 1 - q];
        const int jj = e & 0x3fff;
        if ((e >> 14) == 1) eval_far<T, R, true, (VAR & 2) != 0>(recs[jj], xs, ys, ax, ay);
        else eval_near<T, R, true, NT>(recs[jj], base + jj, raw, g, xs, ys, ax, ay, acc.column());
    }
    tiers.n[3] += n_ot - n_near;
    __syncwarp();                                  // the lists are rewritten by the next tile
    acc.end_tile();
}

// One tile, RAYS mode: the warp votes per record on its actual rays.
template <typename T, int R, int NT>
__device__ __forceinline__ void subhalo_tile_vote(const SubRec<T>* __restrict__ recs, int count, int64_t base, const RawTn<T>& raw,
                                                  const RayGeom& g, const T (&xs)[R], const T (&ys)[R], DAcc<T, R, NT>& acc,
                                                  TierCount& tiers) {
    T (&ax)[R] = acc.tx;
    T (&ay)[R] = acc.ty;
    acc.begin_tile();
#pragma unroll 1
    for (int jj = 0; jj < count; ++jj) {
        const SubRec<T>& s = recs[jj];
        T R2min = (T)3.0e38;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const T dx = xs[r] - s.cx, dy = ys[r] - s.cy;
            R2min = fmin(R2min, fma(dy, dy, dx * dx));
        }
        const T X2min = R2min * s.iRs2;
        if (__all_sync(0xffffffffu, X2min >= s.thr2)) {
            ++tiers.n[0];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T dx = xs[r] - s.cx, dy = ys[r] - s.cy;
                const T f = tnfw_farfar<T>(fma(dy, dy, dx * dx), s);   // full-length series: one level in this mode
                ax[r] = fma(f, dx, ax[r]);
                ay[r] = fma(f, dy, ay[r]);
            }
        } else if (__all_sync(0xffffffffu, X2min >= s.thr)) {
            ++tiers.n[3];
            eval_far<T, R, false>(s, xs, ys, ax, ay);
        } else {
            ++tiers.n[__all_sync(0xffffffffu, X2min >= (T)kMidX2) ? 4 : 5];
            eval_near<T, R, false, NT>(s, base + jj, raw, g, xs, ys, ax, ay, acc.column());
        }
    }
    acc.end_tile();
}

// ---- derived records, once per call ----
// Also zeroes the arrival counters of the split subhalo list and the tier counters, so a call needs no memset.
template <typename T>
__global__ void __launch_bounds__(128) k_make_recs(int64_t M, RawTn<T> raw, SubRec<T>* __restrict__ recs, unsigned int* counter,
                                                   int n_counter, unsigned long long* tier_counts) {
    cudaTriggerProgrammaticLaunchCompletion();      // the ray-tracing kernel may start its prologue
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_counter) counter[i] = 0u;
    if (tier_counts != nullptr && i < kTiers) tier_counts[i] = 0ull;
    if (i < M)
        recs[i] = make_rec<T>((double)raw.p[0][i], (double)raw.p[1][i], (double)raw.p[2][i], (double)raw.p[3][i],
                              (double)raw.p[4][i]);
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

// The same O(rays) work for the CTA-wide tiles: the surface brightness of this thread's R rays -> dst[r * pitch]
// (0 for rays outside the grid and for the spare threads of the tile).
template <typename T, int R>
__device__ __forceinline__ void grid_brightness(const MacroLens& m, const SrcSet& src, const RayGeom& g, bool active,
                                                const double (&axd)[R], const double (&ayd)[R], double* dst, int pitch) {
    double sx[R], sy[R];                        // dynamically indexed below -> local memory, once per ray
#pragma unroll
    for (int r = 0; r < R; ++r) { sx[r] = axd[r]; sy[r] = ayd[r]; }
    const double xd = g.xd();
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        double v = 0.0;
        if (active && g.I < g.NX && g.J0 + r < g.NY) {
            const double yd = g.yd(r);
            double mx, my;
            macro_alpha(m, xd, yd, mx, my);
            v = sersic_sum<T>(src, xd - mx - sx[r], yd - my - sy[r]);
        }
        dst[r * pitch] = v;
    }
}

// shared-memory footprint of k_trace: [float mode: DAcc columns][kStages record tiles][NT/32 x 2 index lists][barriers]
template <typename T, int R, int NT>
__host__ __device__ constexpr size_t trace_smem_bytes(int tile_recs) {
    return dacc_smem_bytes<T, R, NT>() + (size_t)tile_recs * (kStages * sizeof(SubRec<T>) + (NT / 32) * 2 * sizeof(unsigned short)) + 64;
}

template <typename T> struct TraceCfg;       // threads per CTA, CTAs per SM, records per far-far iteration
template <> struct TraceCfg<double> { static constexpr int NT = 128, OCC = 2, VAR = 2; };
template <> struct TraceCfg<float> { static constexpr int NT = 256, OCC = 2, VAR = 3; };

template <typename T, int R, bool GRID>
__global__ void __launch_bounds__(TraceCfg<T>::NT, TraceCfg<T>::OCC) k_trace(const __grid_constant__ TraceArgs<T> a) {
    constexpr int NT = TraceCfg<T>::NT, NW = NT / 32;
    extern __shared__ __align__(32) unsigned char dacc_raw[];
    SubRec<T>* ring = reinterpret_cast<SubRec<T>*>(dacc_raw + dacc_smem_bytes<T, R, NT>());
    unsigned short* lists = reinterpret_cast<unsigned short*>(ring + (size_t)kStages * a.tile_recs);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(lists + (size_t)NW * 2 * a.tile_recs);   // 8-byte aligned: tile_recs % 32 == 0
    unsigned int* done = reinterpret_cast<unsigned int*>(full + kStages);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t tile = (int64_t)blockIdx.x / a.n_chunks;
    const int chunk = (int)((int64_t)blockIdx.x % a.n_chunks);
    const int64_t j_begin = (int64_t)chunk * a.chunk_len;
    const int64_t j_end = min(a.M, j_begin + a.chunk_len);
    const int n_rounds = j_end > j_begin ? (int)((j_end - j_begin + a.tile_recs - 1) / a.tile_recs) : 0;

    cudaTriggerProgrammaticLaunchCompletion();     // a dependent launch (the small convolution) may stage its taps now
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], 1); done[s] = 0u; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    // ---- ray ownership ----
    RayGeom g = {a.hh, a.cx, a.cy, a.NX, a.NY, 0, 0};
    int64_t idx0 = 0;                // ray mode: first ray index (stride NT)
    T xs[R], ys[R];
    if constexpr (GRID) {
        const int64_t wt = tile * NW + warp;
        if (a.wide) {                              // CTA tile: cols_per_cta columns x R rows; the spare threads shadow
            // the tile's last column (their rays must not widen the warp's bounding box) and store nothing
            g.I = (int)(tile % a.ctiles_x) * a.cols_per_cta + min(tid, a.cols_per_cta - 1);
            g.J0 = (int)(tile / a.ctiles_x) * R;
        } else if (wt < a.n_wt) {
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
        idx0 = tile * (int64_t)(R * NT) + tid;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int64_t i = min(idx0 + (int64_t)r * NT, a.n_rays - 1);
            xs[r] = a.tx[i];
            ys[r] = a.ty[i];
        }
    }
    WarpBox<T> box = {xs[0], xs[0], ys[0], ys[R - 1]};
    if constexpr (GRID) {
        box.xlo = __shfl_sync(0xffffffffu, xs[0], 0);
        box.xhi = __shfl_sync(0xffffffffu, xs[0], 31);      // columns ascend with the lane (clamped at the grid edge)
    }

    DAcc<T, R, NT> acc;
    acc.init(reinterpret_cast<double2*>(dacc_raw) + tid);
    TierCount tiers = {};
    const RawTn<T> raw = {{a.tn[0], a.tn[1], a.tn[2], a.tn[3], a.tn[4]}};

    __syncthreads();                               // barriers initialised
    // ---- subhalo sum over this CTA's chunk: kStages tiles in flight ----
    auto issue = [&](int k) {                      // one thread: bulk copy of round k's records into slot k % kStages
        const int s = k % kStages;
        const int64_t j0 = j_begin + (int64_t)k * a.tile_recs;
        const unsigned bytes = (unsigned)(min((int64_t)a.tile_recs, j_end - j0) * sizeof(SubRec<T>));
        mbar_expect_tx(&full[s], bytes);
        bulk_load(ring + (size_t)s * a.tile_recs, a.recs + j0, bytes, &full[s]);
    };
    if (n_rounds > 0) {
        cudaGridDependencySynchronize();           // the records written by k_make_recs are visible
        if (tid == 0)
            for (int k = 0; k < kStages && k < n_rounds; ++k) issue(k);
    }
    unsigned short* list = lists + (size_t)warp * 2 * a.tile_recs;
#pragma unroll 1
    for (int k = 0; k < n_rounds; ++k) {
        const int s = k % kStages;
        const int64_t base = j_begin + (int64_t)k * a.tile_recs;
        const int count = (int)min((int64_t)a.tile_recs, j_end - base);
        mbar_wait(&full[s], (unsigned)((k / kStages) & 1));
        const SubRec<T>* recs = ring + (size_t)s * a.tile_recs;
        if constexpr (GRID) subhalo_tile_sorted<T, R, NT, TraceCfg<T>::VAR>(recs, count, a.tile_recs, base, raw, g, box, xs, ys, acc, list, tiers);
        else subhalo_tile_vote<T, R, NT>(recs, count, base, raw, g, xs, ys, acc, tiers);
        // release the slot; the last warp to finish refills it
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            if (atomicAdd(&done[s], 1u) == (unsigned)(NW - 1)) {
                done[s] = 0u;
                __threadfence_block();
                if (k + kStages < n_rounds) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    issue(k + kStages);
                }
            }
        }
    }
    double axd[R], ayd[R];
    acc.result(axd, ayd);
    if (a.tier_counts != nullptr && lane == 0) {          // measurement aid (jt_profile_tiers): six atomics per warp
#pragma unroll
        for (int k = 0; k < kTiers; ++k) atomicAdd(&a.tier_counts[k], (unsigned long long)tiers.n[k]);
    }

    // ---- split subhalo list: publish partial sums; the last WARP to arrive for a warp tile (over the chunks) adds them
    // in chunk order and runs that warp tile's epilogue.  Per warp, not per CTA: a CTA-wide barrier here kept the warps
    // that had finished waiting for the one with subhalo cores in its rays (ncu: 9-12 % of all warp samples).
    if (a.n_chunks > 1) {
        const int64_t slot0 = ((int64_t)chunk * a.n_tiles + tile) * R;
#pragma unroll
        for (int r = 0; r < R; ++r)
            __stcg(&a.partial[(slot0 + r) * NT + tid], make_double2(axd[r], ayd[r]));
        __threadfence();
        if (GRID && a.wide) {                      // the CTA bins together: CTA-wide completion
            __shared__ int s_last;
            __syncthreads();
            if (tid == 0) s_last = atomicAdd(&a.counter[tile], 1u) == (unsigned int)(a.n_chunks - 1);
            __syncthreads();
            if (!s_last) return;
        } else {
            __syncwarp();
            unsigned int old = 0u;
            if (lane == 0) old = atomicAdd(&a.counter[tile * NW + warp], 1u);
            old = __shfl_sync(0xffffffffu, old, 0);
            if (old != (unsigned int)(a.n_chunks - 1)) return;
        }
        __threadfence();
#pragma unroll
        for (int r = 0; r < R; ++r) { axd[r] = 0.0; ayd[r] = 0.0; }
        for (int c = 0; c < a.n_chunks; ++c) {
            const int64_t s0 = ((int64_t)c * a.n_tiles + tile) * R;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double2 v = __ldcg(&a.partial[(s0 + r) * NT + tid]);
                axd[r] += v.x; ayd[r] += v.y;
            }
        }
    }

    // ---- epilogue: O(rays) work in double ----
    if constexpr (GRID) {
        T* out = a.out;
        const int nx = a.nx;
        if (a.wide) {
            // ray brightness -> shared memory (the accumulator columns in float mode, the record ring in double: both
            // are free once every warp has left the loop), then one thread per pixel sums its s x s rays in fixed order
            __syncthreads();
            double* sB = sizeof(T) == 4 ? reinterpret_cast<double*>(dacc_raw) : reinterpret_cast<double*>(ring);
            grid_brightness<T, R>(a.m, a.src, g, tid < a.cols_per_cta, axd, ayd, sB + tid, NT);
            __syncthreads();
            const int s = a.s, n_px = a.cols_per_cta / s, n_py = R / s;
            const int i0 = (int)(tile % a.ctiles_x) * n_px, j0 = (int)(tile / a.ctiles_x) * n_py;
            for (int p = tid; p < n_px * n_py; p += NT) {
                const int py = p / n_px, px = p - py * n_px;
                double tot = 0.0;
                for (int u = 0; u < s; ++u)
                    for (int v = 0; v < s; ++v) tot += sB[(py * s + u) * NT + px * s + v];
                if (i0 + px < a.nx && j0 + py < a.ny) out[(int64_t)(j0 + py) * nx + i0 + px] = (T)(tot * a.area_over_s2);
            }
        } else {
            grid_epilogue<T, R>(a.m, a.src, g, a.s, a.cols_per_warp, a.area_over_s2, lane, axd, ayd,
                                [out, nx](int j, int i, double v) { out[(int64_t)j * nx + i] = (T)v; });
        }
    } else {
        double sx[R], sy[R];
#pragma unroll
        for (int r = 0; r < R; ++r) { sx[r] = axd[r]; sy[r] = ayd[r]; }
#pragma unroll 1
        for (int r = 0; r < R; ++r) {
            const int64_t i = idx0 + (int64_t)r * NT;
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
        const size_t dsm = trace_smem_bytes<T, RR, TraceCfg<T>::NT>(a.tile_recs);                 \
        static PerDeviceOnce attr;   /* once per instantiation and device: allow the full dynamic shared memory */ \
        if (attr.needed()) {                                                                      \
            JT_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 1024)); \
            attr.mark();                                                                          \
        }                                                                                         \
        cfg.dynamicSmemBytes = dsm;                                                               \
        JT_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, a));                                           \
        break;                                                                                    \
    }

template <typename T, bool GRID>
jt_status launch_trace_impl(const TraceArgs<T>& a, int R, cudaStream_t st) {
    const int64_t grid = a.n_tiles * a.n_chunks;
    if (grid <= 0) return JT_OK;
    if (grid > 0x7fffffffLL) return JT_ERR_UNSUPPORTED;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)TraceCfg<T>::NT);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;     // prologue overlaps k_make_recs (when there is one)
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = a.M > 0 ? 1 : 0;
    if constexpr (GRID) {
        switch (R) {
            JT_TRACE_CASE(1) JT_TRACE_CASE(2) JT_TRACE_CASE(3) JT_TRACE_CASE(4)
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
