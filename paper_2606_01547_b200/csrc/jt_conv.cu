// jt_conv.cu -- step 5a: direct PSF convolution (definition P; PAPER.md:55 third step; PAPER.md:110-114 shapes).
//
//   out[j][i] = sum_a sum_b Kf[a][b] tile[jl+a][il+b],  Kf = kernel flipped in both axes (true convolution),
//   tile = image window with a (ky-1, kx-1) halo in shared memory, zero outside the image.
//
// Design (B200): the FMA pipes are the roofline (FFMA2: 128 FMA/clk/SM, DFMA: 64), and on sm_100 every 32-bit word a
// load writes into the register file costs one FMA issue cycle (the result port is shared: measured with the r01
// probes, 1 LDS.128 + 1 LDS.64 per 8 FFMA2 -> 46 of 63.5 lanes/clk).  So the kernel keeps loaded words per FMA minimal:
//   * TAPS never touch the register file: the flipped kernel sits in __constant__ memory, is fetched by the uniform
//     datapath (LDCU -> uniform registers) and enters FFMA2 / DFMA as a uniform-register operand.
//   * a thread owns OY rows x 2 adjacent columns of outputs and slides a register window of OY tile pairs down the
//     tile: one 64-/128-bit shared load per (kernel-column pair, kernel row) feeds 4 OY FMAs.
//   * float: sm_100 packed FMA (fma.rn.f32x2 -> FFMA2): the two output columns of a row share a 64-bit accumulator.
//   * the halo tile arrives by ONE TMA tiled load (cp.async.bulk.tensor, out-of-bounds elements zero-filled by the
//     hardware = the zero padding of definition P); plain-load fallback when the image pitch is not 16-byte aligned.
//   * parallelism for big kernels / small images: the kernel COLUMN PAIRS of a tile are dealt to Z CTAs (each stages
//     only the tile columns its pairs touch); every CTA publishes its partial sums to the workspace (L2) and the last
//     one to arrive for the tile adds all Z in rank order (deterministic).  No CTA waits for another, so the grid runs
//     in any number of waves.  (A thread-block-cluster version with the reduction through distributed shared memory
//     measured 10-35 % slower: the cluster barrier makes every CTA wait for the slowest SM.)
//   * __constant__ memory holds 60 KB of taps; larger kernels run as several launches over bands of kernel ROWS, each
//     adding its rows to `out` (the bands also bound the tile height, so any kernel size fits).
// A small prep kernel writes the flipped / paired tap table to the workspace; cudaMemcpyToSymbolAsync moves each
// launch's share into the constant bank (stream-ordered).
#include <cuda.h>
#include <cudaTypedefs.h>
#include <mutex>
#include <math.h>
#include "jt_conv.cuh"

namespace jt {

constexpr int kConvTW = 64;                        // output columns per CTA: 32 lanes x 2
constexpr int kTapBytes = 60 * 1024;               // taps of one launch (constant bank 3 holds 64 KB per module)
constexpr size_t kSmemPerSM = 227 * 1024;
constexpr int kMaxSplit = 16;                      // column-pair shares per tile (workspace reduction)

__constant__ __align__(16) unsigned char c_taps[kTapBytes];

// Tap table of one launch (a band of kb kernel rows, all npairs kernel-column pairs), elements of T:
//   E[m'][a][h],  m' in [0, npairs], a in [0, kb), h in {0,1}:   E[0] = 0,  E[m+1][a] = (Kf[a][2m], Kf[a][2m+1])
// with Kf[a][b] = K[ky-1-a][kx-1-(b-pad)], zero outside 0 <= b - pad < kx.  Pair m of the sweep reads E[m+1][a] (both)
// and E[m][a][1].
// The tile's first column must be an EVEN image column: the pair loads stay aligned and the TMA box can start on a
// 16-byte boundary (a TMA requirement: coordinate[0] * sizeof(T) must be a multiple of 16).  With an odd halo kx/2
// that is arranged either by xoff = 1 -- the CTA's 64 output columns start one column to the left (free unless it
// costs an extra tile column) -- or by pad = 1: a zero column in FRONT of the kernel (one more column pair).
__host__ __device__ inline size_t tap_elems_per_launch(int npairs, int kb) { return (size_t)(npairs + 1) * kb * 2; }
// column 0 of a thread needs taps b <= kx' - 1 = 2m + 1, column 1 needs b = 2m - 1 <= kx' - 1 (kx' = kx + pad)
__host__ __device__ inline int conv_npairs(int kx, int pad) { return (kx + pad) / 2 + 1; }
inline void conv_parity(int nx, int kx, int* pad, int* xoff) {
    const bool odd = (kx / 2) & 1;
    *xoff = (odd && (nx + 1 + kConvTW - 1) / kConvTW == (nx + kConvTW - 1) / kConvTW) ? 1 : 0;
    *pad = (odd && !*xoff) ? 1 : 0;
}

// Balanced split of npairs column pairs over Z ranks in units of `unit` pairs: rank z gets floor or ceil of units / Z.
__host__ __device__ inline void rank_share(int npairs, int unit, int Z, int z, int* m_lo, int* m_cnt) {
    const int nu = (npairs + unit - 1) / unit, base = nu / Z, rem = nu - base * Z;
    const int u_lo = z * base + (z < rem ? z : rem), u_cnt = base + (z < rem ? 1 : 0);
    *m_lo = u_lo * unit;
    const int hi = (u_lo + u_cnt) * unit;
    *m_cnt = (hi < npairs ? hi : npairs) - *m_lo;
}

template <typename T>
__global__ void __launch_bounds__(256) k_conv_taps(int ky, int kx, int pad, int kb, int n_launches, const T* __restrict__ K,
                                                   T* __restrict__ table, unsigned int* __restrict__ counter, int n_counters) {
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_counters; i += gridDim.x * blockDim.x) counter[i] = 0u;
    const int npairs = conv_npairs(kx, pad);
    const int per = (int)tap_elems_per_launch(npairs, kb);
    const int total = per * n_launches;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const int l = idx / per, rem = idx - l * per;
        const int h = rem & 1, e = rem >> 1, mp = e / kb, a = e - mp * kb;
        const int ag = l * kb + a, b = 2 * (mp - 1) + h - pad;
        T v = (T)0;
        if (mp >= 1 && ag < ky && b >= 0 && b < kx) v = __ldg(&K[(ky - 1 - ag) * kx + (kx - 1 - b)]);
        table[idx] = v;
    }
}

template <typename T>
struct ConvArgs {
    int ny, nx, ky, kx;
    int kb;                  // row pitch of the tap table = kernel rows per launch
    int a_lo, kbz;           // first flipped-kernel row of this launch and the number of rows it sums (<= kb)
    int unit;                // the column pairs are dealt to the Z cluster ranks in units of `unit` pairs (2 in float: 16-byte tile columns)
    int tws, ths;            // tile pitch (elements) and tile rows = TH + kb - 1
    int pad, xoff;           // parity fix for an odd halo (see tap_elems_per_launch): zero column in front of the kernel / outputs start at column -1
    int shift;               // extra tile columns on the left that bring the TMA box to a 16-byte boundary (even)
    int tiles_y;             // tile rows per image; blockIdx.x = image * tiles_y + tile row, blockIdx.y = tile column
    int accumulate;          // add to the values already in `out` (second and later launches of a call)
    int use_tma;
    T* partial;              // Z > 1: [tile][Z][OY][threads] pairs of partial sums (workspace)
    unsigned int* counter;   // Z > 1: one arrival counter per tile, zero on entry, zero again on exit
    long long img_stride, out_stride;     // elements between consecutive images of a batch
    const T* img;
    T* out;
};

// ---- per-dtype pieces: window element, accumulator of one output row (two adjacent columns), one sweep step ----
template <typename T> struct UrOps;

template <> struct UrOps<double> {
    using Win = double2;
    struct Acc { double c0, c1; };
    static __device__ __forceinline__ Acc zero() { return {0.0, 0.0}; }
    // k0 = Kf[a][2m], k1 = Kf[a][2m+1], km = Kf[a][2m-1]:  col0 += k0 v.x + k1 v.y,  col1 += km v.x + k0 v.y
    static __device__ __forceinline__ void step(Acc& v, const Win& w, double km, double k0, double k1) {
        v.c0 = fma(k0, w.x, v.c0);
        v.c1 = fma(km, w.x, v.c1);
        v.c0 = fma(k1, w.y, v.c0);
        v.c1 = fma(k0, w.y, v.c1);
    }
    static __device__ __forceinline__ double col0(const Acc& v) { return v.c0; }
    static __device__ __forceinline__ double col1(const Acc& v) { return v.c1; }
    static __device__ __forceinline__ void add(Acc& v, double c0, double c1) { v.c0 += c0; v.c1 += c1; }
};

// float: one 64-bit accumulator per output row, low half = column 1, high half = column 0, so that both tap pairs are
// in ascending memory order: (Kf[2m-1], Kf[2m]) multiplies v.x and (Kf[2m], Kf[2m+1]) multiplies v.y.
template <> struct UrOps<float> {
    using Win = float2;
    using Acc = unsigned long long;
    static __device__ __forceinline__ Acc zero() { return 0ull; }
    static __device__ __forceinline__ unsigned long long pack(float lo, float hi) {
        unsigned long long d;
        asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
        return d;
    }
    static __device__ __forceinline__ void step(Acc& v, const Win& w, float km, float k0, float k1) {
        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(v) : "l"(pack(km, k0)), "l"(pack(w.x, w.x)));
        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(v) : "l"(pack(k0, k1)), "l"(pack(w.y, w.y)));
    }
    static __device__ __forceinline__ float col0(const Acc& v) { return __uint_as_float((unsigned)(v >> 32)); }
    static __device__ __forceinline__ float col1(const Acc& v) { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
    static __device__ __forceinline__ void add(Acc& v, float c0, float c1) { v = pack(col1(v) + c1, col0(v) + c0); }
};

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned phase) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(phase) : "memory");
}
// one TMA tiled load: box (tws, ths, 1) of the [B][ny][nx] image at (col, row, image); OOB elements arrive as zeros
__device__ __forceinline__ void tma_load_tile(void* dst, const CUtensorMap* map, unsigned long long* bar, int col, int row, int image) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
            (unsigned)__cvta_generic_to_shared(dst)),
        "l"(map), "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(col), "r"(row), "r"(image)
        : "memory");
}

// One kernel-column pair against kbz kernel rows.  win holds tile rows 0 .. OY-2 of this pair on entry; the first OY-1
// rows of the NEXT pair are loaded into nxt while this pair sweeps (read two columns past the rank's share at its last
// pair: still inside the tile, never used).  prev = E[m] (Kf[.][2m-1] in slot 1), prev + 2 kb = E[m+1] (Kf[.][2m], Kf[.][2m+1]).
template <typename T, int OY>
__device__ __forceinline__ void sweep_pair(typename UrOps<T>::Acc (&acc)[OY], typename UrOps<T>::Win (&win)[OY],
                                           typename UrOps<T>::Win (&nxt)[OY], const T* __restrict__ tp, int tws,
                                           const T* __restrict__ prev, int kb, int kbz) {
    using O = UrOps<T>;
    using Win = typename O::Win;
    const T* cur = prev + (size_t)kb * 2;
    const T* wp = tp + (size_t)(OY - 1) * tws;
#pragma unroll
    for (int r = 0; r < OY - 1; ++r) nxt[r] = *reinterpret_cast<const Win*>(tp + 2 + (size_t)r * tws);
    const int n_chunks = kbz / OY, n_tail = kbz - n_chunks * OY;
#pragma unroll 1
    for (int c = 0; c < n_chunks; ++c) {
#pragma unroll
        for (int aa = 0; aa < OY; ++aa) {
            win[(aa + OY - 1) % OY] = *reinterpret_cast<const Win*>(wp);
            wp += tws;
            const T km = prev[2 * aa + 1], k0 = cur[2 * aa], k1 = cur[2 * aa + 1];
#pragma unroll
            for (int r = 0; r < OY; ++r) O::step(acc[r], win[(aa + r) % OY], km, k0, k1);
        }
        prev += 2 * OY;
        cur += 2 * OY;
    }
#pragma unroll
    for (int aa = 0; aa < OY - 1; ++aa) {                        // tail rows (warp-uniform exit)
        if (aa >= n_tail) break;
        win[(aa + OY - 1) % OY] = *reinterpret_cast<const Win*>(wp);
        wp += tws;
        const T km = prev[2 * aa + 1], k0 = cur[2 * aa], k1 = cur[2 * aa + 1];
#pragma unroll
        for (int r = 0; r < OY; ++r) O::step(acc[r], win[(aa + r) % OY], km, k0, k1);
    }
}

template <typename T, int OY>
__global__ void __launch_bounds__(256) k_conv_ur(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ ConvArgs<T> a) {
    using O = UrOps<T>;
    using Win = typename O::Win;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long s_bar;
    T* tile = reinterpret_cast<T*>(smem_raw);
    const int nthr = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int TH = (nthr >> 5) * OY;
    const int zl = blockIdx.z;                                   // which share of the tile's column pairs
    const int image = blockIdx.x / a.tiles_y, ty = blockIdx.x - image * a.tiles_y;
    const int i0 = blockIdx.y * kConvTW - a.xoff, j0 = ty * TH;
    int m_lo, m_cnt;                                             // this rank's share of the column pairs (>= 1)
    rank_share(conv_npairs(a.kx, a.pad), a.unit, gridDim.z, zl, &m_lo, &m_cnt);
    const int kbz = a.kbz;
    const int col0 = i0 - (a.kx / 2 + a.pad) - a.shift + 2 * m_lo, row0 = j0 - (a.ky - 1 - a.ky / 2) + a.a_lo;
    const int tws = a.tws;

    // ---- halo tile ----
    if (a.use_tma) {
        if (tid == 0) mbar_init(&s_bar, 1);
        __syncthreads();
        if (tid == 0) {
            mbar_expect_tx(&s_bar, (unsigned)((size_t)a.ths * tws * sizeof(T)));
            tma_load_tile(tile, &tmap, &s_bar, col0, row0, image);
        }
        mbar_wait(&s_bar, 0);
    } else {
        const T* img = a.img + (size_t)image * a.img_stride;
        for (int r = warp; r < a.ths; r += nthr >> 5) {
            const int gj = row0 + r;
            const bool rok = gj >= 0 && gj < a.ny;
            for (int c = lane; c < tws; c += 32) {
                const int gi = col0 + c;
                tile[(size_t)r * tws + c] = (rok && gi >= 0 && gi < a.nx) ? __ldg(&img[(size_t)gj * a.nx + gi]) : (T)0;
            }
        }
        __syncthreads();
    }

    // ---- sweep: kernel-column pairs outer, kernel rows inner with a sliding register window ----
    typename O::Acc acc[OY];
#pragma unroll
    for (int r = 0; r < OY; ++r) acc[r] = O::zero();
    const int kb = a.kb;
    const T* E = reinterpret_cast<const T*>(c_taps) + (size_t)m_lo * kb * 2;
    const T* tp0 = tile + (size_t)(warp * OY) * tws + a.shift + 2 * lane;
    Win wA[OY], wB[OY];                                         // the window that sweeps, and the next pair's first rows
#pragma unroll
    for (int r = 0; r < OY - 1; ++r) wA[r] = *reinterpret_cast<const Win*>(tp0 + (size_t)r * tws);
#pragma unroll 1
    for (int m = 0; m < m_cnt; ++m) {
        sweep_pair<T, OY>(acc, wA, wB, tp0 + 2 * m, tws, E + (size_t)m * kb * 2, kb, kbz);
#pragma unroll
        for (int r = 0; r < OY - 1; ++r) wA[r] = wB[r];
    }

    // ---- partial sums of the Z column-pair shares of a tile, added in rank order (deterministic) ----
    const int Z = gridDim.z;
    if (Z > 1) {
        // every CTA publishes its sums (L2); the last CTA to arrive for the tile adds all Z of them in rank order.
        // No CTA ever waits for another, so the grid may run in any number of waves.
        __shared__ int s_last;
        const size_t tile_id = (size_t)blockIdx.x * gridDim.y + blockIdx.y;
        Win* mine = reinterpret_cast<Win*>(a.partial) + (tile_id * Z + zl) * OY * nthr;
#pragma unroll
        for (int r = 0; r < OY; ++r) {
            Win v;
            v.x = O::col0(acc[r]);
            v.y = O::col1(acc[r]);
            __stcg(&mine[r * nthr + tid], v);
        }
        __threadfence();
        __syncthreads();
        if (tid == 0) s_last = atomicAdd(&a.counter[tile_id], 1u) == (unsigned)(Z - 1);
        __syncthreads();
        if (!s_last) return;
        __threadfence();
#pragma unroll
        for (int r = 0; r < OY; ++r) acc[r] = O::zero();
        const Win* all = reinterpret_cast<const Win*>(a.partial) + tile_id * Z * OY * nthr;
        for (int z = 0; z < Z; ++z) {
#pragma unroll
            for (int r = 0; r < OY; ++r) {
                const Win v = __ldcg(&all[(z * OY + r) * nthr + tid]);
                O::add(acc[r], v.x, v.y);
            }
        }
        if (tid == 0) a.counter[tile_id] = 0u;                   // clean for the next launch of this call / the next call
    }

    T* out = a.out + (size_t)image * a.out_stride;
    const int i = i0 + 2 * lane;
#pragma unroll
    for (int r = 0; r < OY; ++r) {
        const int j = j0 + warp * OY + r;
        if (j < a.ny) {
            T* o = out + (size_t)j * a.nx + i;
            if (i >= 0 && i < a.nx) o[0] = a.accumulate ? o[0] + O::col0(acc[r]) : O::col0(acc[r]);
            if (i + 1 < a.nx) o[1] = a.accumulate ? o[1] + O::col1(acc[r]) : O::col1(acc[r]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ host side
struct ConvPlan {
    int OY, NW, kb, launches, Z, mz, unit, occ;
    int tws, ths, shift, pad, xoff, tiles_x, tiles_y;
    size_t smem, table_bytes, counter_bytes, partial_bytes;
    double est_us;
    bool ok;
};

static const int kOYs[] = {8, 7, 6, 5, 4};
// double: beyond OY = 6 the taps of an unrolled chunk no longer fit the 63 uniform registers and ptxas falls back to
// per-thread LDC loads (register-file traffic again); float taps are half the size
constexpr int kMaxOYf64 = 6;
// registers per thread of k_conv_ur<T, OY> (ptxas -v, rounded up), for the occupancy estimate of the planner
static int conv_regs(jt_dtype d, int OY) { return d == JT_F64 ? 16 * OY : 16 + 6 * OY; }   // 60 / 75 / 93;  40 ... 64

// Launch plan and time model (also behind JT_CONV_AUTO), calibrated on B200: a (kernel-column
// pair, kernel row) step of one warp occupies its scheduler's FMA pipe for 4 OY (float: 2 OY FFMA2) or 8 OY (double:
// 4 OY DFMA) cycles plus the window load's register write-back; an SM runs ceil(CTAs / 148) CTAs' worth of such steps
// on 4 schedulers, at an efficiency that grows with the warps resident per scheduler.
static ConvPlan plan_conv_search(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx) {
    ConvPlan best = {};
    best.ok = false;
    const size_t sz = dtype_size(d);
    int pad, xoff;
    conv_parity(nx, kx, &pad, &xoff);
    const int npairs = conv_npairs(kx, pad);
    const int q = 16 / (int)sz;                                 // elements per 16 bytes
    const int halo = kx / 2 + pad + xoff;                       // even: image columns left of the CTA's column 0 in the tile
    const int shift = ((-halo) % q + q) % q;                    // even: 0, or 2 in float when halo % 4 == 2
    int L_min = 1;
    while (L_min <= ky && tap_elems_per_launch(npairs, (ky + L_min - 1) / L_min) * sz > (size_t)kTapBytes) ++L_min;
    if (L_min > ky) return best;                                // one kernel row does not fit the constant bank
    for (int OY : kOYs) {
        if (d == JT_F64 && OY > kMaxOYf64) continue;
        for (int NW = 8; NW >= 2; NW -= 2) {                    // even: odd warp counts measured 5-15 % slower
            const int TH = NW * OY;
            const int tiles_x = (nx + xoff + kConvTW - 1) / kConvTW, tiles_y = (ny + TH - 1) / TH;
            const int64_t tiles = (int64_t)tiles_x * tiles_y * B;
            if ((int64_t)tiles_y * B > 0x7fffffffLL || tiles_x > 65535) continue;
            for (int L = L_min; L <= L_min + 2 && L <= ky; ++L) {
                const int kb = (ky + L - 1) / L;
                if (L > L_min && (ky + kb - 1) / kb != L) continue;
                const int ths = TH + kb - 1;
                if (ths > 256) continue;
                const int unit = sz == 4 ? 2 : 1;               // float: every rank's first tile column stays 16-byte aligned
                for (int Z = 1; Z <= kMaxSplit && Z * unit <= npairs + unit - 1; ++Z) {
                    int m_lo, mz;
                    rank_share(npairs, unit, Z, 0, &m_lo, &mz);  // rank 0 has the largest share
                    const int tws = (int)(align_up((size_t)(shift + kConvTW + 2 * mz - 2) * sz, 16) / sz);
                    const size_t smem = align_up((size_t)ths * tws * sz, 128);
                    const size_t stage = (size_t)OY * NW * 32 * 2 * sz;
                    if (smem + 1024 > kSmemPerSM) continue;
                    int occ = (int)(kSmemPerSM / (smem + 1024));
                    const int occ_r = 65536 / (conv_regs(d, OY) * NW * 32);
                    if (occ_r < occ) occ = occ_r;
                    if (64 / NW < occ) occ = 64 / NW;
                    if (occ > 32) occ = 32;
                    if (occ < 1) continue;
                    // time model, calibrated on B200
                    const double step = (d == JT_F64 ? 8.0 * OY + 4.0 : 4.0 * OY + 2.0);    // FMA pipe cycles per (pair, row) of a warp
                    const double pre = (OY - 1) * (d == JT_F64 ? 4.0 : 2.0) + 30.0;          // per pair: window preload + loop set-up
                    const int64_t ctas = tiles * Z;
                    const double n = (double)ctas / kNumSMs;                                 // CTAs per SM
                    const double n_ceil = (double)((ctas + kNumSMs - 1) / kNumSMs);
                    const double n_eff = n_ceil < n + 0.6 ? n_ceil : n + 0.6;                // dynamic dispatch: the busiest SM
                    const double conc = (n_ceil < occ ? n_ceil : occ) * NW / 4.0;            // warps per scheduler
                    // one wave: the CTAs' warps sit on the 4 schedulers as dealt (the busiest one decides); several waves even out
                    const double res_warps = (n_ceil < occ ? n_ceil : occ) * NW;
                    const double smsp = n_ceil <= occ ? ceil(res_warps / 4.0) / (res_warps / 4.0) : 1.0;
                    const double eff = (d == JT_F64 ? 0.97 : 0.86) / smsp *
                                       (conc >= 4.0 ? 1.0 : (conc >= 3.0 ? 0.96 : (conc >= 2.0 ? 0.88 : (conc >= 1.0 ? 0.6 : 0.6 * conc))));
                    const double t_cta = (NW / 4.0) * ((double)npairs / Z) * (kb * step + pre);
                    const double t_fix = 1200.0 + (double)smem / 64.0 + (Z > 1 ? (double)stage / 16.0 : 0.0);   // tile fill + epilogue (partial sums out and back), mostly overlapped
                    const double cyc = n_eff * (t_cta / eff + 0.3 * t_fix) + 0.7 * t_fix + 1500.0;
                    const double us = L * (cyc / 1.9e3 + 2.5) + 2.5;
                    if (!best.ok || us < best.est_us) {
                        const bool ws = Z > 1;
                        best = {OY, NW, kb, L, Z, mz, unit, occ, tws, ths, shift, pad, xoff, tiles_x, tiles_y, smem,
                                align_up(tap_elems_per_launch(npairs, kb) * sz * L, 256),
                                ws ? align_up((size_t)tiles * sizeof(unsigned int), 256) : 0,
                                ws ? align_up((size_t)tiles * Z * stage, 256) : 0, us, true};
                    }
                }
            }
        }
    }
    return best;
}

// The search visits ~1000 (OY, warps, bands, Z) combinations and an API call asks for the plan several times
// (supported? / estimate / workspace / launch): the last few answers are kept per host thread.
static ConvPlan plan_conv(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx) {
    struct Slot { int d; int64_t B; int ny, nx, ky, kx; ConvPlan p; bool used; };
    static thread_local Slot cache[4] = {};
    static thread_local int next = 0;
    for (const Slot& c : cache)
        if (c.used && c.d == (int)d && c.B == B && c.ny == ny && c.nx == nx && c.ky == ky && c.kx == kx) return c.p;
    Slot& c = cache[next];
    next = (next + 1) & 3;
    c = {(int)d, B, ny, nx, ky, kx, plan_conv_search(d, B, ny, nx, ky, kx), true};
    return c.p;
}

// ------------------------------------------------------------------------------------------------ small problems
// Launch-latency-bound shapes (C0: 60 x 60 (x) 11 x 11 is 0.4 M FMAs; the paper's 60 x 60 sweep): ONE launch instead of
// tap kernel + constant-bank copy + sweep kernel.  A CTA of 64 threads owns a 64 x 8 output tile, stages the packed
// taps (jt_conv.cuh) and its halo tile in shared memory itself and runs the register-window sweep of the batch kernel.
// The taps do not depend on the image, so they are staged BEFORE the grid dependency is awaited: launched as a
// programmatic dependent of the ray-tracing kernel, this part overlaps its tail.
constexpr int kSmallOY = 4, kSmallNW = 2, kSmallTH = kSmallOY * kSmallNW;
constexpr size_t kSmallMaxSmem = 96 * 1024;
constexpr double kSmallMaxFma = 2.0e7;

template <typename T>
__global__ void __launch_bounds__(kSmallNW * 32) k_conv_small(int ny, int nx, int ky, int kx, int kyp, int tws, int ths,
                                                              const T* __restrict__ img, const T* __restrict__ ker,
                                                              T* __restrict__ out) {
    extern __shared__ __align__(128) unsigned char smem_small[];   // (its own name: `smem_raw` is the TMA kernel's, 128-byte aligned)
    const int npairs = (kx + 1) / 2, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    T* Kq = reinterpret_cast<T*>(smem_small);
    T* tile = Kq + (size_t)npairs * kyp * 4;
    stage_taps<T>(Kq, ker, ky, kx, kyp, 0, npairs, tid, kSmallNW * 32);
    cudaGridDependencySynchronize();                           // the image of the previous kernel is complete
    const int i0 = blockIdx.x * kConvTW, j0 = blockIdx.y * kSmallTH, hy = ky / 2, hx = kx / 2;
    for (int idx = tid; idx < ths * tws; idx += kSmallNW * 32) {
        const int r = idx / tws, c = idx - r * tws;
        const int gj = j0 - hy + r, gi = i0 - hx + c;
        tile[idx] = (gj >= 0 && gj < ny && gi >= 0 && gi < nx) ? __ldg(&img[(size_t)gj * nx + gi]) : (T)0;
    }
    __syncthreads();
    ConvAcc<T, kSmallOY> acc;
    acc.zero();
    acc.template sweep<false>(tile + (size_t)(warp * kSmallOY) * tws + 2 * lane, tws, Kq, kyp, npairs);
    const int i = i0 + 2 * lane;
#pragma unroll
    for (int r = 0; r < kSmallOY; ++r) {
        const int j = j0 + warp * kSmallOY + r;
        if (j < ny) {
            if (i < nx) out[(size_t)j * nx + i] = acc.col0(r);
            if (i + 1 < nx) out[(size_t)j * nx + i + 1] = acc.col1(r);
        }
    }
}

struct SmallPlan { int kyp, tws, ths; size_t smem; double est_us; bool ok; };
static SmallPlan plan_small(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx) {
    SmallPlan p = {};
    const size_t sz = dtype_size(d);
    p.kyp = (ky + kSmallOY - 1) / kSmallOY * kSmallOY;
    p.tws = kConvTW + kx - 1;                                  // even (kx odd): pair loads stay aligned
    p.ths = kSmallTH + p.kyp - 1;
    p.smem = ((size_t)((kx + 1) / 2) * p.kyp * 4 + (size_t)p.tws * p.ths) * sz;
    p.ok = B == 1 && (double)ny * nx * ky * kx <= kSmallMaxFma && p.smem <= kSmallMaxSmem;
    // measured on B200 (conv sweep, 60^2 ... 200^2): 3 us + a CTA's FMAs at 12.8 (double) / 24 (float) per clock, per wave
    const double ctas = (double)((nx + kConvTW - 1) / kConvTW) * ((ny + kSmallTH - 1) / kSmallTH);
    const double per_cta = (double)kConvTW * kSmallTH * ((kx + 1) / 2 * 2) * p.kyp;
    p.est_us = 3.0 + ceil(ctas / (kNumSMs * 2.0)) * per_cta * (d == JT_F64 ? 4.1e-5 : 2.2e-5);
    return p;
}
// the one-launch kernel when it is expected to beat the constant-bank kernel (tiny kernels on small images)
static bool use_small(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx, SmallPlan* sp);

template <typename T>
static jt_status conv_small_t(const SmallPlan& p, int ny, int nx, const T* img, int ky, int kx, const T* ker, T* out, cudaStream_t st) {
    auto kern = k_conv_small<T>;
    static PerDeviceOnce attr;                          // once per instantiation and device
    if (attr.needed()) {
        JT_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmallMaxSmem));
        attr.mark();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((nx + kConvTW - 1) / kConvTW), (unsigned)((ny + kSmallTH - 1) / kSmallTH));
    cfg.blockDim = dim3(kSmallNW * 32);
    cfg.dynamicSmemBytes = p.smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    JT_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, ny, nx, ky, kx, p.kyp, p.tws, p.ths, img, ker, out));
    JT_LAUNCH_CHECK();
    return JT_OK;
}

bool conv_direct_supported(jt_dtype d, int ny, int nx, int ky, int kx) { return plan_conv(d, 1, ny, nx, ky, kx).ok; }
size_t conv_direct_workspace_bytes(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx) {
    const ConvPlan p = plan_conv(d, B, ny, nx, ky, kx);
    return p.ok ? p.table_bytes + p.counter_bytes + p.partial_bytes : 0;
}
static bool use_small(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx, SmallPlan* sp) {
    *sp = plan_small(d, B, ny, nx, ky, kx);
    if (!sp->ok) return false;
    const ConvPlan p = plan_conv(d, B, ny, nx, ky, kx);
    return !p.ok || sp->est_us < p.est_us;
}
double conv_direct_estimate_us(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx) {
    SmallPlan sp;
    if (use_small(d, B, ny, nx, ky, kx, &sp)) return sp.est_us;
    const ConvPlan p = plan_conv(d, B, ny, nx, ky, kx);
    return p.ok ? p.est_us : 1e30;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
static PFN_cuTensorMapEncodeTiled_v12000 tensor_map_encoder() {
    static PFN_cuTensorMapEncodeTiled_v12000 fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (PFN_cuTensorMapEncodeTiled_v12000)p;
    });
    return fn;
}

template <typename T>
static bool make_tensor_map(CUtensorMap* map, const T* img, int64_t B, int ny, int nx, int tws, int ths) {
    auto enc = tensor_map_encoder();
    if (!enc) return false;
    const size_t sz = sizeof(T);
    if (((uintptr_t)img & 15) || ((size_t)nx * sz) % 16 || (B > 1 && ((size_t)nx * ny * sz) % 16) || tws > 256 || ths > 256)
        return false;
    const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)B};
    const cuuint64_t strides[2] = {(cuuint64_t)nx * sz, (cuuint64_t)nx * ny * sz};
    const cuuint32_t box[3] = {(cuuint32_t)tws, (cuuint32_t)ths, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = enc(map, sz == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)img, dims,
                           strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// what launch_conv_direct would do for these arguments (jt_psf_convolve_plan); mirrors its decisions, enqueues nothing
void conv_direct_describe(jt_dtype d, int64_t B, int ny, int nx, int ky, int kx, const void* img, jt_conv_plan* out) {
    SmallPlan sp;
    out->method = JT_CONV_DIRECT;
    if (use_small(d, B, ny, nx, ky, kx, &sp)) {
        out->path = JT_PATH_CONV_SMALL;
        out->z_split = 1; out->row_bands = 1; out->oy = kSmallOY; out->warps = kSmallNW;
        out->est_us = sp.est_us;
        return;
    }
    const ConvPlan p = plan_conv(d, B, ny, nx, ky, kx);
    const size_t sz = dtype_size(d);
    out->path = JT_PATH_CONV_TILE;
    out->tma = !(((uintptr_t)img & 15) || ((size_t)nx * sz) % 16 || (B > 1 && ((size_t)nx * ny * sz) % 16) || p.tws > 256 ||
                 p.ths > 256);                                   // make_tensor_map's conditions
    out->z_split = p.Z; out->row_bands = p.launches; out->oy = p.OY; out->warps = p.NW;
    out->est_us = p.est_us;
}

// The constant bank is one per device: calls on different streams take turns through an event (the library's only
// cross-call state besides the error code; not used while the stream is being captured into a graph).
static std::mutex g_const_mu;
static cudaEvent_t g_const_ev[64] = {};

template <typename T, int OY>
static jt_status launch_ur(const ConvPlan& p, const CUtensorMap& map, const ConvArgs<T>& a, int64_t B, cudaStream_t st) {
    const int z = p.Z;
    auto kern = k_conv_ur<T, OY>;
    static PerDeviceOnce attr;                          // once per instantiation and device: allow the full 227 KB
    if (attr.needed()) {
        JT_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSmemPerSM - 1024)));
        attr.mark();
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(p.tiles_y * B), (unsigned)p.tiles_x, (unsigned)z);
    cfg.blockDim = dim3((unsigned)(p.NW * 32));
    cfg.dynamicSmemBytes = p.smem;
    cfg.stream = st;
    JT_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, map, a));
    JT_LAUNCH_CHECK();
    return JT_OK;
}

template <typename T>
static jt_status conv_direct_t(jt_dtype d, int64_t B, int ny, int nx, const T* img, int ky, int kx, const T* ker,
                               void* workspace, T* out, cudaStream_t st) {
    const ConvPlan p = plan_conv(d, B, ny, nx, ky, kx);
    if (!p.ok) return JT_ERR_UNSUPPORTED;
    T* table = (T*)workspace;                                   // [tap table][tile counters][partial sums]
    unsigned int* counter = (unsigned int*)((char*)workspace + p.table_bytes);
    const int npairs = conv_npairs(kx, p.pad);
    const size_t per_launch = tap_elems_per_launch(npairs, p.kb);
    {
        const size_t total = per_launch * p.launches;
        int blocks = (int)((total + 255) / 256);
        if (blocks > 4 * kNumSMs) blocks = 4 * kNumSMs;
        k_conv_taps<T><<<blocks, 256, 0, st>>>(ky, kx, p.pad, p.kb, p.launches, ker, table, counter,
                                               (int)(p.counter_bytes / sizeof(unsigned int)));
        JT_LAUNCH_CHECK();
    }
    CUtensorMap map;
    memset(&map, 0, sizeof(map));
    ConvArgs<T> a = {};
    a.ny = ny; a.nx = nx; a.ky = ky; a.kx = kx; a.kb = p.kb; a.unit = p.unit;
    a.tws = p.tws; a.ths = p.ths; a.shift = p.shift; a.pad = p.pad; a.xoff = p.xoff; a.tiles_y = p.tiles_y;
    a.use_tma = make_tensor_map<T>(&map, img, B, ny, nx, p.tws, p.ths) ? 1 : 0;
    a.img_stride = (long long)ny * nx; a.out_stride = (long long)ny * nx;
    a.img = img; a.out = out;
    a.counter = counter;
    a.partial = (T*)((char*)workspace + p.table_bytes + p.counter_bytes);

    int dev = 0;
    JT_CUDA_TRY(cudaGetDevice(&dev));
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    JT_CUDA_TRY(cudaStreamIsCapturing(st, &cs));
    const bool chain = cs == cudaStreamCaptureStatusNone && dev >= 0 && dev < 64;
    std::lock_guard<std::mutex> lock(g_const_mu);
    if (chain) {
        if (!g_const_ev[dev]) JT_CUDA_TRY(cudaEventCreateWithFlags(&g_const_ev[dev], cudaEventDisableTiming));
        else JT_CUDA_TRY(cudaStreamWaitEvent(st, g_const_ev[dev], 0));
    }
    jt_status s = JT_OK;
    for (int l = 0; l < p.launches && s == JT_OK; ++l) {
        JT_CUDA_TRY(cudaMemcpyToSymbolAsync(c_taps, table + (size_t)l * per_launch, per_launch * sizeof(T), 0,
                                            cudaMemcpyDeviceToDevice, st));
        a.a_lo = l * p.kb;
        a.kbz = ky - a.a_lo < p.kb ? ky - a.a_lo : p.kb;
        a.accumulate = l > 0 ? 1 : 0;
        switch (p.OY) {
            case 4: s = launch_ur<T, 4>(p, map, a, B, st); break;
            case 5: s = launch_ur<T, 5>(p, map, a, B, st); break;
            case 6: s = launch_ur<T, 6>(p, map, a, B, st); break;
            case 7: if constexpr (sizeof(T) == 4) { s = launch_ur<T, 7>(p, map, a, B, st); break; }
            case 8: if constexpr (sizeof(T) == 4) { s = launch_ur<T, 8>(p, map, a, B, st); break; }
            default: s = JT_ERR_UNSUPPORTED;
        }
    }
    if (chain) JT_CUDA_TRY(cudaEventRecord(g_const_ev[dev], st));
    return s;
}

jt_status launch_conv_direct(jt_dtype dtype, int64_t B, int ny, int nx, const void* img, int ky, int kx, const void* ker,
                             void* workspace, void* out, cudaStream_t st) {
    SmallPlan sp;
    if (use_small(dtype, B, ny, nx, ky, kx, &sp))
        return dtype == JT_F32 ? conv_small_t<float>(sp, ny, nx, (const float*)img, ky, kx, (const float*)ker, (float*)out, st)
                               : conv_small_t<double>(sp, ny, nx, (const double*)img, ky, kx, (const double*)ker, (double*)out, st);
    return dtype == JT_F32 ? conv_direct_t<float>(dtype, B, ny, nx, (const float*)img, ky, kx, (const float*)ker, workspace, (float*)out, st)
                           : conv_direct_t<double>(dtype, B, ny, nx, (const double*)img, ky, kx, (const double*)ker, workspace, (double*)out, st);
}

}  // namespace jt
