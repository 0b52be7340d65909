// jt_conv.cu -- step 5a: direct PSF convolution (definition P; PAPER.md:55 third step).
//
// out[j][i] = sum_a sum_b Kf[a][b] tile[jl+a][il+b],  Kf = kernel flipped in both axes (true convolution),
// tile = image window with a (ky-1, kx-1) halo staged in shared memory, zero outside the image.
// CTA = NW warps; tile = 64 columns x NW*OY rows; a thread owns OY x 2 outputs (jt_conv.cuh: pair loads, register
// window, 4 OY FMAs per shared load; float: packed FFMA2).  The flipped kernel is staged in shared memory by the CTA itself (no separate
// flip launch, no workspace), whole when it fits beside the tile, else in bands of kernel-column pairs.
// The host picks (OY, NW) so that the CTA count fills 148 SMs with the fewest, fullest waves.
#include "jt_conv.cuh"

namespace jt {

constexpr int kConvTW = 64;
constexpr size_t kMaxSmem = 227 * 1024;

template <typename T, int OY>
__global__ void __launch_bounds__(256) k_conv_direct(int ny, int nx, const T* __restrict__ img, int ky, int kx, int kyp,
                                                     int band_pairs, const T* __restrict__ K, T* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nthr = blockDim.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int TH = (nthr >> 5) * OY;
    const int tws = kConvTW + kx - 1;                 // even (kx odd)
    const int ths = TH + kyp - 1;                     // rows below TH + ky - 1 only ever meet zero taps: zero-filled
    T* tile = reinterpret_cast<T*>(smem_raw);
    T* Kc = reinterpret_cast<T*>(smem_raw + ((size_t)ths * tws * sizeof(T) + 15) / 16 * 16);
    const int i0 = blockIdx.x * kConvTW, j0 = blockIdx.y * TH;
    const int col0 = i0 - (kx - 1 - kx / 2), row0 = j0 - (ky - 1 - ky / 2);

    // fill with cp.async (LDGSTS): every thread queues all of its elements without waiting on any of them; elements
    // outside the image (and the padded rows below TH + ky - 1) are zero-filled by a source size of 0
    {
        const unsigned tile_s = (unsigned)__cvta_generic_to_shared(tile);
        for (int idx = tid; idx < ths * tws; idx += nthr) {
            const int r = idx / tws, c = idx - r * tws;
            const int gj = row0 + r, gi = col0 + c;
            const bool ok = r < TH + ky - 1 && gj >= 0 && gj < ny && gi >= 0 && gi < nx;
            const T* src = img + (ok ? (size_t)gj * nx + gi : 0);
            const unsigned dst = tile_s + (unsigned)idx * (unsigned)sizeof(T);
            const int nbytes = ok ? (int)sizeof(T) : 0;
            if constexpr (sizeof(T) == 4)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(nbytes) : "memory");
            else
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(nbytes) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }

    ConvAcc<T, OY> acc;
    acc.zero();
    const T* tp0 = tile + (size_t)(warp * OY) * tws + 2 * lane;
    const int npairs = (kx + 1) / 2;
    for (int m0 = 0; m0 < npairs; m0 += band_pairs) {
        const int mb = min(band_pairs, npairs - m0);
        if (m0 > 0) __syncthreads();                  // every warp is done with the previous band's taps
        stage_taps<T>(Kc, K, ky, kx, kyp, m0, mb, tid, nthr);
        if (m0 == 0) asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                              // taps (and, first time, the tile) are in place
        acc.template sweep<true>(tp0 + 2 * m0, tws, Kc, kyp, mb);
    }

    const int i = i0 + 2 * lane;
#pragma unroll
    for (int r = 0; r < OY; ++r) {
        const int j = j0 + warp * OY + r;
        if (j < ny) {
            if (i < nx) out[(size_t)j * nx + i] = acc.col0(r);
            if (i + 1 < nx) out[(size_t)j * nx + i + 1] = acc.col1(r);
        }
    }
}

struct ConvCfg { int OY, NW, kyp, band_pairs; size_t smem; };

// Equal-work CTAs run in waves of 148: cost = waves x rows per CTA (x 1.1 for OY = 4: twice the shared loads per FMA).
static bool pick_cfg(jt_dtype d, int ny, int nx, int ky, int kx, ConvCfg* best) {
    const size_t sz = dtype_size(d);
    const int npairs = (kx + 1) / 2;
    double best_cost = -1.0;
    for (int OY = (d == JT_F64 ? 4 : 8); OY >= 4; OY -= 4) {
        const int kyp = (ky + OY - 1) / OY * OY;
        for (int NW = 8; NW >= 4; --NW) {
            const int TH = NW * OY;
            const size_t tile = align_up((size_t)(TH + kyp - 1) * (kConvTW + kx - 1) * sz, 16);
            if (tile + (size_t)4 * kyp * sz > kMaxSmem) continue;
            // taps: whole kernel if it fits (and stays under 48 KB so that small kernels leave room for several CTAs)
            int bp = npairs;
            const size_t tap_budget = kMaxSmem - tile < 48 * 1024 ? kMaxSmem - tile : 48 * 1024;
            while (bp > 1 && (size_t)4 * bp * kyp * sz > tap_budget) --bp;
            const int64_t tiles = (int64_t)((nx + kConvTW - 1) / kConvTW) * ((ny + TH - 1) / TH);
            const int64_t waves = (tiles + kNumSMs - 1) / kNumSMs;
            const int n_bands = (npairs + bp - 1) / bp;
            const double cost = (double)waves * TH * (OY == 8 ? 1.0 : 1.1) * (1.0 + 0.01 * (n_bands - 1));
            if (best_cost < 0.0 || cost < best_cost) {
                best_cost = cost;
                *best = {OY, NW, kyp, bp, tile + (size_t)4 * bp * kyp * sz};
            }
        }
    }
    return best_cost >= 0.0;
}

bool conv_direct_supported(jt_dtype d, int ny, int nx, int ky, int kx) {
    ConvCfg c;
    return pick_cfg(d, ny, nx, ky, kx, &c);
}

size_t conv_direct_workspace_bytes(jt_dtype, int, int) { return 0; }

// Time model behind JT_CONV_AUTO, calibrated on B200 with `bench.py --conv-sweep`: a warp spends
// 4 OY (float, FFMA2) or 8 OY (double, DFMA) pipe cycles per kernel-column pair and kernel row, the warps of a
// scheduler share the pipe, the measured pipe efficiency is one half, and CTAs run in waves of 148.
double conv_direct_estimate_us(jt_dtype d, int ny, int nx, int ky, int kx) {
    ConvCfg c;
    if (!pick_cfg(d, ny, nx, ky, kx, &c)) return 1e30;
    const int64_t tiles = (int64_t)((nx + kConvTW - 1) / kConvTW) * ((ny + c.NW * c.OY - 1) / (c.NW * c.OY));
    const double waves = (double)((tiles + kNumSMs - 1) / kNumSMs);
    const double per_warp = (double)((kx + 1) / 2) * c.kyp * (d == JT_F32 ? 4.0 : 8.0) * c.OY;
    const double share = c.NW > 4 ? c.NW / 4.0 : 1.0;
    return 3.0 + waves * per_warp * share / 0.5 / 1.9e3;
}

template <typename T, int OY>
static jt_status run_cfg(const ConvCfg& c, int ny, int nx, const T* img, int ky, int kx, const T* ker, T* out, cudaStream_t st) {
    auto kern = k_conv_direct<T, OY>;
    JT_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem));
    dim3 grid((nx + kConvTW - 1) / kConvTW, (ny + c.NW * OY - 1) / (c.NW * OY));
    kern<<<grid, c.NW * 32, c.smem, st>>>(ny, nx, img, ky, kx, c.kyp, c.band_pairs, ker, out);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

template <typename T>
static jt_status conv_direct_t(jt_dtype d, int ny, int nx, const T* img, int ky, int kx, const T* ker, T* out, cudaStream_t st) {
    ConvCfg c;
    if (!pick_cfg(d, ny, nx, ky, kx, &c)) return JT_ERR_UNSUPPORTED;
    if constexpr (sizeof(T) == 4) {
        if (c.OY == 8) return run_cfg<T, 8>(c, ny, nx, img, ky, kx, ker, out, st);
    }
    return run_cfg<T, 4>(c, ny, nx, img, ky, kx, ker, out, st);
}

jt_status launch_conv_direct(jt_dtype dtype, int ny, int nx, const void* img, int ky, int kx, const void* ker,
                             void* workspace, void* out, cudaStream_t st) {
    (void)workspace;
    return dtype == JT_F32 ? conv_direct_t<float>(dtype, ny, nx, (const float*)img, ky, kx, (const float*)ker, (float*)out, st)
                           : conv_direct_t<double>(dtype, ny, nx, (const double*)img, ky, kx, (const double*)ker, (double*)out, st);
}

}  // namespace jt
