// jt_conv.cu -- step 5a: direct PSF convolution (definition P; PAPER.md:55 third step).
//
// out[j][i] = sum_a sum_b Kf[a][b] tile[jl+a][il+b],  Kf = kernel flipped in both axes (true convolution),
// tile = image window with a (ky-1, kx-1) halo staged in shared memory, zero outside the image.
// Each thread owns OY vertically adjacent outputs of one column: for a kernel column b it slides a
// register window of OY tile values down the column, so one shared-memory load (lanes on consecutive
// addresses: conflict-free) feeds OY FMAs; kernel taps are warp-uniform vector loads from a flipped,
// column-major copy (Kc[b][a], built by k_flip_kernel in the workspace).  FMA : LDS = OY : 1.25.
#include "jt_conv.cuh"

namespace jt {

template <typename T>
__global__ void k_flip_kernel(int ky, int kx, int kyp, const T* __restrict__ K, T* __restrict__ Kc) {
    const int n = kx * kyp;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int b = i / kyp, a = i % kyp;
        Kc[i] = (a < ky) ? K[(size_t)(ky - 1 - a) * kx + (kx - 1 - b)] : (T)0;
    }
}

template <typename T, int OY, int TW, int NTR>
__global__ void __launch_bounds__(TW* NTR) k_conv_direct(int ny, int nx, const T* __restrict__ img, int ky, int kx,
                                                         int kyp, const T* __restrict__ Kc, T* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* tile = reinterpret_cast<T*>(smem_raw);
    constexpr int TH = NTR * OY;
    const int tws = TW + kx - 1, ths = TH + ky - 1;
    const int i0 = blockIdx.x * TW, j0 = blockIdx.y * TH;
    const int col0 = i0 - (kx - 1 - kx / 2), row0 = j0 - (ky - 1 - ky / 2);
    const int tid = threadIdx.x;

    for (int idx = tid; idx < ths * tws; idx += TW * NTR) {
        const int r = idx / tws, c = idx - r * tws;
        const int gj = row0 + r, gi = col0 + c;
        tile[idx] = (gj >= 0 && gj < ny && gi >= 0 && gi < nx) ? __ldg(&img[(size_t)gj * nx + gi]) : (T)0;
    }
    __syncthreads();

    const int il = tid % TW, jl0 = (tid / TW) * OY;
    T acc[OY];
#pragma unroll
    for (int r = 0; r < OY; ++r) acc[r] = (T)0;
    conv_sweep<T, OY, true>(tile + jl0 * tws + il, tws, Kc, ky, kx, kyp, acc);

    const int i = i0 + il;
    if (i < nx) {
#pragma unroll
        for (int r = 0; r < OY; ++r) {
            const int j = j0 + jl0 + r;
            if (j < ny) out[(size_t)j * nx + i] = acc[r];
        }
    }
}

constexpr size_t kMaxSmem = 227 * 1024;

struct ConvCfg { int OY, TW, NTR; size_t smem; };

static bool pick_cfg(jt_dtype d, int ny, int nx, int ky, int kx, ConvCfg* c) {
    const size_t sz = dtype_size(d);
    // wide tile first (better FMA:LDS), narrow tile when the halo would not fit
    const ConvCfg cands[2] = {{8, 64, 4, 0}, {4, 32, 8, 0}};
    for (int k = 0; k < 2; ++k) {
        ConvCfg x = cands[k];
        if (k == 0 && nx <= 32) continue;
        x.smem = (size_t)(x.NTR * x.OY + ky - 1) * (size_t)(x.TW + kx - 1) * sz;
        if (x.smem <= kMaxSmem) { *c = x; return true; }
    }
    (void)ny;
    return false;
}

bool conv_direct_supported(jt_dtype d, int ny, int nx, int ky, int kx) {
    ConvCfg c;
    return pick_cfg(d, ny, nx, ky, kx, &c);
}

size_t conv_direct_workspace_bytes(jt_dtype d, int ky, int kx) {
    const int kyp = (ky + 7) / 8 * 8;
    return align_up((size_t)kx * kyp * dtype_size(d), 256);
}

template <typename T, int OY, int TW, int NTR>
static jt_status run_cfg(int ny, int nx, const T* img, int ky, int kx, int kyp, const T* Kc, T* out, size_t smem,
                         cudaStream_t st) {
    auto kern = k_conv_direct<T, OY, TW, NTR>;
    JT_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid((nx + TW - 1) / TW, (ny + NTR * OY - 1) / (NTR * OY));
    kern<<<grid, TW * NTR, smem, st>>>(ny, nx, img, ky, kx, kyp, Kc, out);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

template <typename T>
static jt_status conv_direct_t(jt_dtype d, int ny, int nx, const T* img, int ky, int kx, const T* ker, void* workspace,
                               T* out, cudaStream_t st) {
    ConvCfg c;
    if (!pick_cfg(d, ny, nx, ky, kx, &c)) return JT_ERR_UNSUPPORTED;
    const int kyp = (ky + 7) / 8 * 8;
    T* Kc = (T*)workspace;
    const int n = kx * kyp;
    k_flip_kernel<T><<<(n + 255) / 256, 256, 0, st>>>(ky, kx, kyp, ker, Kc);
    JT_LAUNCH_CHECK();
    if (c.OY == 8) return run_cfg<T, 8, 64, 4>(ny, nx, img, ky, kx, kyp, Kc, out, c.smem, st);
    return run_cfg<T, 4, 32, 8>(ny, nx, img, ky, kx, kyp, Kc, out, c.smem, st);
}

jt_status launch_conv_direct(jt_dtype dtype, int ny, int nx, const void* img, int ky, int kx, const void* ker,
                             void* workspace, void* out, cudaStream_t st) {
    return dtype == JT_F32
               ? conv_direct_t<float>(dtype, ny, nx, (const float*)img, ky, kx, (const float*)ker, workspace, (float*)out, st)
               : conv_direct_t<double>(dtype, ny, nx, (const double*)img, ky, kx, (const double*)ker, workspace, (double*)out, st);
}

}  // namespace jt
