// jt_probe.cu -- ALU peak microbenchmarks ("all to be re-measured by microbenchmark in the
// same run").  MEASURED_PEAKS.json holds only HBM and bf16 tensor numbers; the ray-tracing kernels are bound by the
// FP32 issue port / FP64 pipe / MUFU, so bench.py measures those rates with these kernels and reports them beside
// the derived peaks.  Each thread runs 8 independent dependency chains of one instruction kind; a launch executes
// blocks * 256 * iters * 8 * 4 instructions of that kind per thread-lane (4 = inner unroll).
#include "jt_internal.h"

namespace jt {

constexpr int kProbeChains = 8;
constexpr int kProbeUnroll = 4;

template <int KIND>
__global__ void __launch_bounds__(256) k_probe(int64_t iters, float seed, float* __restrict__ sink) {
    const float a0 = seed + (float)threadIdx.x * 1e-7f;
    if constexpr (KIND == JT_PROBE_FFMA) {
        float v[kProbeChains];
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) v[c] = a0 + (float)c;
        const float m = 0.999f + seed * 1e-9f, b = 1e-3f * seed;
        for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
                for (int c = 0; c < kProbeChains; ++c) v[c] = fmaf(v[c], m, b);
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) s += v[c];
        if (s == 123.456f) sink[0] = s;
    } else if constexpr (KIND == JT_PROBE_FFMA2) {
        unsigned long long v[kProbeChains];
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) {
            const float lo = a0 + (float)c, hi = a0 - (float)c;
            v[c] = ((unsigned long long)__float_as_uint(hi) << 32) | __float_as_uint(lo);
        }
        const float mf = 0.999f + seed * 1e-9f, bf = 1e-3f * seed;
        const unsigned long long m = ((unsigned long long)__float_as_uint(mf) << 32) | __float_as_uint(mf);
        const unsigned long long b = ((unsigned long long)__float_as_uint(bf) << 32) | __float_as_uint(bf);
        for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
                for (int c = 0; c < kProbeChains; ++c)
                    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(v[c]) : "l"(v[c]), "l"(m), "l"(b));
        }
        unsigned long long s = 0;
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) s ^= v[c];
        if (s == 0x123456789abcdefull) sink[0] = 1.f;
    } else if constexpr (KIND == JT_PROBE_DFMA) {
        double v[kProbeChains];
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) v[c] = (double)a0 + (double)c;
        const double m = 0.999 + (double)seed * 1e-9, b = 1e-3 * (double)seed;
        for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
                for (int c = 0; c < kProbeChains; ++c) v[c] = fma(v[c], m, b);
        }
        double s = 0.0;
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) s += v[c];
        if (s == 123.456) sink[0] = (float)s;
    } else if constexpr (KIND == JT_PROBE_FFMA2_RF) {
        // the direct convolution's operand pattern: 8 accumulators x 4 packed taps x 8 broadcast tile values, all in
        // distinct registers (5 register reads per FFMA2, only the tap reusable)
        unsigned long long acc[8], t[4];
        float w[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) { acc[c] = 0ull; w[c] = a0 * (float)(c + 1); }
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const float x = 1e-3f * (float)(c + 1) * seed;
            t[c] = ((unsigned long long)__float_as_uint(x) << 32) | __float_as_uint(-x);
        }
        for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
                for (int c = 0; c < kProbeChains; ++c) {
                    unsigned long long wb;
                    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(wb) : "f"(w[(c + u) % 8]));
                    asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[c]) : "l"(t[u]), "l"(wb));
                }
        }
        unsigned long long s = 0;
#pragma unroll
        for (int c = 0; c < 8; ++c) s ^= acc[c];
        if (s == 0x123456789abcdefull) sink[0] = 1.f;
    } else if constexpr (KIND == JT_PROBE_DFMA_RF) {
        // DFMA with the direct convolution's operand pattern: 8 accumulators, 4 taps, 8 tile values, all distinct doubles
        double acc[8], t[4], w[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) { acc[c] = 0.0; w[c] = (double)a0 * (double)(c + 1); }
#pragma unroll
        for (int c = 0; c < 4; ++c) t[c] = 1e-3 * (double)(c + 1) * (double)seed;
        for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
                for (int c = 0; c < kProbeChains; ++c)
                    asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(acc[c]) : "d"(t[u]), "d"(w[(c + u) % 8]));
        }
        double s = 0.0;
#pragma unroll
        for (int c = 0; c < 8; ++c) s += acc[c];
        if (s == 123.456) sink[0] = (float)s;
    } else if constexpr (KIND == JT_PROBE_FFMA2_LDS) {
        // the direct convolution's inner loop with its shared-memory traffic: per kernel row one broadcast 128-bit tap
        // load and one 64-bit window load feed 16 FFMA2 (8 accumulators x two products), window rotating in registers
        __shared__ __align__(16) float smem[8 * 16 * 4 + 72 * 64];
        for (int i = threadIdx.x; i < 8 * 16 * 4 + 72 * 64; i += 256) smem[i] = 1e-3f * (float)(i % 17) * seed;
        __syncthreads();
        const float* taps = smem;
        const float* tile = smem + 8 * 16 * 4 + 2 * (threadIdx.x & 31);
        unsigned long long acc[8];
        float2 win[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) { acc[c] = 0ull; win[c] = make_float2(a0, a0 * (float)c); }
        for (int64_t i = 0; i < iters; ++i) {
            const float* kp = taps + (i & 7) * 64;
            const float* wp = tile + (i & 7) * 8 * 64;
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u) {        // 4 kernel rows x 8 accumulators = 32 FFMA2 ... x2 products below
                const ulonglong2 t = *reinterpret_cast<const ulonglong2*>(kp + 4 * u);
                win[(u + 7) % 8] = *reinterpret_cast<const float2*>(wp + u * 64);
                if (u & 1) {                                 // count stays 8 per (u): alternate x and y products
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        unsigned long long wb;
                        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(wb) : "f"(win[(c + u) % 8].y));
                        asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[c]) : "l"(t.y), "l"(wb));
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        unsigned long long wb;
                        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(wb) : "f"(win[(c + u) % 8].x));
                        asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc[c]) : "l"(t.x), "l"(wb));
                    }
                }
            }
        }
        unsigned long long s2 = 0;
#pragma unroll
        for (int c = 0; c < 8; ++c) s2 ^= acc[c];
        if (s2 == 0x123456789abcdefull) sink[0] = 1.f;
    } else {   // JT_PROBE_MUFU_RSQ
        float v[kProbeChains];
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) v[c] = 1.5f + a0 + (float)c;
        for (int64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
                for (int c = 0; c < kProbeChains; ++c) asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(v[c]) : "f"(v[c]));
        }
        float s = 0.f;
#pragma unroll
        for (int c = 0; c < kProbeChains; ++c) s += v[c];
        if (s == 123.456f) sink[0] = s;
    }
}

}  // namespace jt

using namespace jt;

extern "C" jt_status jt_probe_alu(int32_t kind, int32_t blocks, int64_t iters, void* sink, int64_t* lane_ops, void* stream) {
    if (blocks < 1 || iters < 1 || !sink) return JT_ERR_INVALID_VALUE;
    cudaStream_t st = (cudaStream_t)stream;
    switch (kind) {
        case JT_PROBE_FFMA: k_probe<JT_PROBE_FFMA><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_FFMA2: k_probe<JT_PROBE_FFMA2><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_DFMA: k_probe<JT_PROBE_DFMA><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_FFMA2_RF: k_probe<JT_PROBE_FFMA2_RF><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_DFMA_RF: k_probe<JT_PROBE_DFMA_RF><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_FFMA2_LDS: k_probe<JT_PROBE_FFMA2_LDS><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_MUFU_RSQ: k_probe<JT_PROBE_MUFU_RSQ><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        default: return JT_ERR_UNSUPPORTED;
    }
    JT_LAUNCH_CHECK();
    if (lane_ops) *lane_ops = (int64_t)blocks * 256 * iters * kProbeChains * kProbeUnroll;
    return JT_OK;
}
