// jt_probe.cu -- libjtprobe.so (include/jt_probe.h), separate from the product library: ALU peak microbenchmarks ("all to be re-measured by microbenchmark in the
// same run").  MEASURED_PEAKS.json holds only HBM and bf16 tensor numbers; the ray-tracing kernels are bound by the
// FP32 issue port / FP64 pipe / MUFU, so bench.py measures those rates with these kernels and reports them beside
// the derived peaks.  Each thread runs 8 independent dependency chains of one instruction kind; a launch executes
// blocks * 256 * iters * 8 * 4 instructions of that kind per thread-lane (4 = inner unroll).
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/jt_probe.h"

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

extern "C" int jt_probe_alu(int32_t kind, int32_t blocks, int64_t iters, void* sink, int64_t* lane_ops, void* stream) {
    if (blocks < 1 || iters < 1 || !sink) return 1;
    cudaStream_t st = (cudaStream_t)stream;
    switch (kind) {
        case JT_PROBE_FFMA: k_probe<JT_PROBE_FFMA><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_FFMA2: k_probe<JT_PROBE_FFMA2><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_DFMA: k_probe<JT_PROBE_DFMA><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        case JT_PROBE_MUFU_RSQ: k_probe<JT_PROBE_MUFU_RSQ><<<blocks, 256, 0, st>>>(iters, 1.0f, (float*)sink); break;
        default: return 2;
    }
    if (cudaGetLastError() != cudaSuccess) return 4;
    if (lane_ops) *lane_ops = (int64_t)blocks * 256 * iters * kProbeChains * kProbeUnroll;
    return 0;
}
