// jt_conv.cuh -- the register-window column sweep shared by the direct convolution kernel (jt_conv.cu) and
// the in-CTA convolution of the batch kernel (jt_batch.cu).  Definition P (true convolution, zero padding).
#pragma once
#include "jt_internal.h"

namespace jt {

template <typename T, int OY, bool LDG>
__device__ __forceinline__ void load_taps(const T* __restrict__ p, T (&kv)[OY]) {
    if constexpr (sizeof(T) == 4) {
#pragma unroll
        for (int i = 0; i < OY; i += 4) {
            float4 v;
            if constexpr (LDG) v = __ldg(reinterpret_cast<const float4*>(p + i));
            else v = *reinterpret_cast<const float4*>(p + i);
            kv[i] = v.x; kv[i + 1] = v.y; kv[i + 2] = v.z; kv[i + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int i = 0; i < OY; i += 2) {
            double2 v;
            if constexpr (LDG) v = __ldg(reinterpret_cast<const double2*>(p + i));
            else v = *reinterpret_cast<const double2*>(p + i);
            kv[i] = v.x; kv[i + 1] = v.y;
        }
    }
}

// acc[r] += sum_b sum_a Kc[b][a] * tcol0[(r + a) * tws + b],  r < OY, a < ky, b < kx.
// tcol0 = shared-memory tile at this thread's first output row and its column; Kc = flipped kernel, column-major,
// columns padded with zeros to kyp (a multiple of 8).  One shared load feeds OY FMAs.
template <typename T, int OY, bool LDG>
__device__ __forceinline__ void conv_sweep(const T* __restrict__ tcol0, int tws, const T* __restrict__ Kc, int ky, int kx,
                                           int kyp, T (&acc)[OY]) {
    for (int b = 0; b < kx; ++b) {
        const T* tcol = tcol0 + b;
        const T* kcol = Kc + (size_t)b * kyp;
        T win[OY];
#pragma unroll
        for (int r = 0; r < OY - 1; ++r) win[r] = tcol[r * tws];
        int a0 = 0;
        for (; a0 + OY <= ky; a0 += OY) {
            T kv[OY];
            load_taps<T, OY, LDG>(kcol + a0, kv);
#pragma unroll
            for (int aa = 0; aa < OY; ++aa) {
                win[(aa + OY - 1) % OY] = tcol[(a0 + aa + OY - 1) * tws];
#pragma unroll
                for (int r = 0; r < OY; ++r) acc[r] = fma(kv[aa], win[(aa + r) % OY], acc[r]);
            }
        }
        if (a0 < ky) {
            T kv[OY];
            load_taps<T, OY, LDG>(kcol + a0, kv);       // zero-padded up to kyp
#pragma unroll
            for (int aa = 0; aa < OY; ++aa) {
                if (a0 + aa < ky) {
                    win[(aa + OY - 1) % OY] = tcol[(a0 + aa + OY - 1) * tws];
#pragma unroll
                    for (int r = 0; r < OY; ++r) acc[r] = fma(kv[aa], win[(aa + r) % OY], acc[r]);
                }
            }
        }
    }
}

}  // namespace jt
