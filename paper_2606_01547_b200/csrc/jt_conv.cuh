// jt_conv.cuh -- the register-blocked sweep shared by the direct convolution kernel (jt_conv.cu) and the in-CTA
// convolution of the batch kernel (jt_batch.cu).  Definition P (true convolution, zero padding).
//
// A thread owns OY x 2 outputs: OY vertically adjacent rows of two adjacent columns (2 lane, 2 lane + 1).  It walks
// the tile in column PAIRS (one 64-bit / 128-bit shared load fetches both columns of a row) and, per pair, slides a
// register window of OY rows down the tile.  Every loaded pair feeds 4 OY FMAs:
//   out col 0 += Kf[a][2m]   v.x + Kf[a][2m+1] v.y          out col 1 += Kf[a][2m-1] v.x + Kf[a][2m] v.y
// Taps come from shared memory as warp-uniform (broadcast) vector loads of 4 taps of one flipped-kernel column.
#pragma once
#include "jt_internal.h"

namespace jt {

template <typename T> struct pair_of;
template <> struct pair_of<float> { using type = float2; };
template <> struct pair_of<double> { using type = double2; };
template <typename T> using Pair = typename pair_of<T>::type;

template <typename T>
__device__ __forceinline__ void load_taps4(const T* __restrict__ p, T (&k)[4]) {
    if constexpr (sizeof(T) == 4) {
        const float4 v = *reinterpret_cast<const float4*>(p);
        k[0] = v.x; k[1] = v.y; k[2] = v.z; k[3] = v.w;
    } else {
        const double2 u = *reinterpret_cast<const double2*>(p);
        const double2 v = *reinterpret_cast<const double2*>(p + 2);
        k[0] = u.x; k[1] = u.y; k[2] = v.x; k[3] = v.y;
    }
}

// Flipped kernel columns in shared memory: column c of `Kc` (c = b + 1, b = -1 ... last) holds Kf[.][b] padded with
// zeros to kyp rows (kyp a multiple of OY, OY a multiple of 4); columns b = -1 and b >= kx are zero.
// Fills columns for b in [b_first, b_first + ncols) into Kc[0 .. ncols).
template <typename T>
__device__ __forceinline__ void stage_taps(T* __restrict__ Kc, const T* __restrict__ K, int ky, int kx, int kyp, int b_first,
                                           int ncols, int tid, int nthr) {
    for (int i = tid; i < ncols * kyp; i += nthr) {
        const int c = i / kyp, a = i - c * kyp;
        const int b = b_first + c;
        Kc[i] = (b >= 0 && b < kx && a < ky) ? K[(size_t)(ky - 1 - a) * kx + (kx - 1 - b)] : (T)0;
    }
}

// acc[r][ox] += sum over pairs m in [0, npairs) and taps a in [0, kyp) -- tp0: this thread's pair (row 0 of its
// strip, pair 0 of the band) in the tile, tws: tile row pitch in elements (even); Kc: taps of column b = 2 m0 - 1
// of the band at index 0.  The tile must hold finite values (zeros) down to row kyp + OY - 2 of the strip.
template <typename T, int OY>
__device__ __forceinline__ void conv_sweep2(const T* __restrict__ tp0, int tws, const T* __restrict__ Kc, int kyp, int npairs,
                                            T (&acc)[OY][2]) {
    static_assert(OY % 4 == 0, "window unrolling loads taps four at a time");
#pragma unroll 1
    for (int m = 0; m < npairs; ++m) {
        const T* tp = tp0 + 2 * m;
        const T* k0 = Kc + (size_t)(2 * m) * kyp;          // column b = 2m - 1
        const T* k1 = k0 + kyp;                            //          2m
        const T* k2 = k1 + kyp;                            //          2m + 1
        Pair<T> win[OY];
#pragma unroll
        for (int r = 0; r < OY - 1; ++r) win[r] = *reinterpret_cast<const Pair<T>*>(tp + r * tws);
#pragma unroll 1
        for (int a0 = 0; a0 < kyp; a0 += OY) {
#pragma unroll
            for (int a4 = 0; a4 < OY; a4 += 4) {
                T t0[4], t1[4], t2[4];
                load_taps4<T>(k0 + a0 + a4, t0);
                load_taps4<T>(k1 + a0 + a4, t1);
                load_taps4<T>(k2 + a0 + a4, t2);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int aa = a4 + q;
                    win[(aa + OY - 1) % OY] = *reinterpret_cast<const Pair<T>*>(tp + (a0 + aa + OY - 1) * tws);
#pragma unroll
                    for (int r = 0; r < OY; ++r) {
                        const Pair<T> w = win[(aa + r) % OY];
                        acc[r][0] = fma(t1[q], w.x, acc[r][0]);
                        acc[r][0] = fma(t2[q], w.y, acc[r][0]);
                        acc[r][1] = fma(t0[q], w.x, acc[r][1]);
                        acc[r][1] = fma(t1[q], w.y, acc[r][1]);
                    }
                }
            }
        }
    }
}

}  // namespace jt
