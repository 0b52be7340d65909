// jt_conv.cuh -- the register-blocked sweep shared by the direct convolution kernel (jt_conv.cu) and the in-CTA
// convolution of the batch kernel (jt_batch.cu).  Definition P (true convolution, zero padding).
//
// A thread owns OY x 2 outputs: OY vertically adjacent rows of two adjacent columns (2 lane, 2 lane + 1).  It walks
// the tile in column PAIRS (one 64-bit / 128-bit shared load fetches both columns of a row) and, per pair, slides a
// register window of OY rows down the tile.  Every loaded pair feeds 4 OY FMAs:
//   out col 0 += Kf[a][2m]   v.x + Kf[a][2m+1] v.y          out col 1 += Kf[a][2m-1] v.x + Kf[a][2m] v.y
// Taps come from shared memory as warp-uniform (broadcast) 128-bit loads of packed entries (see stage_taps).
#pragma once
#include "jt_internal.h"

namespace jt {

// Packed taps in shared memory: entry (m, a) of `Kq` (m = kernel-column pair, a = flipped-kernel row, kyp rows per
// pair, zero padded) holds the four taps one loaded tile pair (v.x, v.y) needs:
//   { Kf[a][2m], Kf[a][2m-1], Kf[a][2m+1], Kf[a][2m] }   = { col0 x v.x, col1 x v.x, col0 x v.y, col1 x v.y }
// with Kf[a][-1] = Kf[a][kx] = 0.  One 128-bit broadcast load (two for double) fetches an entry.
// Stages pairs [m_first, m_first + npairs) into Kq[0 .. npairs * kyp).
template <typename T>
__device__ __forceinline__ void stage_taps(T* __restrict__ Kq, const T* __restrict__ K, int ky, int kx, int kyp, int m_first,
                                           int npairs, int tid, int nthr) {
    for (int i = tid; i < npairs * kyp; i += nthr) {
        const int m = m_first + i / kyp, a = i % kyp;
        T t[3];                                                       // Kf[a][2m-1], Kf[a][2m], Kf[a][2m+1]
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int b = 2 * m - 1 + d;
            t[d] = (b >= 0 && b < kx && a < ky) ? K[(size_t)(ky - 1 - a) * kx + (kx - 1 - b)] : (T)0;
        }
        T* q = Kq + (size_t)i * 4;
        q[0] = t[1]; q[1] = t[0]; q[2] = t[2]; q[3] = t[1];
    }
}

// acc[r] (two adjacent output columns of row r) += sum over pairs m in [0, npairs) and taps a in [0, kyp).
// tp0: this thread's pair (row 0 of its strip, pair 0 of the band) in the tile; tws: tile row pitch in elements
// (even); Kq: packed taps of the band.  The tile must hold finite values (zeros) down to row kyp + OY - 2 of the strip.
// Per-dtype pieces of the sweep: window element (one tile pair), packed tap entry, accumulator of one output row.
template <typename T> struct ConvOps;

template <> struct ConvOps<double> {              // plain DFMA, 4 per row and loaded pair
    using Win = double2;
    struct Tap { double2 a, b; };
    struct Acc { double c0, c1; };
    static __device__ __forceinline__ Acc zero() { return {0.0, 0.0}; }
    static __device__ __forceinline__ Tap load_tap(const double* p) {
        return {*reinterpret_cast<const double2*>(p), *reinterpret_cast<const double2*>(p + 2)};
    }
    static __device__ __forceinline__ void fma_x(Acc& v, const Tap& t, const Win& w) { v.c0 = fma(t.a.x, w.x, v.c0); v.c1 = fma(t.a.y, w.x, v.c1); }
    static __device__ __forceinline__ void fma_y(Acc& v, const Tap& t, const Win& w) { v.c0 = fma(t.b.x, w.y, v.c0); v.c1 = fma(t.b.y, w.y, v.c1); }
    static __device__ __forceinline__ double col0(const Acc& v) { return v.c0; }
    static __device__ __forceinline__ double col1(const Acc& v) { return v.c1; }
};

// float: sm_100 packed FMA (fma.rn.f32x2 -> SASS FFMA2 with a broadcast .F32 operand): the two output columns of a
// row share one 64-bit accumulator, a tap pair comes packed from shared memory and the tile value is broadcast to
// both halves, so one issue slot does two FMAs -- the FP32 pipe, not the issue port, is then the limit
// (measured with jt_probe_alu: FFMA 122, FFMA2 63.5 instr-lanes/clk/SM).
template <> struct ConvOps<float> {
    using Win = float2;
    using Tap = ulonglong2;
    using Acc = unsigned long long;
    static __device__ __forceinline__ Acc zero() { return 0ull; }
    static __device__ __forceinline__ Tap load_tap(const float* p) { return *reinterpret_cast<const ulonglong2*>(p); }
    static __device__ __forceinline__ unsigned long long bcast(float x) {
        unsigned long long d;
        asm("mov.b64 %0, {%1, %1};" : "=l"(d) : "f"(x));
        return d;
    }
    static __device__ __forceinline__ void fma_x(Acc& v, const Tap& t, const Win& w) {
        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(v) : "l"(t.x), "l"(bcast(w.x)));
    }
    static __device__ __forceinline__ void fma_y(Acc& v, const Tap& t, const Win& w) {
        asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(v) : "l"(t.y), "l"(bcast(w.y)));
    }
    static __device__ __forceinline__ float col0(const Acc& v) { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
    static __device__ __forceinline__ float col1(const Acc& v) { return __uint_as_float((unsigned)(v >> 32)); }
};

// acc row r (two adjacent output columns) += sum over pairs m in [0, npairs) and taps a in [0, kyp).
// tp0: this thread's pair (row 0 of its strip, pair 0 of the band) in the tile; tws: tile row pitch in elements
// (even); Kq: packed taps of the band.  The tile must hold finite values (zeros) down to row kyp + OY - 2 of the
// strip.  The taps and tile rows of the NEXT chunk of OY kernel rows are loaded into a second register set before
// the current chunk's FMAs issue (software pipelining: with one or two resident warps per scheduler the shared-
// memory latency is otherwise exposed).
template <typename T, int OY>
struct ConvAcc {
    using O = ConvOps<T>;
    typename O::Acc v[OY];
    __device__ __forceinline__ void zero() {
#pragma unroll
        for (int r = 0; r < OY; ++r) v[r] = O::zero();
    }
    __device__ __forceinline__ T col0(int r) const { return O::col0(v[r]); }
    __device__ __forceinline__ T col1(int r) const { return O::col1(v[r]); }

    static __device__ __forceinline__ void load_chunk(typename O::Tap (&t)[OY], typename O::Win (&w)[OY], const T* kp,
                                                      const T* wp, int tws) {
#pragma unroll
        for (int aa = 0; aa < OY; ++aa) {
            t[aa] = O::load_tap(kp + 4 * aa);
            w[aa] = *reinterpret_cast<const typename O::Win*>(wp + (size_t)aa * tws);
        }
    }
    __device__ __forceinline__ void chunk(const typename O::Tap (&t)[OY], const typename O::Win (&w)[OY],
                                          typename O::Win (&win)[OY]) {
#pragma unroll
        for (int aa = 0; aa < OY; ++aa) {
            win[(aa + OY - 1) % OY] = w[aa];
#pragma unroll
            for (int r = 0; r < OY; ++r) O::fma_x(v[r], t[aa], win[(aa + r) % OY]);
#pragma unroll
            for (int r = 0; r < OY; ++r) O::fma_y(v[r], t[aa], win[(aa + r) % OY]);
        }
    }
    // PIPE = false: loads issue in program order, one kernel row at a time (enough when >= 4 warps per scheduler are
    // resident, as in the batch kernel, and much lighter on registers).
    template <bool PIPE = true>
    __device__ __forceinline__ void sweep(const T* __restrict__ tp0, int tws, const T* __restrict__ Kq, int kyp, int npairs) {
#pragma unroll 1
        for (int m = 0; m < npairs; ++m) {
            const T* wp = tp0 + 2 * m;
            const T* kp = Kq + (size_t)m * kyp * 4;
            typename O::Win win[OY];
#pragma unroll
            for (int r = 0; r < OY - 1; ++r) { win[r] = *reinterpret_cast<const typename O::Win*>(wp); wp += tws; }
            if constexpr (!PIPE) {
#pragma unroll 1
                for (int a0 = 0; a0 < kyp; a0 += OY) {
#pragma unroll
                    for (int aa = 0; aa < OY; ++aa) {
                        const typename O::Tap t = O::load_tap(kp + 4 * aa);
                        win[(aa + OY - 1) % OY] = *reinterpret_cast<const typename O::Win*>(wp);
                        wp += tws;
#pragma unroll
                        for (int r = 0; r < OY; ++r) O::fma_x(v[r], t, win[(aa + r) % OY]);
#pragma unroll
                        for (int r = 0; r < OY; ++r) O::fma_y(v[r], t, win[(aa + r) % OY]);
                    }
                    kp += 4 * OY;
                }
                continue;
            }
            typename O::Tap tA[OY], tB[OY];
            typename O::Win wA[OY], wB[OY];
            load_chunk(tA, wA, kp, wp, tws);
            int a0 = 0;
#pragma unroll 1
            for (; a0 + 2 * OY <= kyp; a0 += 2 * OY) {
                load_chunk(tB, wB, kp + 4 * OY, wp + (size_t)OY * tws, tws);
                chunk(tA, wA, win);
                const bool more = a0 + 2 * OY < kyp;                 // else reload a valid chunk and ignore it
                load_chunk(tA, wA, more ? kp + 8 * OY : kp, more ? wp + (size_t)2 * OY * tws : wp, tws);
                chunk(tB, wB, win);
                kp += 8 * OY;
                wp += (size_t)2 * OY * tws;
            }
            if (a0 < kyp) chunk(tA, wA, win);
        }
    }
};

}  // namespace jt
