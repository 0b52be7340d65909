// jt_internal.h -- host-side plumbing shared by the translation units of libjt (not installed).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <stddef.h>
#include <stdint.h>
#include "../../include/jt.h"
#include "jt_device.cuh"

namespace jt {

constexpr int kNumSMs = 148;            // B200
constexpr int kBatchThreads = 256;      // 8 warps per CTA in the batch kernel

// thread-local last CUDA error (jt_last_cuda_error)
void set_last_cuda_error(int e);
void count_launch();
#define JT_CUDA_TRY(expr)                                                    \
    do {                                                                     \
        cudaError_t _e = (expr);                                             \
        if (_e != cudaSuccess) { jt::set_last_cuda_error((int)_e); return JT_ERR_CUDA; } \
    } while (0)
#define JT_LAUNCH_CHECK()                                                    \
    do {                                                                     \
        jt::count_launch();                                                  \
        cudaError_t _e = cudaGetLastError();                                 \
        if (_e != cudaSuccess) { jt::set_last_cuda_error((int)_e); return JT_ERR_CUDA; } \
    } while (0)

// "Done once" for set-up that belongs to a DEVICE (cudaFuncSetAttribute acts on the device that is current): one bit per
// device ordinal, safe against host threads racing (both then do the idempotent set-up).  Devices beyond bit 63 and a
// failing cudaGetDevice simply repeat the set-up on every call.
struct PerDeviceOnce {
    std::atomic<uint64_t> done{0};
    bool needed() {
        int d = -1;
        if (cudaGetDevice(&d) != cudaSuccess || d < 0 || d >= 64) return true;
        return (done.load(std::memory_order_acquire) >> d & 1ull) == 0;
    }
    void mark() {
        int d = -1;
        if (cudaGetDevice(&d) == cudaSuccess && d >= 0 && d < 64) done.fetch_or(1ull << d, std::memory_order_release);
    }
};

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
inline size_t dtype_size(jt_dtype d) { return d == JT_F32 ? 4 : 8; }

// ---- host-side derived parameters (definition E and the constants of S, R) ----
MacroLens make_macro(const jt_lens* lens);
jt_status make_sources(const jt_sources* src, SrcSet* out);

// ---- ray tracing (jt_trace.cu) ----
struct TracePlan {
    int R;                 // rays per thread
    int threads;           // threads per CTA
    int cols_per_warp;     // active lanes per warp (grid mode: floor(32/s)*s; ray mode: 32)
    int tiles_x, tiles_y;  // grid mode: warp tiles (cols_per_warp x R rays) per axis
    int64_t n_wt;          // grid mode: warp tiles in all
    bool wide;             // grid mode, single-image kernel: CTA-wide tiles (s does not divide 32)
    int cols_per_cta, ctiles_x;
    int64_t n_tiles_wide;
    int64_t n_tiles;       // CTAs per subhalo chunk (threads/32 warp tiles, or threads * R rays in ray mode)
    int n_chunks;          // subhalo list split (1 = no workspace traffic)
    int64_t chunk_len;     // subhalos per chunk
    size_t partial_bytes;  // n_chunks > 1: double2 per (chunk, ray slot)
    size_t counter_bytes;  // one uint32 per tile
    size_t tier_bytes;     // four uint64 tier counters (jt_profile_tiers), always reserved
    size_t rec_bytes;      // derived subhalo records, written by k_make_recs at the start of every call
    size_t total_bytes;
};
TracePlan plan_trace_grid(jt_dtype dtype, const jt_grid* g, int64_t n_tnfw);
TracePlan plan_trace_rays(jt_dtype dtype, int64_t n_rays, int64_t n_tnfw);

int       trace_tile_recs(jt_dtype dtype, const TracePlan& plan);
jt_status launch_trace_grid(jt_dtype dtype, const jt_grid* g, const jt_lens* lens, const SrcSet& src,
                            const TracePlan& plan, void* workspace, void* pre_psf, bool count_tiers, cudaStream_t st);
void*     trace_tier_counters(const TracePlan& plan, void* workspace);
jt_status launch_trace_rays(jt_dtype dtype, int64_t n, const void* tx, const void* ty, const jt_lens* lens,
                            const TracePlan& plan, void* workspace, void* bx, void* by, cudaStream_t st);
jt_status launch_source_brightness(jt_dtype dtype, int64_t n, const void* bx, const void* by, const SrcSet& src,
                                   void* flux, cudaStream_t st);

// ---- convolution (jt_conv.cu, jt_fft.cu) ----
jt_conv_method resolve_conv_method(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx, jt_conv_method m);
bool      conv_direct_supported(jt_dtype dtype, int ny, int nx, int ky, int kx);
size_t    conv_direct_workspace_bytes(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx);
double    conv_direct_estimate_us(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx);
double    conv_fft_estimate_us(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx);
jt_status launch_conv_direct(jt_dtype dtype, int64_t B, int ny, int nx, const void* img, int ky, int kx, const void* ker,
                             void* workspace, void* out, cudaStream_t st);   // B images [B][ny][nx], one kernel
void      conv_direct_describe(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx, const void* img, jt_conv_plan* out);
void      conv_fft_describe(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx, jt_conv_plan* out);
bool      conv_fft_supported(jt_dtype dtype, int ny, int nx, int ky, int kx);
size_t    fft_conv_workspace_bytes(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx);
jt_status launch_conv_fft(jt_dtype dtype, int64_t B, int ny, int nx, const void* img, int ky, int kx, const void* ker,
                          void* workspace, void* out, cudaStream_t st);   // B images [B][ny][nx], one kernel

// ---- batch (jt_batch.cu); data / sigma / chi2 non-null: chi^2 accumulated in the kernel, out may then be null ----
jt_status launch_batch(jt_dtype dtype, int64_t B, const jt_grid* g, const jt_batch_params* p, void* out,
                       const void* data, const void* sigma, double* chi2, cudaStream_t st);

// ---- SURVEY 8(f) rows (jt_next.cu) ----
jt_status launch_chi2(jt_dtype dtype, int64_t B, int64_t n_pix, const void* models, const void* data, const void* sigma,
                      double* chi2, cudaStream_t st);
jt_status launch_lensing_maps(jt_dtype dtype, int64_t n, const void* tx, const void* ty, const jt_lens* lens, void* kappa,
                              void* gamma1, void* gamma2, void* mu, cudaStream_t st);
jt_status launch_ray_shoot_profiles(jt_dtype dtype, int64_t n, const void* tx, const void* ty, int64_t n_def,
                                    const jt_profile* defs, void* bx, void* by, cudaStream_t st);
jt_status launch_light_profiles(jt_dtype dtype, int64_t n, const void* bx, const void* by, int64_t n_comp,
                                const jt_profile* comps, void* flux, cudaStream_t st);

jt_status launch_core_sersic(jt_dtype dtype, int64_t n, const void* bx, const void* by, const double* params10, void* flux,
                             cudaStream_t st);
jt_status launch_shapelets(jt_dtype dtype, int64_t n, const void* bx, const void* by, int n_max, double beta, double cx, double cy,
                           const void* coef, void* flux, cudaStream_t st);
jt_status launch_bin_sum(jt_dtype dtype, int ny, int nx, int s, const void* fine, void* out, cudaStream_t st);

}  // namespace jt
