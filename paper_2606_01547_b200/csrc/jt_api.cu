// jt_api.cu -- the C ABI declared in include/jt.h: argument validation, workspace layout, launches.
#include <string.h>
#include "jt_internal.h"

namespace jt {

static thread_local int g_last_cuda_error = 0;
void set_last_cuda_error(int e) { g_last_cuda_error = e; }
static thread_local uint64_t g_launches = 0;
void count_launch() { ++g_launches; }

// ---- profiling events (jt_profile_enable / jt_profile_read) ----
struct ProfileState {
    bool on = false, recorded = false, had_conv = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};      // start, after trace, after conv, after the counter copy
    uint64_t* host_tiers = nullptr;    // pinned host copy of the last profiled call's JT_N_TIERS tier counters
    bool have_tiers = false;
};
static thread_local ProfileState g_prof;

static jt_status check_device() {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { set_last_cuda_error((int)e); return JT_ERR_CUDA; }
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) { set_last_cuda_error((int)e); return JT_ERR_CUDA; }
    return major == 10 ? JT_OK : JT_ERR_UNSUPPORTED;
}

static bool valid_dtype(jt_dtype d) { return d == JT_F32 || d == JT_F64; }
static bool valid_method(jt_conv_method m) { return m == JT_CONV_AUTO || m == JT_CONV_DIRECT || m == JT_CONV_FFT; }
static bool valid_grid(const jt_grid* g) {
    return g && g->nx >= 1 && g->ny >= 1 && g->pixel_scale > 0.0 && g->supersample >= 1 &&
           g->supersample <= JT_MAX_SUPERSAMPLE && (int64_t)g->nx * g->supersample < (1 << 30) &&
           (int64_t)g->ny * g->supersample < (1 << 30);
}
static bool valid_lens(const jt_lens* l) {
    if (!l || l->n_tnfw < 0) return false;
    if (l->n_tnfw > 0 && (!l->tnfw_cx || !l->tnfw_cy || !l->tnfw_Rs || !l->tnfw_alpha_Rs || !l->tnfw_r_trunc)) return false;
    return true;
}
static bool valid_kernel_size(int ky, int kx) { return ky >= 1 && kx >= 1 && (ky & 1) && (kx & 1); }

// AUTO: whichever of the two supported paths the calibrated time models expect to be faster.
jt_conv_method resolve_conv_method(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx, jt_conv_method m) {
    if (m == JT_CONV_DIRECT || m == JT_CONV_FFT) return m;
    if (!conv_direct_supported(dtype, ny, nx, ky, kx)) return JT_CONV_FFT;
    if (!conv_fft_supported(dtype, ny, nx, ky, kx)) return JT_CONV_DIRECT;
    return conv_fft_estimate_us(dtype, B, ny, nx, ky, kx) < conv_direct_estimate_us(dtype, B, ny, nx, ky, kx) ? JT_CONV_FFT
                                                                                                                     : JT_CONV_DIRECT;
}

static size_t conv_ws(jt_dtype dtype, int64_t B, int ny, int nx, int ky, int kx, jt_conv_method method) {
    const jt_conv_method m = resolve_conv_method(dtype, B, ny, nx, ky, kx, method);
    return m == JT_CONV_DIRECT ? conv_direct_workspace_bytes(dtype, B, ny, nx, ky, kx) : fft_conv_workspace_bytes(dtype, B, ny, nx, ky, kx);
}

// B images [B][ny][nx] with one kernel
static jt_status conv_dispatch(jt_dtype dtype, int64_t B, int ny, int nx, const void* image, int ky, int kx, const void* kernel,
                               jt_conv_method method, void* workspace, void* out, cudaStream_t st) {
    const jt_conv_method m = resolve_conv_method(dtype, B, ny, nx, ky, kx, method);
    if (m == JT_CONV_DIRECT) return launch_conv_direct(dtype, B, ny, nx, image, ky, kx, kernel, workspace, out, st);
    return launch_conv_fft(dtype, B, ny, nx, image, ky, kx, kernel, workspace, out, st);
}

}  // namespace jt

using namespace jt;

extern "C" {

const char* jt_status_string(jt_status s) {
    switch (s) {
        case JT_OK: return "JT_OK";
        case JT_ERR_INVALID_VALUE: return "JT_ERR_INVALID_VALUE";
        case JT_ERR_UNSUPPORTED: return "JT_ERR_UNSUPPORTED";
        case JT_ERR_WORKSPACE: return "JT_ERR_WORKSPACE";
        case JT_ERR_CUDA: return "JT_ERR_CUDA";
    }
    return "JT_ERR_UNKNOWN";
}
int jt_last_cuda_error(void) { return g_last_cuda_error; }
int jt_version(void) { return JT_VERSION; }
uint64_t jt_kernel_launches(void) { return g_launches; }

// ------------------------------------------------------------------ step 1
size_t jt_ray_shoot_workspace_bytes(jt_dtype dtype, int64_t n_rays, int64_t n_tnfw) {
    if (!valid_dtype(dtype) || n_rays <= 0 || n_tnfw < 0) return 0;
    return plan_trace_rays(dtype, n_rays, n_tnfw).total_bytes;
}

jt_status jt_ray_shoot(jt_dtype dtype, int64_t n_rays, const void* theta_x, const void* theta_y, const jt_lens* lens,
                       void* workspace, size_t workspace_bytes, void* beta_x, void* beta_y, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (n_rays < 0 || !valid_lens(lens)) return JT_ERR_INVALID_VALUE;
    if (n_rays == 0) return JT_OK;
    if (!theta_x || !theta_y || !beta_x || !beta_y) return JT_ERR_INVALID_VALUE;
    if (theta_x == beta_x || theta_y == beta_y || theta_x == beta_y || theta_y == beta_x) return JT_ERR_INVALID_VALUE;
    const TracePlan plan = plan_trace_rays(dtype, n_rays, lens->n_tnfw);
    if (plan.total_bytes > 0 && (!workspace || workspace_bytes < plan.total_bytes)) return JT_ERR_WORKSPACE;
    if ((uintptr_t)workspace & 15) return JT_ERR_INVALID_VALUE;              // the records are fetched by 16-byte bulk copies
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_trace_rays(dtype, n_rays, theta_x, theta_y, lens, plan, workspace, beta_x, beta_y, (cudaStream_t)stream);
}

// ------------------------------------------------------------------ step 2
jt_status jt_source_brightness(jt_dtype dtype, int64_t n, const void* beta_x, const void* beta_y,
                               const jt_sources* sources, void* flux, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (n < 0) return JT_ERR_INVALID_VALUE;
    SrcSet S;
    jt_status s = make_sources(sources, &S);
    if (s != JT_OK) return s;
    if (n == 0) return JT_OK;
    if (!beta_x || !beta_y || !flux || flux == beta_x || flux == beta_y) return JT_ERR_INVALID_VALUE;
    s = check_device();
    if (s != JT_OK) return s;
    return launch_source_brightness(dtype, n, beta_x, beta_y, S, flux, (cudaStream_t)stream);
}

// ------------------------------------------------------------------ step 3
size_t jt_psf_convolve_workspace_bytes(jt_dtype dtype, int32_t ny, int32_t nx, int32_t ky, int32_t kx,
                                       jt_conv_method method) {
    if (!valid_dtype(dtype) || !valid_method(method) || ny < 1 || nx < 1 || !valid_kernel_size(ky, kx)) return 0;
    return conv_ws(dtype, 1, ny, nx, ky, kx, method);
}

static jt_status psf_convolve_impl(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, const void* image, int32_t ky, int32_t kx,
                                   const void* kernel, jt_conv_method method, void* workspace, size_t workspace_bytes,
                                   void* out, void* stream) {
    if (!valid_dtype(dtype) || !valid_method(method)) return JT_ERR_UNSUPPORTED;
    if (B < 0 || ny < 1 || nx < 1 || !valid_kernel_size(ky, kx)) return JT_ERR_INVALID_VALUE;
    if (B == 0) return JT_OK;
    if (!image || !kernel || !out || image == out) return JT_ERR_INVALID_VALUE;
    if (method == JT_CONV_DIRECT && !conv_direct_supported(dtype, ny, nx, ky, kx)) return JT_ERR_UNSUPPORTED;
    if (resolve_conv_method(dtype, B, ny, nx, ky, kx, method) == JT_CONV_FFT && !conv_fft_supported(dtype, ny, nx, ky, kx))
        return JT_ERR_UNSUPPORTED;
    const size_t need = conv_ws(dtype, B, ny, nx, ky, kx, method);
    if (need > 0 && (!workspace || workspace_bytes < need)) return JT_ERR_WORKSPACE;
    if (need > 0 && ((uintptr_t)workspace & 15)) return JT_ERR_INVALID_VALUE;    // double2 partial sums, complex planes
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return conv_dispatch(dtype, B, ny, nx, image, ky, kx, kernel, method, workspace, out, (cudaStream_t)stream);
}

jt_status jt_psf_convolve_plan(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, int32_t ky, int32_t kx, jt_conv_method method,
                               const void* image, jt_conv_plan* plan) {
    if (!valid_dtype(dtype) || !valid_method(method)) return JT_ERR_UNSUPPORTED;
    if (!plan || B < 1 || ny < 1 || nx < 1 || !valid_kernel_size(ky, kx)) return JT_ERR_INVALID_VALUE;
    if (method == JT_CONV_DIRECT && !conv_direct_supported(dtype, ny, nx, ky, kx)) return JT_ERR_UNSUPPORTED;
    const jt_conv_method m = resolve_conv_method(dtype, B, ny, nx, ky, kx, method);
    if (m == JT_CONV_FFT && !conv_fft_supported(dtype, ny, nx, ky, kx)) return JT_ERR_UNSUPPORTED;
    jt_conv_plan p = {};
    if (m == JT_CONV_FFT) conv_fft_describe(dtype, B, ny, nx, ky, kx, &p);
    else conv_direct_describe(dtype, B, ny, nx, ky, kx, image, &p);
    *plan = p;
    return JT_OK;
}

jt_status jt_trace_plan_query(jt_dtype dtype, const jt_grid* grid, int64_t n_rays, int64_t n_tnfw, jt_trace_plan* plan) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (!plan || n_tnfw < 0 || (grid ? !valid_grid(grid) : n_rays < 1)) return JT_ERR_INVALID_VALUE;
    const TracePlan t = grid ? plan_trace_grid(dtype, grid, n_tnfw) : plan_trace_rays(dtype, n_rays, n_tnfw);
    jt_trace_plan p = {};
    p.rays_per_thread = t.R; p.threads = t.threads; p.wide = grid && t.wide ? 1 : 0;
    p.n_chunks = t.n_chunks; p.chunk_len = t.chunk_len; p.n_ctas = t.n_tiles * t.n_chunks;
    p.tile_recs = n_tnfw > 0 ? trace_tile_recs(dtype, t) : 0;
    *plan = p;
    return JT_OK;
}

jt_status jt_psf_convolve(jt_dtype dtype, int32_t ny, int32_t nx, const void* image, int32_t ky, int32_t kx,
                          const void* kernel, jt_conv_method method, void* workspace, size_t workspace_bytes, void* out,
                          void* stream) {
    return psf_convolve_impl(dtype, 1, ny, nx, image, ky, kx, kernel, method, workspace, workspace_bytes, out, stream);
}

size_t jt_psf_convolve_batch_workspace_bytes(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, int32_t ky, int32_t kx,
                                             jt_conv_method method) {
    if (!valid_dtype(dtype) || !valid_method(method) || B < 1 || ny < 1 || nx < 1 || !valid_kernel_size(ky, kx)) return 0;
    return conv_ws(dtype, B, ny, nx, ky, kx, method);
}

jt_status jt_psf_convolve_batch(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, const void* images, int32_t ky, int32_t kx,
                                const void* kernel, jt_conv_method method, void* workspace, size_t workspace_bytes,
                                void* out, void* stream) {
    return psf_convolve_impl(dtype, B, ny, nx, images, ky, kx, kernel, method, workspace, workspace_bytes, out, stream);
}

// ------------------------------------------------------------------ fused image
// workspace layout: [trace partials + counters][pre-PSF image][convolution scratch]
size_t jt_simulate_image_workspace_bytes(jt_dtype dtype, const jt_grid* grid, int64_t n_tnfw, int32_t ky, int32_t kx,
                                         jt_conv_method method) {
    if (!valid_dtype(dtype) || !valid_method(method) || !valid_grid(grid) || n_tnfw < 0) return 0;
    const TracePlan plan = plan_trace_grid(dtype, grid, n_tnfw);
    size_t total = align_up(plan.total_bytes, 256);
    if (ky > 0 || kx > 0) {
        if (!valid_kernel_size(ky, kx)) return 0;
        total += align_up((size_t)grid->nx * grid->ny * dtype_size(dtype), 256);
        total += conv_ws(dtype, 1, grid->ny, grid->nx, ky, kx, method);
    }
    return total;
}

jt_status jt_simulate_image(jt_dtype dtype, const jt_grid* grid, const jt_lens* lens, const jt_sources* sources,
                            int32_t ky, int32_t kx, const void* kernel, jt_conv_method method, void* workspace,
                            size_t workspace_bytes, void* out, void* stream) {
    if (!valid_dtype(dtype) || !valid_method(method)) return JT_ERR_UNSUPPORTED;
    if (!valid_grid(grid) || !valid_lens(lens) || !out) return JT_ERR_INVALID_VALUE;
    SrcSet S;
    jt_status s = make_sources(sources, &S);
    if (s != JT_OK) return s;
    const bool conv = !(ky == 0 && kx == 0 && kernel == nullptr);
    if (conv && (!valid_kernel_size(ky, kx) || !kernel)) return JT_ERR_INVALID_VALUE;
    if (conv && method == JT_CONV_DIRECT && !conv_direct_supported(dtype, grid->ny, grid->nx, ky, kx)) return JT_ERR_UNSUPPORTED;
    if (conv && resolve_conv_method(dtype, 1, grid->ny, grid->nx, ky, kx, method) == JT_CONV_FFT &&
        !conv_fft_supported(dtype, grid->ny, grid->nx, ky, kx))
        return JT_ERR_UNSUPPORTED;
    const size_t need = jt_simulate_image_workspace_bytes(dtype, grid, lens->n_tnfw, conv ? ky : 0, conv ? kx : 0, method);
    if (need > 0 && (!workspace || workspace_bytes < need)) return JT_ERR_WORKSPACE;
    if ((uintptr_t)workspace & 15) return JT_ERR_INVALID_VALUE;              // the records are fetched by 16-byte bulk copies
    s = check_device();
    if (s != JT_OK) return s;
    const TracePlan plan = plan_trace_grid(dtype, grid, lens->n_tnfw);
    char* ws = (char*)workspace;
    void* trace_ws = ws;
    cudaStream_t st = (cudaStream_t)stream;
    const bool prof = g_prof.on;
    if (prof) { g_prof.recorded = false; JT_CUDA_TRY(cudaEventRecord(g_prof.ev[0], st)); }
    // profiling: the kernel's tier counters (in the workspace) are copied to the library's pinned buffer right behind
    // the kernel, so nothing points into the caller's workspace once the call returns
    auto fetch_tiers = [&]() -> jt_status {
        JT_CUDA_TRY(cudaMemcpyAsync(g_prof.host_tiers, trace_tier_counters(plan, trace_ws), JT_N_TIERS * sizeof(uint64_t),
                                    cudaMemcpyDeviceToHost, st));
        g_prof.have_tiers = true;
        return JT_OK;
    };
    if (!conv) {
        s = launch_trace_grid(dtype, grid, lens, S, plan, trace_ws, out, prof, st);
        if (s == JT_OK && prof) {
            JT_CUDA_TRY(cudaEventRecord(g_prof.ev[1], st));
            s = fetch_tiers();
            if (s == JT_OK) JT_CUDA_TRY(cudaEventRecord(g_prof.ev[3], st));
            g_prof.had_conv = false;
            g_prof.recorded = s == JT_OK;
        }
        return s;
    }
    void* pre = ws + align_up(plan.total_bytes, 256);
    void* conv_ws_ptr = (char*)pre + align_up((size_t)grid->nx * grid->ny * dtype_size(dtype), 256);
    s = launch_trace_grid(dtype, grid, lens, S, plan, trace_ws, pre, prof, st);
    if (s != JT_OK) return s;
    if (prof) JT_CUDA_TRY(cudaEventRecord(g_prof.ev[1], st));
    s = conv_dispatch(dtype, 1, grid->ny, grid->nx, pre, ky, kx, kernel, method, conv_ws_ptr, out, st);
    if (s == JT_OK && prof) {
        JT_CUDA_TRY(cudaEventRecord(g_prof.ev[2], st));
        s = fetch_tiers();
        // a fourth record so that jt_profile_tiers can wait for the copy without a device-wide synchronisation
        if (s == JT_OK) JT_CUDA_TRY(cudaEventRecord(g_prof.ev[3], st));
        g_prof.had_conv = true;
        g_prof.recorded = s == JT_OK;
    }
    return s;
}

// ------------------------------------------------------------------ profiling
jt_status jt_profile_enable(int on) {
    if (on && !g_prof.on) {
        for (int i = 0; i < 4; ++i) JT_CUDA_TRY(cudaEventCreate(&g_prof.ev[i]));
        JT_CUDA_TRY(cudaHostAlloc((void**)&g_prof.host_tiers, JT_N_TIERS * sizeof(uint64_t), cudaHostAllocDefault));
        g_prof.on = true;
        g_prof.recorded = false;
        g_prof.have_tiers = false;
    } else if (!on && g_prof.on) {
        for (int i = 0; i < 4; ++i) { cudaEventDestroy(g_prof.ev[i]); g_prof.ev[i] = nullptr; }
        cudaFreeHost(g_prof.host_tiers);
        g_prof.host_tiers = nullptr;
        g_prof.on = false;
        g_prof.recorded = false;
        g_prof.have_tiers = false;
    }
    return JT_OK;
}

jt_status jt_profile_read(float* trace_ms, float* conv_ms) {
    if (!g_prof.on || !g_prof.recorded || !trace_ms || !conv_ms) return JT_ERR_INVALID_VALUE;
    JT_CUDA_TRY(cudaEventSynchronize(g_prof.ev[g_prof.had_conv ? 2 : 1]));
    JT_CUDA_TRY(cudaEventElapsedTime(trace_ms, g_prof.ev[0], g_prof.ev[1]));
    *conv_ms = 0.f;
    if (g_prof.had_conv) JT_CUDA_TRY(cudaEventElapsedTime(conv_ms, g_prof.ev[1], g_prof.ev[2]));
    return JT_OK;
}

jt_status jt_profile_tiers(uint64_t* counts) {
    if (!g_prof.on || !g_prof.recorded || !g_prof.have_tiers || !counts) return JT_ERR_INVALID_VALUE;
    JT_CUDA_TRY(cudaEventSynchronize(g_prof.ev[3]));
    for (int k = 0; k < JT_N_TIERS; ++k) counts[k] = g_prof.host_tiers[k];
    return JT_OK;
}

// ------------------------------------------------------------------ batch
static jt_status simulate_batch_impl(jt_dtype dtype, int64_t B, const jt_grid* grid, const jt_batch_params* p, void* out,
                                     const void* data, const void* sigma, double* chi2, bool want_chi2, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (B < 0 || !valid_grid(grid) || !p) return JT_ERR_INVALID_VALUE;
    if (B == 0) return JT_OK;
    if ((!want_chi2 && !out) || !p->sie || !p->shear || p->n_tnfw < 0 || (p->n_tnfw > 0 && !p->tnfw) || p->n_src < 0 ||
        p->n_src > JT_MAX_SOURCES || (p->n_src > 0 && !p->sersic))
        return JT_ERR_INVALID_VALUE;
    if (want_chi2 && (!data || !sigma || !chi2)) return JT_ERR_INVALID_VALUE;
    const bool conv = !(p->ky == 0 && p->kx == 0 && p->psf == nullptr);
    if (conv && (!valid_kernel_size(p->ky, p->kx) || !p->psf)) return JT_ERR_INVALID_VALUE;
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_batch(dtype, B, grid, p, out, data, sigma, chi2, (cudaStream_t)stream);
}

jt_status jt_simulate_batch(jt_dtype dtype, int64_t B, const jt_grid* grid, const jt_batch_params* p, void* out,
                            void* stream) {
    return simulate_batch_impl(dtype, B, grid, p, out, nullptr, nullptr, nullptr, false, stream);
}

// ------------------------------------------------------------------ SURVEY 8(f) rows
jt_status jt_simulate_batch_chi2(jt_dtype dtype, int64_t B, const jt_grid* grid, const jt_batch_params* p, const void* data,
                                 const void* sigma, void* images, double* chi2, void* stream) {
    return simulate_batch_impl(dtype, B, grid, p, images, data, sigma, chi2, true, stream);
}

jt_status jt_chi2_batch(jt_dtype dtype, int64_t B, int32_t ny, int32_t nx, const void* models, const void* data,
                        const void* sigma, double* chi2, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (B < 0 || ny < 1 || nx < 1) return JT_ERR_INVALID_VALUE;
    if (B == 0) return JT_OK;
    if (!models || !data || !sigma || !chi2) return JT_ERR_INVALID_VALUE;
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_chi2(dtype, B, (int64_t)ny * nx, models, data, sigma, chi2, (cudaStream_t)stream);
}

jt_status jt_lensing_maps(jt_dtype dtype, int64_t n, const void* theta_x, const void* theta_y, const jt_lens* lens,
                          void* kappa, void* gamma1, void* gamma2, void* mu, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (n < 0 || !valid_lens(lens)) return JT_ERR_INVALID_VALUE;
    if (n == 0) return JT_OK;
    if (!theta_x || !theta_y) return JT_ERR_INVALID_VALUE;
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_lensing_maps(dtype, n, theta_x, theta_y, lens, kappa, gamma1, gamma2, mu, (cudaStream_t)stream);
}

jt_status jt_ray_shoot_profiles(jt_dtype dtype, int64_t n, const void* theta_x, const void* theta_y, int64_t n_def,
                                const jt_profile* deflectors, void* beta_x, void* beta_y, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (n < 0 || n_def < 0 || (n_def > 0 && !deflectors)) return JT_ERR_INVALID_VALUE;
    if (n == 0) return JT_OK;
    if (!theta_x || !theta_y || !beta_x || !beta_y || theta_x == beta_x || theta_y == beta_y) return JT_ERR_INVALID_VALUE;
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_ray_shoot_profiles(dtype, n, theta_x, theta_y, n_def, deflectors, beta_x, beta_y, (cudaStream_t)stream);
}

jt_status jt_light_profiles(jt_dtype dtype, int64_t n, const void* beta_x, const void* beta_y, int64_t n_comp,
                            const jt_profile* components, void* flux, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (n < 0 || n_comp < 0 || (n_comp > 0 && !components)) return JT_ERR_INVALID_VALUE;
    if (n == 0) return JT_OK;
    if (!beta_x || !beta_y || !flux || flux == beta_x || flux == beta_y) return JT_ERR_INVALID_VALUE;
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_light_profiles(dtype, n, beta_x, beta_y, n_comp, components, flux, (cudaStream_t)stream);
}

jt_status jt_light_core_sersic(jt_dtype dtype, int64_t n, const void* beta_x, const void* beta_y, const double* params, void* flux,
                               void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (n < 0 || !params || !(params[1] > 0.0) || !(params[2] > 0.0) || !(params[3] > 0.0) || !(params[5] > 0.0))
        return JT_ERR_INVALID_VALUE;
    if (n == 0) return JT_OK;
    if (!beta_x || !beta_y || !flux || flux == beta_x || flux == beta_y) return JT_ERR_INVALID_VALUE;
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_core_sersic(dtype, n, beta_x, beta_y, params, flux, (cudaStream_t)stream);
}

jt_status jt_light_shapelets(jt_dtype dtype, int64_t n, const void* beta_x, const void* beta_y, int32_t n_max, double beta, double cx,
                             double cy, const void* coef, void* flux, void* stream) {
    if (!valid_dtype(dtype)) return JT_ERR_UNSUPPORTED;
    if (n < 0 || n_max < 0 || n_max > JT_MAX_SHAPELET_ORDER || !(beta > 0.0) || !coef) return JT_ERR_INVALID_VALUE;
    if (n == 0) return JT_OK;
    if (!beta_x || !beta_y || !flux || flux == beta_x || flux == beta_y) return JT_ERR_INVALID_VALUE;
    jt_status s = check_device();
    if (s != JT_OK) return s;
    return launch_shapelets(dtype, n, beta_x, beta_y, n_max, beta, cx, cy, coef, flux, (cudaStream_t)stream);
}

// NEXT-4: the ray grid is a grid of its own with supersample 1: [jt_simulate_image workspace on it][fine output]
static jt_grid fine_grid(const jt_grid* g) {
    jt_grid f = *g;
    f.nx = g->nx * g->supersample;
    f.ny = g->ny * g->supersample;
    f.pixel_scale = g->pixel_scale / (double)g->supersample;
    f.supersample = 1;
    return f;
}

size_t jt_simulate_image_supersampled_psf_workspace_bytes(jt_dtype dtype, const jt_grid* grid, int64_t n_tnfw, int32_t ky, int32_t kx,
                                                          jt_conv_method method) {
    if (!valid_dtype(dtype) || !valid_method(method) || !valid_grid(grid) || n_tnfw < 0 || !valid_kernel_size(ky, kx)) return 0;
    const jt_grid f = fine_grid(grid);
    const size_t inner = jt_simulate_image_workspace_bytes(dtype, &f, n_tnfw, ky, kx, method);
    return align_up(inner, 256) + align_up((size_t)f.nx * f.ny * dtype_size(dtype), 256);
}

jt_status jt_simulate_image_supersampled_psf(jt_dtype dtype, const jt_grid* grid, const jt_lens* lens, const jt_sources* sources,
                                             int32_t ky, int32_t kx, const void* kernel_fine, jt_conv_method method, void* workspace,
                                             size_t workspace_bytes, void* out, void* stream) {
    if (!valid_dtype(dtype) || !valid_method(method)) return JT_ERR_UNSUPPORTED;
    if (!valid_grid(grid) || !valid_lens(lens) || !out || !kernel_fine || !valid_kernel_size(ky, kx)) return JT_ERR_INVALID_VALUE;
    const size_t need = jt_simulate_image_supersampled_psf_workspace_bytes(dtype, grid, lens->n_tnfw, ky, kx, method);
    if (!workspace || workspace_bytes < need) return JT_ERR_WORKSPACE;
    const jt_grid f = fine_grid(grid);
    const size_t inner = align_up(jt_simulate_image_workspace_bytes(dtype, &f, lens->n_tnfw, ky, kx, method), 256);
    void* fine_out = (char*)workspace + inner;
    jt_status s = jt_simulate_image(dtype, &f, lens, sources, ky, kx, kernel_fine, method, workspace, inner, fine_out, stream);
    if (s != JT_OK) return s;
    return launch_bin_sum(dtype, grid->ny, grid->nx, grid->supersample, fine_out, out, (cudaStream_t)stream);
}

}  // extern "C"
