// jt_trace.cu -- host side of the ray-tracing kernels: derived parameters, launch plans, launches;
// plus the unfused step-2 kernel (jt_source_brightness).
#include <math.h>
#include "jt_trace.cuh"

namespace jt {

template <typename T, bool GRID>
jt_status launch_trace_t(const TraceArgs<T>& a, int R, cudaStream_t st);

MacroLens make_macro(const jt_lens* lens) {
    return derive_macro(lens->has_sie, lens->sie_theta_E, lens->sie_e1, lens->sie_e2, lens->sie_cx, lens->sie_cy,
                        lens->has_shear, lens->shear_gamma1, lens->shear_gamma2);
}

jt_status make_sources(const jt_sources* src, SrcSet* out) {
    SrcSet S = {};
    if (!src || src->n < 0 || src->n > JT_MAX_SOURCES) return JT_ERR_INVALID_VALUE;
    S.n = src->n;
    if (S.n > 0 && (!src->amp || !src->R_sersic || !src->n_sersic || !src->e1 || !src->e2 || !src->cx || !src->cy))
        return JT_ERR_INVALID_VALUE;
    for (int k = 0; k < S.n; ++k)
        derive_source(S, k, src->amp[k], src->R_sersic[k], src->n_sersic[k], src->e1[k], src->e2[k], src->cx[k], src->cy[k]);
    *out = S;
    return JT_OK;
}

// ---- plans ----
static int rays_per_thread(int s, bool f64, int64_t M) {
    // next to no subhalos: nothing to amortise over a thread's rays, and the O(rays) epilogue runs ray after ray -- one
    // pixel row per thread puts the most warps on it (C0: 29 CTAs instead of 4, C1: 235 instead of 118)
    if (M <= 16 && s <= 4) return s;
    if (f64) {
        switch (s) { case 1: case 2: case 4: case 8: return 8; case 3: return 6; case 5: return 10; default: return s; }
    }
    switch (s) { case 1: case 2: case 4: case 8: return 8; case 3: return 6; case 5: return 10; case 7: return 14; default: return s; }   // even where it fits: rays go two to a packed instruction
}

// Split of the subhalo list over CTAs.  All CTAs of a launch do the same work, so the launch runs in waves of
// `slots` CTAs (148 SMs x resident CTAs per SM); pick the chunk count c that minimises
//   waves(n_tiles * c) * (records per chunk + fixed per-CTA cost in record units)
// -- e.g. C2 (91 ray tiles, 10,000 subhalos, float): c = 13 gives 1183 CTAs = 4 full waves of 296.
static int trace_threads(bool f64) { return f64 ? TraceCfg<double>::NT : TraceCfg<float>::NT; }

static void plan_chunks(TracePlan* p, int64_t M, int R, bool f64) {
    const int64_t slots = (int64_t)kNumSMs * (f64 ? TraceCfg<double>::OCC : TraceCfg<float>::OCC);
    const int64_t ovh = 48, ovh_split = 24;          // prologue + epilogue; partial-sum publish + reduce
    int64_t best_c = 1;
    if (M > 0 && p->n_tiles > 0) {
        int64_t c_max = M / 64;                      // at least 64 records per chunk
        if (c_max > 4096) c_max = 4096;
        double best = -1.0;
        for (int64_t c = 1; c <= (c_max < 1 ? 1 : c_max); ++c) {
            const int64_t len = (M + c - 1) / c;
            const int64_t nc = (M + len - 1) / len;
            const int64_t waves = (p->n_tiles * nc + slots - 1) / slots;
            const double cost = (double)waves * (double)(len + ovh + (nc > 1 ? ovh_split : 0));
            if (best < 0.0 || cost < best * 0.999) { best = cost; best_c = nc; }
        }
    }
    p->chunk_len = M > 0 ? (M + best_c - 1) / best_c : 1;
    p->n_chunks = M > 0 ? (int)((M + p->chunk_len - 1) / p->chunk_len) : 1;
    if (p->n_chunks < 1) p->n_chunks = 1;
    p->partial_bytes = p->n_chunks > 1 ? (size_t)p->n_chunks * p->n_tiles * R * p->threads * sizeof(double2) : 0;
    p->counter_bytes = p->n_chunks > 1 ? align_up((size_t)p->n_tiles * (p->threads / 32) * sizeof(unsigned int), 256) : 0;   // one per warp tile
    p->rec_bytes = align_up((size_t)M * (f64 ? sizeof(SubRec<double>) : sizeof(SubRec<float>)), 256);
    p->total_bytes = p->partial_bytes + p->counter_bytes + p->tier_bytes + p->rec_bytes;
}

// Ray ownership: a warp tile is cols_per_warp ray columns x R ray rows; the warp tiles of the grid are numbered
// row-major and dealt to CTAs eight at a time, so only the last CTA can be partly empty whatever the grid shape.
static TracePlan plan_trace_grid_t(const jt_grid* g, int64_t n_tnfw, bool f64) {
    TracePlan p = {};
    const int s = g->supersample;
    p.R = rays_per_thread(s, f64, n_tnfw);
    p.cols_per_warp = (32 / s) * s;
    const int NX = g->nx * s, NY = g->ny * s;
    p.tiles_x = (NX + p.cols_per_warp - 1) / p.cols_per_warp;       // warp tiles per row of warp tiles
    p.tiles_y = (NY + p.R - 1) / p.R;
    p.n_wt = (int64_t)p.tiles_x * p.tiles_y;
    p.threads = trace_threads(f64);
    p.n_tiles = (p.n_wt + p.threads / 32 - 1) / (p.threads / 32);
    // s does not divide 32 (3, 5, 6, 7, 9 ...): 2-4 lanes of every warp tile would idle (s = 5: 30 of 32).  The
    // single-image kernel then gives a CTA floor(threads/s)*s adjacent columns and bins through shared memory.
    p.wide = (32 % s) != 0;
    p.cols_per_cta = (p.threads / s) * s;
    p.ctiles_x = (NX + p.cols_per_cta - 1) / p.cols_per_cta;
    p.n_tiles_wide = (int64_t)p.ctiles_x * p.tiles_y;
    p.tier_bytes = 256;
    if (p.wide) p.n_tiles = p.n_tiles_wide;          // the batch kernel keeps warp tiles (n_wt, tiles_x, cols_per_warp)
    plan_chunks(&p, n_tnfw, p.R, f64);
    return p;
}
TracePlan plan_trace_grid(jt_dtype d, const jt_grid* g, int64_t n_tnfw) { return plan_trace_grid_t(g, n_tnfw, d == JT_F64); }

TracePlan plan_trace_rays(jt_dtype d, int64_t n_rays, int64_t n_tnfw) {
    TracePlan p = {};
    p.R = 8;
    p.cols_per_warp = 32;
    p.tiles_x = 1; p.tiles_y = 1;
    p.threads = trace_threads(d == JT_F64);
    p.n_tiles = (n_rays + (int64_t)p.R * p.threads - 1) / ((int64_t)p.R * p.threads);
    p.tier_bytes = 0;
    plan_chunks(&p, n_tnfw, p.R, d == JT_F64);
    return p;
}

// records per shared-memory tile: what fits kStages times beside the float mode's accumulator columns with
// TraceCfg<T>::OCC CTAs per SM, at most 256 (more only delays the first tile), a multiple of 32
template <typename T>
static int pick_tile_recs(int R, int64_t chunk_len) {
    const size_t budget = (size_t)227 * 1024 / TraceCfg<T>::OCC - 2048;
    const size_t dacc = sizeof(T) == 4 ? (size_t)R * TraceCfg<T>::NT * sizeof(double2) : 0;
    const size_t per = kStages * sizeof(SubRec<T>) + (TraceCfg<T>::NT / 32) * 2 * sizeof(unsigned short);
    int64_t tr = budget > dacc + 32 * per ? (int64_t)((budget - dacc) / per) / 32 * 32 : 32;
    if (tr > 256) tr = 256;
    const int64_t need = (chunk_len < 1 ? 1 : chunk_len + 31) / 32 * 32;       // the whole chunk in one tile when it is short
    return (int)(need < tr ? (need < 32 ? 32 : need) : tr);
}

int trace_tile_recs(jt_dtype dtype, const TracePlan& plan) {
    return dtype == JT_F64 ? pick_tile_recs<double>(plan.R, plan.chunk_len) : pick_tile_recs<float>(plan.R, plan.chunk_len);
}

// Fills the lens part of the arguments and enqueues k_make_recs (derived records, zeroed counters).
template <typename T>
static jt_status fill_lens(TraceArgs<T>& a, const jt_lens* lens, const TracePlan& plan, void* workspace, bool count_tiers,
                           cudaStream_t st) {
    a.m = make_macro(lens);
    a.M = lens->n_tnfw;
    a.tn[0] = (const T*)lens->tnfw_cx; a.tn[1] = (const T*)lens->tnfw_cy; a.tn[2] = (const T*)lens->tnfw_Rs;
    a.tn[3] = (const T*)lens->tnfw_alpha_Rs; a.tn[4] = (const T*)lens->tnfw_r_trunc;
    a.n_chunks = plan.n_chunks;
    a.chunk_len = plan.chunk_len;
    a.tile_recs = pick_tile_recs<T>(plan.R, plan.chunk_len);
    a.n_tiles = plan.n_tiles;
    a.partial = (double2*)workspace;
    a.counter = (unsigned int*)((char*)workspace + plan.partial_bytes);
    a.tier_counts = count_tiers ? (unsigned long long*)trace_tier_counters(plan, workspace) : nullptr;
    a.recs = (const SubRec<T>*)((char*)workspace + plan.partial_bytes + plan.counter_bytes + plan.tier_bytes);
    if (a.M > 0) {
        const int64_t n_counter = plan.n_chunks > 1 ? plan.n_tiles * (plan.threads / 32) : 0;
        const int64_t n = a.M > n_counter ? a.M : n_counter;
        const RawTn<T> raw = {{a.tn[0], a.tn[1], a.tn[2], a.tn[3], a.tn[4]}};
        k_make_recs<T><<<(unsigned)((n + 127) / 128), 128, 0, st>>>(a.M, raw, const_cast<SubRec<T>*>(a.recs), a.counter, (int)n_counter,
                                                                   a.tier_counts);
        JT_LAUNCH_CHECK();
    } else if (count_tiers) {
        JT_CUDA_TRY(cudaMemsetAsync(a.tier_counts, 0, kTiers * sizeof(unsigned long long), st));
    }
    return JT_OK;
}

template <typename T>
static jt_status trace_grid_t(const jt_grid* g, const jt_lens* lens, const SrcSet& src, const TracePlan& plan,
                              void* workspace, void* pre_psf, bool count_tiers, cudaStream_t st) {
    TraceArgs<T> a = {};
    const int s = g->supersample;
    a.nx = g->nx; a.ny = g->ny; a.s = s; a.NX = g->nx * s; a.NY = g->ny * s;
    a.hh = 0.5 * (g->pixel_scale / (double)s);
    a.cx = g->cx;
    a.cy = g->cy;
    a.area_over_s2 = g->pixel_scale * g->pixel_scale / ((double)s * (double)s);
    a.cols_per_warp = plan.cols_per_warp;
    a.wtiles_x = plan.tiles_x;
    a.n_wt = plan.n_wt;
    a.wide = plan.wide ? 1 : 0;
    a.cols_per_cta = plan.cols_per_cta;
    a.ctiles_x = plan.ctiles_x;
    const jt_status fs = fill_lens(a, lens, plan, workspace, count_tiers, st);
    if (fs != JT_OK) return fs;
    a.out = (T*)pre_psf;
    a.src = src;
    return launch_trace_t<T, true>(a, plan.R, st);
}

void* trace_tier_counters(const TracePlan& plan, void* workspace) {
    return (char*)workspace + plan.partial_bytes + plan.counter_bytes;
}

jt_status launch_trace_grid(jt_dtype dtype, const jt_grid* g, const jt_lens* lens, const SrcSet& src,
                            const TracePlan& plan, void* workspace, void* pre_psf, bool count_tiers, cudaStream_t st) {
    return dtype == JT_F32 ? trace_grid_t<float>(g, lens, src, plan, workspace, pre_psf, count_tiers, st)
                           : trace_grid_t<double>(g, lens, src, plan, workspace, pre_psf, count_tiers, st);
}

template <typename T>
static jt_status trace_rays_t(int64_t n, const void* tx, const void* ty, const jt_lens* lens, const TracePlan& plan,
                              void* workspace, void* bx, void* by, cudaStream_t st) {
    TraceArgs<T> a = {};
    a.n_rays = n;
    a.tx = (const T*)tx; a.ty = (const T*)ty; a.bx = (T*)bx; a.by = (T*)by;
    const jt_status fs = fill_lens(a, lens, plan, workspace, false, st);
    if (fs != JT_OK) return fs;
    return launch_trace_t<T, false>(a, plan.R, st);
}

jt_status launch_trace_rays(jt_dtype dtype, int64_t n, const void* tx, const void* ty, const jt_lens* lens,
                            const TracePlan& plan, void* workspace, void* bx, void* by, cudaStream_t st) {
    return dtype == JT_F32 ? trace_rays_t<float>(n, tx, ty, lens, plan, workspace, bx, by, st)
                           : trace_rays_t<double>(n, tx, ty, lens, plan, workspace, bx, by, st);
}

// ---- step 2 on caller arrays ----
template <typename T>
__global__ void __launch_bounds__(256) k_source(int64_t n, const T* __restrict__ bx, const T* __restrict__ by,
                                                const __grid_constant__ SrcSet src, T* __restrict__ flux) {
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        flux[i] = (T)sersic_sum<T>(src, (double)bx[i], (double)by[i]);
}

jt_status launch_source_brightness(jt_dtype dtype, int64_t n, const void* bx, const void* by, const SrcSet& src,
                                   void* flux, cudaStream_t st) {
    if (n == 0) return JT_OK;
    int64_t blocks = (n + 255) / 256;
    if (blocks > (int64_t)kNumSMs * 32) blocks = (int64_t)kNumSMs * 32;
    if (dtype == JT_F32)
        k_source<float><<<(unsigned)blocks, 256, 0, st>>>(n, (const float*)bx, (const float*)by, src, (float*)flux);
    else
        k_source<double><<<(unsigned)blocks, 256, 0, st>>>(n, (const double*)bx, (const double*)by, src, (double*)flux);
    JT_LAUNCH_CHECK();
    return JT_OK;
}

}  // namespace jt
