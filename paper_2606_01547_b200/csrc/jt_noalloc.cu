// jt_noalloc.cu -- jt_ray_shoot_noalloc: jt_ray_shoot for callers that have no way to provide device scratch.
//
// Who this is for.  jt_ray_shoot needs a workspace (the derived subhalo records k_make_recs writes, and -- when the
// subhalo list is split over thread blocks -- the partial sums and arrival counters of k_trace), and jt.h leaves its
// allocation to the caller.  Some callers cannot allocate device memory at the point where they call us:
//   * code running inside a host framework that hands it finished input / output buffers and forbids any allocation
//     in the callback (an XLA / JAX custom call, a plug-in of a serving runtime, a render or acquisition loop with a
//     fixed memory budget): cudaMalloc there either is not allowed or synchronises the whole device;
//   * code that must not disturb another component's memory pool (cudaMalloc outside the pool fragments or fails when
//     the pool already owns nearly all of the 180 GB), or that runs after the process has dropped the privilege /
//     quota to create allocations.
// For them the scratch lives in a file-scope __device__ array of fixed size that is part of the library image: every
// GPU whose context loads libjt holds JT_NOALLOC_SCRATCH_BYTES of it from module load until the process exits,
// whether or not this entry point is ever called.  The inputs and outputs still belong to the caller.
//
// The kernels are the ones jt_ray_shoot launches (launch_trace_rays); nothing in this file or below it calls
// cudaMalloc, cudaFree or a library routine that allocates.
#include <mutex>
#include "jt_internal.h"

namespace {

// The scratch itself.  256-byte alignment covers the 16-byte bulk copies of the record ring and the 256-byte
// sub-buffer alignment of the plan.  In HOST code this name is only a handle for the runtime's symbol table -- not a
// device address; passing it to a kernel would hand the kernel a host pointer.  Host code gets the real address from
// cudaGetSymbolAddress (scratch_of_current_device below).
static __device__ __align__(256) unsigned char g_noalloc_scratch[JT_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_addr[kMaxDevices];     // device address of g_noalloc_scratch on each device, 0 = not looked up yet

// Set-up, once per device, with that device current: each device has its own copy of the array at its own address.
jt_status scratch_of_current_device(void** out) {
    int dev = -1;
    JT_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return JT_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        JT_CUDA_TRY(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return JT_ERR_CUDA;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return JT_OK;
}

}  // namespace

extern "C" {

size_t jt_ray_shoot_noalloc_capacity(void) { return (size_t)JT_NOALLOC_SCRATCH_BYTES; }

jt_status jt_ray_shoot_noalloc(jt_dtype dtype, int64_t n_rays, const void* theta_x, const void* theta_y, const jt_lens* lens,
                               void* beta_x, void* beta_y, void* stream) {
    using namespace jt;
    if (dtype != JT_F32 && dtype != JT_F64) return JT_ERR_UNSUPPORTED;
    if (n_rays < 0 || !lens || lens->n_tnfw < 0) return JT_ERR_INVALID_VALUE;
    if (lens->n_tnfw > 0 && (!lens->tnfw_cx || !lens->tnfw_cy || !lens->tnfw_Rs || !lens->tnfw_alpha_Rs || !lens->tnfw_r_trunc))
        return JT_ERR_INVALID_VALUE;
    if (n_rays == 0) return JT_OK;
    if (!theta_x || !theta_y || !beta_x || !beta_y) return JT_ERR_INVALID_VALUE;
    if (theta_x == beta_x || theta_y == beta_y || theta_x == beta_y || theta_y == beta_x) return JT_ERR_INVALID_VALUE;
    // the same plan jt_ray_shoot would make; its scratch has to fit the array -- a larger problem is refused here,
    // before anything is enqueued, never truncated
    const TracePlan plan = plan_trace_rays(dtype, n_rays, lens->n_tnfw);
    if (plan.total_bytes > (size_t)JT_NOALLOC_SCRATCH_BYTES) return JT_ERR_WORKSPACE;
    int dev = 0, major = 0;
    JT_CUDA_TRY(cudaGetDevice(&dev));
    JT_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return JT_ERR_UNSUPPORTED;
    void* scratch = nullptr;
    const jt_status s = scratch_of_current_device(&scratch);
    if (s != JT_OK) return s;
    // What must start at zero -- the arrival counters of a split subhalo list -- is cleared by k_make_recs at the start
    // of this call like in jt_ray_shoot; records and partial sums are fully written before they are read, so whatever
    // the previous call left in the array is never seen.
    return launch_trace_rays(dtype, n_rays, theta_x, theta_y, lens, plan, scratch, beta_x, beta_y, (cudaStream_t)stream);
}

}  // extern "C"
