// float instantiations of the ray-tracing kernel (separate TU so the two dtypes compile in parallel)
#include "jt_trace.cuh"
namespace jt {
template <> jt_status launch_trace_t<float, true>(const TraceArgs<float>& a, int R, cudaStream_t st) { return launch_trace_impl<float, true>(a, R, st); }
template <> jt_status launch_trace_t<float, false>(const TraceArgs<float>& a, int R, cudaStream_t st) { return launch_trace_impl<float, false>(a, R, st); }
}  // namespace jt
