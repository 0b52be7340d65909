// double instantiations of the ray-tracing kernel
#include "jt_trace.cuh"
namespace jt {
template <> jt_status launch_trace_t<double, true>(const TraceArgs<double>& a, int R, cudaStream_t st) { return launch_trace_impl<double, true>(a, R, st); }
template <> jt_status launch_trace_t<double, false>(const TraceArgs<double>& a, int R, cudaStream_t st) { return launch_trace_impl<double, false>(a, R, st); }
}  // namespace jt
