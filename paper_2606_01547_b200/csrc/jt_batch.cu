#include "jt_internal.h"
namespace jt {
jt_status launch_batch(jt_dtype, int64_t, const jt_grid*, const jt_batch_params*, void*, cudaStream_t) { return JT_ERR_UNSUPPORTED; }
}
