// jt_fft.cu -- step 5b placeholder until the hand-written FFT lands.
#include "jt_internal.h"
namespace jt {
size_t fft_conv_workspace_bytes(jt_dtype, int, int, int, int) { return 0; }
jt_status launch_conv_fft(jt_dtype, int, int, const void*, int, int, const void*, void*, void*, cudaStream_t) { return JT_ERR_UNSUPPORTED; }
}
