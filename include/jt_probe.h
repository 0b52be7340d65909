/*
 * jt_probe.h -- C ABI of libjtprobe: ALU-rate microbenchmarks for bench.py's roofline denominators.
 *
 * NOT part of the product library (libjt, include/jt.h).  SURVEY.md section 8(d) asks that the FP32 / FP64 / SFU
 * rates the ray-tracing kernels are measured against be re-measured in the same run (MEASURED_PEAKS.json holds only
 * HBM and bf16 tensor numbers).  bench.py loads this library, times jt_probe_alu with CUDA events and reports the
 * rates beside the derived peaks (148 SMs x lanes x clock) of DESIGN.md section 6.
 */
#ifndef JT_PROBE_H
#define JT_PROBE_H

#include <stdint.h>

#if defined(__GNUC__)
#define JT_PROBE_API __attribute__((visibility("default")))
#else
#define JT_PROBE_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { JT_PROBE_FFMA = 0, JT_PROBE_FFMA2 = 1, JT_PROBE_DFMA = 2, JT_PROBE_MUFU_RSQ = 3 } jt_probe_kind;

/* Launches `blocks` CTAs of 256 threads on `stream` (a cudaStream_t passed as void*), each thread running 8 independent
 * dependency chains of instruction `kind` for iters * 4 rounds.  *lane_ops (host, may be NULL) receives the number of
 * thread-level instructions of that kind the launch executes (an FFMA2 counts once but performs two FMAs).
 * sink: device scratch of >= 4 bytes.  Returns 0 on success, 1 for bad arguments, 2 for an unknown kind, 4 when the
 * launch failed.  Never synchronises: time it with events on `stream`. */
JT_PROBE_API int jt_probe_alu(int32_t kind, int32_t blocks, int64_t iters, void *sink, int64_t *lane_ops, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* JT_PROBE_H */
