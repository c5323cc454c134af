/*
 * kcs_probe.h -- C ABI of libkcs_probe.so: machine-peak microbenchmarks for bench.py's roofline denominators.
 *
 * BENCH-ONLY.  Not part of the product library (libkcs.so, include/kcs.h).  SURVEY.md 8(d): MEASURED_PEAKS.json
 * holds the HBM copy bandwidth and the bf16 GEMM rate only; the L2 -> SM bandwidth and the FP32 / FP64 FMA rates
 * that bound this path "must be measured in the same run".  Each probe launches a small kernel on `stream`
 * (a cudaStream_t passed as void*, NULL = legacy default stream), takes the best of 5 timed repetitions (CUDA
 * events), SYNCHRONISES that stream and writes *out [host].  Returns 0, or -1 with a message in
 * kcs_probe_last_error().
 */
#ifndef KCS_PROBE_H
#define KCS_PROBE_H

#ifdef __cplusplus
extern "C" {
#endif

#define KCS_PEAK_FP32_TFLOPS 0   /* dependent-free FFMA chains, 2 flop per FMA */
#define KCS_PEAK_FP64_TFLOPS 1   /* the same with DFMA */
#define KCS_PEAK_L2_GBS 2        /* L2-resident 32 MB buffer streamed by every CTA with ld.global.cg */
#define KCS_PEAK_L1_GBS 3        /* 16 KB window per CTA re-read with coalesced LDG.128 (L1 hits) */
#define KCS_PEAK_L2_GATHER_GBS 4 /* whole 128 B lines at random addresses of a 64 MB buffer, ld.global.cg (L1 bypassed) */

int kcs_probe_peak(int what, double *out, void *stream);
const char *kcs_probe_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
