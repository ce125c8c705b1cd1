/*
 * su2_probe.h -- measurement aid of bench.py (libsu2probe.so), NOT part of the product ABI (su2_heff.h).
 *
 * MEASURED_PEAKS.json carries no FP64 entry, so the roofline denominator of the FP64 tensor path (SURVEY.md 8(d):
 * "measured best of a register-resident DFMA loop, a DMMA.8x8x4 loop ...") is measured live, in the same run.
 */
#ifndef SU2_PROBE_H
#define SU2_PROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Register-resident FP64 throughput of the current device in TFLOP/s (best of 3 timed launches, CUDA events on
 * cuda_stream; synchronises).  kind 0: DFMA loop (FP64 vector pipe); kind 1: mma.sync.m8n8k4.f64 loop (SASS
 * DMMA.8x8x4).  tflops: HOST.  Returns 0, -1 (bad argument) or -5 (a CUDA call failed). */
int32_t su2_probe_fp64_peak(int32_t kind, int32_t iters, int32_t ctas_per_sm, double* tflops, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
