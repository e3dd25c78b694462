/*
 * rubix_peaks.h -- measurement helpers of the B200 build (NOT part of the paper's method).
 *
 * the accumulate kernel (steps 4-6) is bound by on-chip traffic and plain
 * fp32 issue, not by HBM, and MEASURED_PEAKS.json carries no L2 or shared-memory peak -- "the
 * builder must measure both first".  These entry points do that, and expose per-stage device
 * times so bench.py can report the dominant kernel's duration from CUDA events recorded on the
 * launching stream inside the timed region.
 */
#ifndef RUBIX_B200_PEAKS_H
#define RUBIX_B200_PEAKS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Micro-benchmarks, each timed with CUDA events on `stream` (the call synchronises the stream):
 *   out[0]  L2 -> SM read bandwidth, GB/s: every CTA streams a 32 MiB L2-resident buffer with
 *           16-byte loads (L1 cannot hold it)
 *   out[1]  shared-memory read bandwidth, GB/s: conflict-free 16-byte loads from all SMs
 *   out[2]  fp32 FMA rate, TFLOP/s (2 flop per FMA), independent chains, 3-register form
 *   out[3]  HBM read+write copy bandwidth, GB/s, over min(scratch/2, 1 GiB) bytes
 * scratch: DEVICE, >= 64 MiB.  Returns 0 on success, else a rubix_status value. */
int32_t rubix_measure_peaks(float out[4], void *scratch, size_t scratch_bytes, void *stream);

/* Stage timing.  After rubix_stage_timing_enable(1) every compute call records a CUDA event pair
 * around each of its stages on the caller's stream (about 1 us each, no synchronisation).
 * rubix_stage_timing_read synchronises on the recorded events, adds each stage's elapsed ms into
 * ms[stage] and its launch count into calls[stage], then clears the record.  Stages:
 *   0 particle pass (K1, K2, K2c)   1 accumulate (K3)   2 partial reduce (K3b)
 *   3 PSF/LSF (K4-K6)               4 adjoint (K7) */
#define RUBIX_N_STAGES 5
void rubix_stage_timing_enable(int32_t on);
int32_t rubix_stage_timing_read(float ms[RUBIX_N_STAGES], int32_t calls[RUBIX_N_STAGES]);

#ifdef __cplusplus
}
#endif
#endif
