/*
 * rqr_probe.h -- bench-only measurement helper (librqr_probe.so, NOT part of librqr.so or of include/): FP64 peak
 * probes used as the roofline denominator.  MEASURED_PEAKS.json has no FP64 figure, so bench.py
 * measures it with these register-resident kernels and CUDA events.
 */
#ifndef RQR_PROBE_H
#define RQR_PROBE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define RQR_PROBE_DFMA 0 /* chains of independent double fma                         */
#define RQR_PROBE_DMMA 1 /* chains of independent mma.sync.m8n8k4.f64 (SASS DMMA)     */
#define RQR_PROBE_MIX 2  /* even warps DFMA chains, odd warps DMMA chains, in the same CTA: shows whether
                          * the two kinds share one FP64 data path (sum = one peak) or not (sum of peaks) */

/* Launches one probe kernel on `stream` (asynchronous): grid = blocks CTAs of 256 threads, each
 * thread/warp running `iters` rounds of 8 independent accumulator updates.  `d_sink` is a device
 * buffer of at least blocks*256 doubles (results are stored so nothing is optimised away).
 * *flops_out (HOST pointer, may be NULL) receives the flop count of the launch.
 * Returns 0, -k for a bad argument, or -1000 on a launch failure.                            */
int rqr_probe_fp64(int kind, int iters, int blocks, double* d_sink, double* flops_out, void* stream);

#ifdef __cplusplus
}
#endif
#endif
