/*
 * rw_probe.h -- measurement helper of bench.py, NOT part of the method and not in librw.so:
 * register-resident FP64 issue-rate probes that give the denominators of the FP64 roofline
 * (DESIGN.md section 6).  Built as the separate library librw_probe.so.
 *
 * Like librw.so it never allocates device memory: the caller passes a scratch buffer.
 */
#ifndef RW_PROBE_H_
#define RW_PROBE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Bytes of device scratch rw_probe_fp64_peak needs on the current device (0 on error). */
size_t rw_probe_scratch_bytes(void);

/* kind 0 = DFMA chains (16 independent accumulators per thread), 1 = DMMA m8n8k4 (8 independent accumulator
 * tiles per warp).  Runs 4 timed launches of `iters` iterations on `cuda_stream` (a cudaStream_t), synchronises,
 * and returns the best in TFLOP/s.  scratch_dev: device pointer, >= rw_probe_scratch_bytes().
 * Returns 0, -1 (bad argument) or -3 (a CUDA call failed). */
int rw_probe_fp64_peak(int32_t kind, int32_t iters, void *scratch_dev, size_t scratch_bytes, double *tflops,
                       void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* RW_PROBE_H_ */
