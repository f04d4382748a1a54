/*
 * gcamb_probe.h -- roofline denominators measured on the device (libgcamb_probe.so).
 *
 * NOT part of the method and not part of libgcamb_los.so: bench.py loads this small library to
 * measure, in its own process, what the FP64 units of the GPU it runs on deliver, so that the
 * derived peak of DESIGN.md section 7 (148 SMs x 64 DFMA lanes x 2 flop x SM clock; reading R20)
 * stands beside a measured number.  Both calls enqueue one kernel on `cuda_stream` (a cudaStream_t
 * cast to void*) and return a cudaError_t value as int (0 = success); the caller times them with
 * CUDA events.  d_out is a DEVICE buffer of blocks*threads doubles (a sink that keeps the work live).
 */
#ifndef GCAMB_PROBE_H
#define GCAMB_PROBE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Pure dependent-chain DFMA kernel: 8 independent chains per thread, `iters` FMAs per chain;
 * exactly blocks * threads * 8 * iters DFMAs = 2 flop each.  1 <= threads <= 1024. */
int gcamb_probe_dfma(int32_t blocks, int32_t threads, int64_t iters, double *d_out, void *cuda_stream);

/* FP64 tensor-core probe: 8 independent mma.sync.m8n8k4.f64 accumulator chains per warp, `iters`
 * MMAs per chain; exactly blocks * (threads/32) * 8 * iters MMAs = 256 FMA = 512 flop each.
 * threads must be a multiple of 32.  (the batched tau-sum is a dense
 * contraction; this is the rate its accumulate could run at on the tensor pipe.) */
int gcamb_probe_dmma(int32_t blocks, int32_t threads, int64_t iters, double *d_out, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* GCAMB_PROBE_H */
