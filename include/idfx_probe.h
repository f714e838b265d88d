/* idfx_probe.h — machine probes used only by bench.py for roofline denominators.  Not part of the method. */
#ifndef IDFX_PROBE_H
#define IDFX_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif

/* Measures the fp64 FMA issue rate of the current device: a grid of 8 CTAs per SM runs chains of independent
 * DFMAs (no memory traffic), timed with CUDA events on `cuda_stream` (best of `repeats`).
 * Writes the rate in TFLOP/s (2 flops per DFMA) to *h_tflops and in 1e12 fp64 instructions/s to *h_tinst.
 * Returns 0, or -4 on a CUDA error.  Synchronises. */
int idfx_probe_fp64(void* cuda_stream, int repeats, double* h_tflops, double* h_tinst);

#ifdef __cplusplus
}
#endif
#endif
