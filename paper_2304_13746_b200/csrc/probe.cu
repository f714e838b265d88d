// probe.cu — fp64 issue-rate probe for the roofline denominator (include/idfx_probe.h).
#include <cuda_runtime.h>

#include "../../include/idfx_probe.h"

namespace {

constexpr int kChains = 8;
constexpr int kIters = 4096;

__global__ void __launch_bounds__(256) k_dfma_chains(double* out, double a, double b) {
  double x[kChains];
#pragma unroll
  for (int c = 0; c < kChains; ++c) x[c] = threadIdx.x * 1e-3 + c;
  for (int it = 0; it < kIters; ++it) {
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = fma(x[c], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < kChains; ++c) s += x[c];
  if (s == 123.456) out[0] = s;  // never true; keeps the chains alive
}

}  // namespace

extern "C" int idfx_probe_fp64(void* cuda_stream, int repeats, double* h_tflops, double* h_tinst) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -4;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -4;
  double* d = nullptr;
  if (cudaMalloc(&d, 8) != cudaSuccess) return -4;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int blocks = sms * 8;
  float best = 1e30f;
  for (int r = 0; r < repeats + 1; ++r) {
    cudaEventRecord(e0, st);
    k_dfma_chains<<<blocks, 256, 0, st>>>(d, 0.999999, 1e-6);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return -4;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (r > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  const double inst = (double)blocks * 256 * kChains * (double)kIters;
  if (h_tinst) *h_tinst = inst / (best * 1e-3) * 1e-12;
  if (h_tflops) *h_tflops = 2.0 * inst / (best * 1e-3) * 1e-12;
  return cudaGetLastError() == cudaSuccess ? 0 : -4;
}
