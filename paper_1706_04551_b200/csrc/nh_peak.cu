// nh_peak.cu -- measurement hook, not on the path: the fp64 instruction rate of this device, the
// denominator of the predictor's roofline (the fused predictor is bounded by the
// plain fp64 ALUs, not by HBM; "builder measures it").  k_dfma_chains keeps NCHAIN independent
// dependent chains of fused multiply-adds per thread, 8 CTAs of 256 threads per SM, so that the
// fp64 pipe is the only limit; the rate is thread-level DFMA instructions per second from CUDA
// events (2 flops each; divide by 32 for warp instructions as ncu counts them).
#include <cuda_runtime.h>

#include "../../include/nh_b200.h"

namespace {

constexpr int NCHAIN = 8, INNER = 4096;

__global__ void __launch_bounds__(256) k_dfma_chains(double* sink, double a, double b) {
  double x[NCHAIN];
#pragma unroll
  for (int k = 0; k < NCHAIN; ++k) x[k] = 1.0 + 1e-3 * (threadIdx.x + k);
  for (int it = 0; it < INNER; ++it) {
#pragma unroll
    for (int k = 0; k < NCHAIN; ++k) x[k] = fma(x[k], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < NCHAIN; ++k) s += x[k];
  if (s == 12345.678) sink[0] = s;  // never true: keeps the chains alive
}

}  // namespace

extern "C" int nh_fp64_rate(void* cuda_stream, double* dfma_per_second) {
  if (!dfma_per_second) return NH_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return NH_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return NH_ECUDA;
  double* sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return NH_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = sms * 8, reps = 20;
  k_dfma_chains<<<grid, 256, 0, st>>>(sink, 0.999999, 1e-6);  // warm-up
  cudaEventRecord(e0, st);
  for (int r = 0; r < reps; ++r) k_dfma_chains<<<grid, 256, 0, st>>>(sink, 0.999999, 1e-6);
  cudaEventRecord(e1, st);
  cudaError_t err = cudaEventSynchronize(e1);
  float ms = 0.f;
  if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(sink);
  if (err != cudaSuccess || !(ms > 0.f)) { (void)cudaGetLastError(); return NH_ECUDA; }
  *dfma_per_second = (double)reps * grid * 256.0 * NCHAIN * INNER / (1e-3 * (double)ms);
  return NH_OK;
}
