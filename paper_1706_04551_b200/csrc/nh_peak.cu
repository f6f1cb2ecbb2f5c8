// nh_peak.cu -- measurement hooks, not on the path.  First: the fp64 instruction rate of this device, the
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

// Second hook: what the DRAM system gives a plain streaming kernel with the SAME mix of read and
// written planes as one pass of the matrix-free solver (pass B: 5 read + 1 written, pass CA: 8 + 4;
// nh_solver.cu), with ideal access (16-byte loads, fully coalesced, no halo, no arithmetic worth
// naming, no grid barrier).  The copy bandwidth in MEASURED_PEAKS.json is a 1 + 1 mix; HBM gives a
// mix with more streams and a different read : write ratio a different rate, and that rate -- not
// the copy figure -- is the floor the solver's two passes can be held against (bench.py --streammix).
struct MixP { const double2* in[8]; double2* out[4]; };

template <int NR, int NW>
__global__ void __launch_bounds__(256) k_stream_mix(MixP P, size_t n2) {
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n2; k += (size_t)gridDim.x * blockDim.x) {
    double2 a = P.in[0][k];
#pragma unroll
    for (int r = 1; r < NR; ++r) { double2 b = P.in[r][k]; a.x += b.x; a.y += b.y; }
#pragma unroll
    for (int w = 0; w < NW; ++w) P.out[w][k] = make_double2(a.x + w, a.y - w);
  }
}

template <int NR, int NW>
void launch_mix(const MixP& P, size_t n2, int grid, cudaStream_t st) {
  k_stream_mix<NR, NW><<<grid, 256, 0, st>>>(P, n2);
}

}  // namespace

extern "C" int nh_stream_mix_rate(void* cuda_stream, int nread, int nwrite, long long doubles_per_plane,
                                  double* gbytes_per_second) {
  if (!gbytes_per_second || doubles_per_plane < 2 || (doubles_per_plane & 1)) return NH_EINVAL;
  void (*launch)(const MixP&, size_t, int, cudaStream_t) = nullptr;
  if (nread == 1 && nwrite == 1) launch = launch_mix<1, 1>;
  else if (nread == 5 && nwrite == 1) launch = launch_mix<5, 1>;
  else if (nread == 8 && nwrite == 4) launch = launch_mix<8, 4>;
  else if (nread == 6 && nwrite == 1) launch = launch_mix<6, 1>;   // one sweep of k_srj
  else return NH_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return NH_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return NH_ECUDA;
  const size_t bytes = (size_t)doubles_per_plane * sizeof(double), n2 = (size_t)doubles_per_plane / 2;
  MixP P{};
  void* planes[12] = {};
  int np = 0, rc = NH_OK;
  for (int k = 0; k < nread + nwrite && rc == NH_OK; ++k) {
    if (cudaMalloc(&planes[np], bytes) != cudaSuccess) { (void)cudaGetLastError(); rc = NH_ENOMEM; break; }
    cudaMemsetAsync(planes[np], 0, bytes, st);
    if (k < nread) P.in[k] = (const double2*)planes[np]; else P.out[k - nread] = (double2*)planes[np];
    ++np;
  }
  if (rc == NH_OK) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int grid = sms * 8, reps = 10;
    for (int r = 0; r < 3; ++r) launch(P, n2, grid, st);  // warm-up
    cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r) launch(P, n2, grid, st);
    cudaEventRecord(e1, st);
    cudaError_t err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    if (err == cudaSuccess) err = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (err != cudaSuccess || !(ms > 0.f)) { (void)cudaGetLastError(); rc = NH_ECUDA; }
    else *gbytes_per_second = (double)reps * (nread + nwrite) * (double)bytes / (1e-3 * (double)ms) / 1e9;
  }
  for (int k = 0; k < np; ++k) cudaFree(planes[k]);
  return rc;
}

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
