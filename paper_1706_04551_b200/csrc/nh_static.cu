// nh_static.cu -- nh_cfl_dt_static: the CFL time step (eq. (23); R20) of a
// state that lives in the CALLER's device buffers, computed without a context and without a single
// allocation.  include/nh_b200.h says who needs that and what the limits are.
//
// It is a variant of the k_lambda / k_set_dt pair of nh_predictor.cu.  That pair reduces the maximum
// of the per-cell rate into a scalar that belongs to a context (NhScal::lam_bits, cudaMalloc'ed by
// nh_create).  Here the reduction goes through per-CTA partial maxima instead, and those partials
// are the kernel's scratch memory.  They live in the file-scope __device__ array below, which is
// part of the library image: every GPU that loads libnh_b200.so carries its own copy (128 KiB) from
// the moment the module is loaded until the process exits, whether or not this entry point is used.
//
// fp64 only; same operation order as the context path (-fmad=false), and a maximum is exact and
// order independent, so the result is bit-identical to nh_compute_dt on the same state.
#include <cuda_runtime.h>
#include <stdio.h>

#include <mutex>

#define NH_PREC 64
#include "nh_internal.cuh"

constexpr int kThreads = 256;
constexpr int kCellsPerThread = 16;
constexpr int kCellsPerCta = kThreads * kCellsPerThread;                 // 4096
constexpr long long kMaxCells = NH_STATIC_MAX_CELLS;                     // 8192 x 8192
constexpr int kMaxParts = (int)((kMaxCells + kCellsPerCta - 1) / kCellsPerCta);  // 16384 doubles
constexpr int kMaxDevices = 64;

// THE scratch: one partial maximum per CTA of k_cfl_partials.  One array per device, shared by every
// call on that device; it keeps whatever the last call left in it.
static __device__ __align__(256) double g_cfl_partials[kMaxParts];

namespace {

// In host code `g_cfl_partials` is only a handle for the runtime (a host-side shadow variable), NOT
// the device address: handing it to a kernel makes the kernel touch unrelated memory.  The address a
// kernel may use is asked for once per device, with that device current, and remembered here.
std::mutex g_setup_lock;
double* g_partials_of_device[kMaxDevices] = {};

thread_local char g_err[256] = "";

int fail(int code, const char* fmt, const char* detail = "") {
  snprintf(g_err, sizeof(g_err), fmt, detail);
  return code;
}

// per-cell rate (|u| + sqrt(g h)) / dx + (|v| + sqrt(g h)) / dy with the desingularised velocities
// of L447-451 -- restated from nh_predictor.cu so that no existing code had to change
__device__ __forceinline__ double rate_of_cell(double g, double delta, double dx, double dy, double h,
                                               double qx, double qy) {
  double cc = sqrt(g * h);
  double uu = nh64::nh_dsg(h, qx, delta), vv = nh64::nh_dsg(h, qy, delta);
  return (fabs(uu) + cc) / dx + (fabs(vv) + cc) / dy;
}

// CTA b owns cells [b * 4096, (b + 1) * 4096) and writes their maximum rate to partials[b].  Every
// slot a call reads has been written by that same call first, so nothing in the scratch has to
// start at zero and nothing is cleared.
__global__ void __launch_bounds__(kThreads)
k_cfl_partials(size_t nc, double g, double delta, double dx, double dy, const double* __restrict__ h,
               const double* __restrict__ qx, const double* __restrict__ qy,
               double* __restrict__ partials) {
  size_t base = (size_t)blockIdx.x * kCellsPerCta + threadIdx.x;
  double l = 0.0;
#pragma unroll 4
  for (int r = 0; r < kCellsPerThread; ++r) {
    size_t k = base + (size_t)r * kThreads;
    if (k < nc) {
      double v = rate_of_cell(g, delta, dx, dy, h[k], qx[k], qy[k]);
      if (v > l) l = v;
    }
  }
  for (int o = 16; o > 0; o >>= 1) l = fmax(l, __shfl_xor_sync(0xffffffffu, l, o));
  __shared__ double wm[kThreads / 32];
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) wm[wid] = l;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < kThreads / 32; ++w) l = fmax(l, wm[w]);
    partials[blockIdx.x] = l;
  }
}

// one CTA: maximum of the first nparts partials, then dt = CFL / lam (0 when no cell has a rate)
__global__ void __launch_bounds__(1024)
k_cfl_finish(int nparts, const double* __restrict__ partials, double cfl, double* __restrict__ dt_out) {
  double l = 0.0;
  for (int k = threadIdx.x; k < nparts; k += blockDim.x) l = fmax(l, partials[k]);
  for (int o = 16; o > 0; o >>= 1) l = fmax(l, __shfl_xor_sync(0xffffffffu, l, o));
  __shared__ double wm[32];
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) wm[wid] = l;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) l = fmax(l, wm[w]);
    dt_out[0] = (l > 0.0) ? cfl / l : 0.0;
  }
}

// Once per device: check that it can run this library's code and fetch the scratch's device
// address.  Called with the device current.  No allocation: the array already exists on the device.
int scratch_of_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(NH_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e)); }
  if (dev < 0 || dev >= kMaxDevices) return fail(NH_EINVAL, "nh_cfl_dt_static: device ordinal beyond %s", "63");
  std::lock_guard<std::mutex> hold(g_setup_lock);
  if (!g_partials_of_device[dev]) {
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(NH_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e)); }
    if (major != 10) return fail(NH_ECUDA, "nh_cfl_dt_static: %s", "the current device is not sm_100 (the library carries sm_100a code only)");
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_cfl_partials);
    if (e != cudaSuccess || !p) {
      (void)cudaGetLastError();
      return fail(NH_ECUDA, "cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e));
    }
    g_partials_of_device[dev] = (double*)p;
  }
  *out = g_partials_of_device[dev];
  return NH_OK;
}

// a kernel handed a host pointer faults and takes the whole CUDA context with it: refuse it here
bool on_device(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" {

long long nh_cfl_dt_static_max_cells(void) { return kMaxCells; }

const char* nh_static_last_error(void) { return g_err; }

int nh_cfl_dt_static(int nx, int ny, double dx, double dy, double g, double cfl, double delta,
                     const double* h, const double* qx, const double* qy, double* dt_out,
                     void* cuda_stream) {
  g_err[0] = 0;
  if (nx < 1 || ny < 1) return fail(NH_EINVAL, "nh_cfl_dt_static: %s", "nx and ny must be >= 1");
  const long long nc = (long long)nx * (long long)ny;
  if (nc > kMaxCells) {
    snprintf(g_err, sizeof(g_err),
             "nh_cfl_dt_static: %d x %d = %lld cells exceed the %lld cells the built-in scratch array "
             "is sized for (NH_STATIC_MAX_CELLS); use a context (nh_create + nh_compute_dt) instead",
             nx, ny, nc, kMaxCells);
    return NH_EINVAL;
  }
  if (!(dx > 0.0) || !(dy > 0.0) || !(g > 0.0) || !(delta > 0.0) || !(cfl > 0.0 && cfl <= 1.0))
    return fail(NH_EINVAL, "nh_cfl_dt_static: %s", "dx, dy, g, delta must be > 0 and cfl in (0, 1]");
  if (!h || !qx || !qy || !dt_out) return fail(NH_EINVAL, "nh_cfl_dt_static: %s", "null array pointer");
  if (!on_device(h) || !on_device(qx) || !on_device(qy) || !on_device(dt_out))
    return fail(NH_EINVAL, "nh_cfl_dt_static: %s", "h, qx, qy and dt_out must be device pointers");

  double* partials = nullptr;
  int st = scratch_of_current_device(&partials);  // first call on this device: the set-up
  if (st != NH_OK) return st;

  cudaStream_t stream = (cudaStream_t)cuda_stream;
  const int nparts = (int)((nc + kCellsPerCta - 1) / kCellsPerCta);
  k_cfl_partials<<<nparts, kThreads, 0, stream>>>((size_t)nc, g, delta, dx, dy, h, qx, qy, partials);
  k_cfl_finish<<<1, 1024, 0, stream>>>(nparts, partials, cfl, dt_out);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(NH_ECUDA, "nh_cfl_dt_static: kernel launch: %s", cudaGetErrorString(e));
  return NH_OK;
}

}  // extern "C"
