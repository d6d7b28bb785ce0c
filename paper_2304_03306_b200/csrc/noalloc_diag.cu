// noalloc_diag.cu — ttsh_diagnostics_noalloc: the a7 diagnostics (E, Z, Psi of Eq. 11, polar order, max|v|,
// non-finite count; sums over the entire grid) for callers that have device pointers to v_x, v_y, omega but
// no device memory of their own to lend the library.
//
// Who that is.  Every other call of this library works inside a workspace the caller allocated (ttsh_workspace_bytes ->
// ttsh_create).  Some callers cannot produce one: a monitoring hook that another solver invokes between its steps with
// nothing but the three field pointers; a process in which the framework's caching allocator has already taken all of the
// device memory, so that a raw cudaMalloc fails; code inside a latency-critical loop, where cudaMalloc / cudaFree stall the
// whole device because they synchronise it.  For them the one piece of scratch this reduction needs — one partial record per
// thread block — lives in a file-scope __device__ array below.  It is part of the library image: every GPU on which the
// library gets loaded holds NOALLOC_BYTES (37 KB) of it until the process exits, whether or not this call is ever made.
//
// What follows from a shared, static array (also stated in include/ttsh.h):
//   - the host-side name `g_partial` is only a stand-in for the symbol; the device address comes from cudaGetSymbolAddress,
//     asked once per device with that device current (device_scratch() below), and THAT pointer goes to the kernels.
//     The first call on a device performs this set-up (it may load the module on that device), so make it before any
//     stream capture starts;
//   - the array keeps what the previous call left in it.  Nothing here needs to start at zero: each call launches exactly
//     NOALLOC_BLOCKS blocks, every block overwrites its own record — also a block that found no grid point to work on — and
//     the second kernel reads those NOALLOC_BLOCKS records only after the first has finished on the same stream;
//   - all calls on one device use the same array: two calls whose kernels may overlap on the GPU (different streams, or
//     different host threads on different streams) race on it and return garbage.  Order them on one stream or with events;
//   - no cudaMalloc, cudaFree or allocating library routine is called here, on any path.
//
// The arithmetic is that of k_diag_partial / k_diag_final (pointwise.cuh) in the same launch shape, so the sums agree with
// ttsh_diagnostics on the same fields; this file shares no state with the handle-based path and changes none of it.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>
#include "../../include/ttsh.h"

namespace {

constexpr int NOALLOC_BLOCKS = 592;                    // 4 x 148 SMs, the launch shape of the handle-based diagnostics
constexpr int NOALLOC_THREADS = 256;
constexpr int REC = 8;                                 // [0] sum|v|^2 [1] sum w^2 [2] sum|v| [3] sum|e_theta.v| [4] sum vx [5] sum vy [6] max|v| [7] #nonfinite
constexpr size_t NOALLOC_BYTES = (size_t)NOALLOC_BLOCKS * REC * sizeof(double);   // 37,888 bytes per GPU
constexpr int MAX_SIDE = 16384;                        // the largest grid of the library (ttsh.h: TTSH_ERR_UNSUPPORTED_SIZE)
constexpr int MAX_DEVICES = 64;

// the scratch: one partial record per block.  Host code must never pass `g_partial` itself to a kernel.
static __device__ __align__(256) double g_partial[NOALLOC_BLOCKS * REC];
static_assert(NOALLOC_BYTES == 37888, "the size ttsh.h and the README state");

__device__ __forceinline__ void warp_reduce(double* a) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
    for (int k = 0; k < REC; ++k) {
      const double o = __shfl_down_sync(0xffffffffu, a[k], off);
      if (k == 6) a[k] = fmax(a[k], o); else a[k] += o;
    }
  }
}

__device__ __forceinline__ void block_reduce(double* a, double* out) {
  __shared__ double sh[32][REC];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  warp_reduce(a);
  if (lane == 0)
    for (int k = 0; k < REC; ++k) sh[wid][k] = a[k];
  __syncthreads();
  if (wid == 0) {
    for (int k = 0; k < REC; ++k) a[k] = lane < nw ? sh[lane][k] : 0.0;
    warp_reduce(a);
    if (lane == 0)
      for (int k = 0; k < REC; ++k) out[k] = a[k];
  }
}

// stage 1: grid-stride accumulation in fp64, one record per block into `partial` (= the device address of g_partial)
template <typename T>
__global__ void __launch_bounds__(NOALLOC_THREADS)
k_diag_partial_static(int Nx, int Ny, double dx, double cx, double cy, const T* __restrict__ vx, const T* __restrict__ vy,
                      const T* __restrict__ w, double* __restrict__ partial) {
  double a[REC];
#pragma unroll
  for (int k = 0; k < REC; ++k) a[k] = 0.0;
  const size_t n = (size_t)Nx * Ny;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const double u = (double)vx[i], v = (double)vy[i], ww = (double)w[i];
    const int ix = (int)(i % Nx), iy = (int)(i / Nx);
    const double x = ix * dx - cx, y = iy * dx - cy;
    const double r = sqrt(x * x + y * y);
    const double s2 = u * u + v * v;
    const double vth = r == 0.0 ? 0.0 : (-y * u + x * v) / r;       // e_theta . v  (Eq. 11); r = 0: denominator only
    a[0] += s2;
    a[1] += ww * ww;
    a[2] += sqrt(s2);
    a[3] += fabs(vth);
    a[4] += u;
    a[5] += v;
    a[6] = fmax(a[6], sqrt(s2));
    a[7] += (isfinite(u) ? 0.0 : 1.0) + (isfinite(v) ? 0.0 : 1.0) + (isfinite(ww) ? 0.0 : 1.0);
  }
  block_reduce(a, partial + (size_t)blockIdx.x * REC);              // written by every block, work or no work
}

// stage 2: one block folds the records in a fixed order (deterministic) into the caller's 8 doubles
__global__ void __launch_bounds__(NOALLOC_THREADS)
k_diag_final_static(int nblocks, const double* __restrict__ partial, double* __restrict__ out) {
  double a[REC];
#pragma unroll
  for (int k = 0; k < REC; ++k) a[k] = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x)
#pragma unroll
    for (int k = 0; k < REC; ++k) {
      const double o = partial[(size_t)b * REC + k];
      if (k == 6) a[k] = fmax(a[k], o); else a[k] += o;
    }
  block_reduce(a, out);
}

std::mutex g_setup_lock;
double* g_scratch_of_device[MAX_DEVICES] = {};         // device address of g_partial, per device; nullptr = not asked yet
thread_local char t_error[256] = "";

int fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(t_error, sizeof(t_error), fmt, ap);
  va_end(ap);
  return code;
}

// Once per device, with that device current: the address the kernels must be given.  No allocation: the array already exists
// in the module image on this device.
cudaError_t device_scratch(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> hold(g_setup_lock);
  if (!g_scratch_of_device[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_partial);
    if (e != cudaSuccess) return e;
    g_scratch_of_device[dev] = p;
  }
  *out = g_scratch_of_device[dev];
  return cudaSuccess;
}

}  // namespace

extern "C" {

int ttsh_diagnostics_noalloc(int Nx, int Ny, double dx, ttsh_dtype t, const void* vx, const void* vy, const void* omega,
                             double cx, double cy, double* sums, ttsh_diag* host_out, void* cuda_stream) {
  t_error[0] = 0;
  if (!vx || !vy || !omega || !sums) return fail(TTSH_ERR_INVALID_ARG, "ttsh_diagnostics_noalloc: vx, vy, omega and sums must be non-NULL device pointers");
  if (t != TTSH_F64 && t != TTSH_F32) return fail(TTSH_ERR_INVALID_ARG, "ttsh_diagnostics_noalloc: dtype must be TTSH_F64 (8) or TTSH_F32 (4), got %d", (int)t);
  if (!(dx > 0.0) || !std::isfinite(dx) || !std::isfinite(cx) || !std::isfinite(cy))
    return fail(TTSH_ERR_INVALID_ARG, "ttsh_diagnostics_noalloc: dx must be positive and dx, cx, cy finite");
  if (Nx < 1 || Ny < 1) return fail(TTSH_ERR_INVALID_ARG, "ttsh_diagnostics_noalloc: Nx = %d, Ny = %d must be >= 1", Nx, Ny);
  if (Nx > MAX_SIDE || Ny > MAX_SIDE)
    return fail(TTSH_ERR_UNSUPPORTED_SIZE, "ttsh_diagnostics_noalloc: grid %d x %d exceeds the maximum of %d points per side (%lld points) "
                "this entry point accepts", Nx, Ny, MAX_SIDE, (long long)TTSH_NOALLOC_MAX_POINTS);
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  double* scratch = nullptr;
  cudaError_t e = device_scratch(&scratch);
  if (e != cudaSuccess) return fail(TTSH_ERR_CUDA, "ttsh_diagnostics_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
  if (t == TTSH_F64)
    k_diag_partial_static<double><<<NOALLOC_BLOCKS, NOALLOC_THREADS, 0, s>>>(Nx, Ny, dx, cx, cy, (const double*)vx, (const double*)vy, (const double*)omega, scratch);
  else
    k_diag_partial_static<float><<<NOALLOC_BLOCKS, NOALLOC_THREADS, 0, s>>>(Nx, Ny, dx, cx, cy, (const float*)vx, (const float*)vy, (const float*)omega, scratch);
  e = cudaGetLastError();
  if (e == cudaSuccess) {
    k_diag_final_static<<<1, NOALLOC_THREADS, 0, s>>>(NOALLOC_BLOCKS, scratch, sums);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) return fail(TTSH_ERR_CUDA, "ttsh_diagnostics_noalloc: launch: %s", cudaGetErrorString(e));
  if (!host_out) return TTSH_OK;                       // asynchronous: the caller reads sums[8] in stream order

  double rec[REC];
  e = cudaMemcpyAsync(rec, sums, sizeof(rec), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(TTSH_ERR_CUDA, "ttsh_diagnostics_noalloc: reading the sums back: %s", cudaGetErrorString(e));
  const double P = (double)Nx * (double)Ny;
  ttsh_diag d;
  d.t = 0.0; d.step = 0;                               // no handle, no clock
  d.kinetic_energy = 0.5 * rec[0] / P;
  d.enstrophy = 0.5 * rec[1] / P;
  d.sum_speed = rec[2]; d.sum_abs_vtheta = rec[3];
  d.mean_vx = rec[4] / P; d.mean_vy = rec[5] / P;
  d.max_speed = rec[6];
  d.nonfinite = (long long)rec[7];
  if (rec[2] > 0.0) {
    const double two_over_pi = 2.0 / acos(-1.0);
    d.vortex_order = (rec[3] / rec[2] - two_over_pi) / (1.0 - two_over_pi);   // Eq. (11)
    d.polar_order = hypot(rec[4], rec[5]) / rec[2];
  } else {
    d.vortex_order = 0.0;
    d.polar_order = 0.0;
  }
  *host_out = d;
  return TTSH_OK;
}

const char* ttsh_diagnostics_noalloc_error(void) { return t_error; }

}  // extern "C"
