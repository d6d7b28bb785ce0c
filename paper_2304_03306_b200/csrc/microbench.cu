// microbench.cu — ttsh_microbench_fma: a dense fused-multiply-add loop, the arithmetic roof of this GPU as bench.py measures it.
//
// Not part of the method.  The fused row kernel (row_step.cuh) is bound by the plain fp64 / fp32 FMA pipe, not by HBM and not by a
// tensor-core contraction, and MEASURED_PEAKS.json has no figure for that pipe ("measure with an FMA
// micro-benchmark").  This kernel gives the figure: every thread carries CHAINS independent chains x <- x a + b in registers, so the
// only limit is the issue rate of the FMA pipe; bench.py times it with CUDA events and uses flops / time as `roofline.peak`.
#include <cuda_runtime.h>
#include "../../include/ttsh.h"

namespace {

constexpr int CHAINS = 8;       // independent dependency chains per thread (x 8 warps per scheduler: the pipe never waits on latency)
constexpr int UNROLL = 16;

template <typename T>
__global__ void __launch_bounds__(256) k_fma_peak(int rounds, T a, T b, T* __restrict__ sink) {
  T x[CHAINS];
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) x[c] = (T)(threadIdx.x + 32 * c) * (T)0.0009765625;    // exact in both types
  for (int r = 0; r < rounds; ++r) {
#pragma unroll
    for (int u = 0; u < UNROLL; ++u)
#pragma unroll
      for (int c = 0; c < CHAINS; ++c) x[c] = fma(x[c], a, b);
  }
  T s = (T)0;
#pragma unroll
  for (int c = 0; c < CHAINS; ++c) s += x[c];
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;          // keeps the chains alive
}

}  // namespace

extern "C" int ttsh_microbench_fma(ttsh_dtype t, int blocks, int rounds, double a, double b, void* sink, void* cuda_stream,
                                   double* flops_out) {
  if (!sink || blocks < 1 || rounds < 0 || (t != TTSH_F64 && t != TTSH_F32)) return TTSH_ERR_INVALID_ARG;
  cudaStream_t s = reinterpret_cast<cudaStream_t>(cuda_stream);
  if (t == TTSH_F64) k_fma_peak<double><<<blocks, 256, 0, s>>>(rounds, a, b, (double*)sink);
  else k_fma_peak<float><<<blocks, 256, 0, s>>>(rounds, (float)a, (float)b, (float*)sink);
  if (cudaGetLastError() != cudaSuccess) return TTSH_ERR_CUDA;
  if (flops_out) *flops_out = 2.0 * CHAINS * UNROLL * (double)rounds * 256.0 * (double)blocks;
  return TTSH_OK;
}
