// xf_probe.cu -- fp64 FMA-throughput probe: the measured denominator of the fp64-pipe roofline (DESIGN.md
// "Roofline").  16 independent register-resident FMA chains per thread, 8 dependent FMAs per chain per round,
// 8 blocks of 256 threads per SM: nothing but the fp64 pipe can limit it.
#include "xf_common.cuh"

namespace {
__global__ void __launch_bounds__(256) probe_fp64_kernel(int iters, double *__restrict__ sink) {
  double x[16];
  const double a = 1.0 + 1e-9 * (double)(threadIdx.x & 7), b = 1e-12 * (double)(blockIdx.x & 3);
#pragma unroll
  for (int q = 0; q < 16; ++q) x[q] = (double)(q + 1) * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int q = 0; q < 16; ++q) x[q] = fma(x[q], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int q = 0; q < 16; ++q) s += x[q];
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace

int xf_probe_fp64_launch(int blocks, int threads, int iters, double *sink, cudaStream_t s) {
  probe_fp64_kernel<<<blocks, threads, 0, s>>>(iters, sink);
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}
