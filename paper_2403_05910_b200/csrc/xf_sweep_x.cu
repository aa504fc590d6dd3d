// xf_sweep_x.cu -- instantiations and launcher of the x-direction sweep (see xf_sweeps.cuh).
#include "xf_sweeps.cuh"

int xf_launch_sweep_x(const XfGrid &G, int N, const double *U, const double *p, const double *c, const double *Gam,
                      const double *chi, const XfEpilogue &E, int *status, cudaStream_t s) {
  using namespace xf;
  const long long L = (long long)G.n[1] * G.np[0];
  const int SEG = XCHUNKS * TX - 1;
  const int segs = (int)((L + SEG - 1) / SEG);
  const unsigned blocks = (unsigned)(segs * G.n[2]);
  const size_t smem = sweep_x_smem(N);
#define CALL(NT) sweep_x_kernel<NT><<<blocks, TX, smem, s>>>(G, N, U, p, c, Gam, chi, E, status, segs)
  XF_DISPATCH_SWEEP_N(N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

int xf_sweep_x_init() {
  using namespace xf;
  cudaError_t e = cudaSuccess;
#define CALL(NT)                                                                                          \
  e = cudaFuncSetAttribute(sweep_x_kernel<NT>, cudaFuncAttributeMaxDynamicSharedMemorySize,               \
                           (int)sweep_x_smem(NT > 0 ? NT : XF_MAXN));                                     \
  if (e != cudaSuccess) return XF_ECUDA;
  CALL(0) CALL(1) CALL(2) CALL(3) CALL(4) CALL(10)
#undef CALL
  return XF_OK;
}
