// xf_sweep_x.cu -- instantiations and launcher of the x-direction sweep (see xf_sweeps.cuh).
#include "xf_sweeps.cuh"

int xf_launch_sweep_x(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      cudaStream_t s) {
  using namespace xf;
  const long long L = (long long)G.n[1] * G.np[0];
  const int SEGC = X_NCH * 32 - 1;
  const int segs = (int)((L + SEGC - 1) / SEGC);
  const unsigned blocks = (unsigned)(segs * G.n[2]);
  const size_t smem = sizeof(double) * warp_smem_doubles(N, X_LI, X_LJ);
#define CALL(NT) sweep_kernel<NT, 0, X_LI, X_LJ><<<blocks, 32, smem, s>>>(G, N, U, prim, E, status, segs)
  XF_DISPATCH_SWEEP_N(N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

int xf_sweep_x_init() {
  using namespace xf;
  cudaError_t e = cudaSuccess;
#define CALL(NT)                                                                                           \
  e = cudaFuncSetAttribute(sweep_kernel<NT, 0, X_LI, X_LJ>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                           (int)(sizeof(double) * warp_smem_doubles(NT > 0 ? NT : XF_MAXN, X_LI, X_LJ))); \
  if (e != cudaSuccess) return XF_ECUDA;
  CALL(0) CALL(1) CALL(2) CALL(3) CALL(4) CALL(10)
#undef CALL
  return XF_OK;
}
