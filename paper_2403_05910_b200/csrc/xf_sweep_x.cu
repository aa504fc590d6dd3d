// xf_sweep_x.cu -- instantiations and launcher of the x-direction sweep (see xf_sweeps.cuh).
#include "xf_sweeps.cuh"

namespace {
using namespace xf;

template <int NT>
int launch(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status, cudaStream_t s) {
  const long long L = (long long)G.n[1] * G.np[0];
  const int SEGC = X_NCH * 32 - 1;
  const int segs = (int)((L + SEGC - 1) / SEGC);
  const unsigned blocks = (unsigned)(segs * G.n[2]);
  const size_t smem = sizeof(double) * warp_smem_doubles(N, X_LI, X_RR);
  sweep_kernel<NT, 0, X_LI, X_LJ, X_RR, X_MINB><<<blocks, 32, smem, s>>>(G, N, U, prim, E, status, segs);
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}
}  // namespace

int xf_launch_sweep_x(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      cudaStream_t s) {
#define CALL(NT) return launch<NT>(G, N, U, prim, E, status, s)
  XF_DISPATCH_SWEEP_N(N, CALL)
#undef CALL
  return XF_EINVAL;
}

int xf_sweep_x_init() {
  cudaError_t e = cudaSuccess;
#define CALL(NT)                                                                                                   \
  e = cudaFuncSetAttribute(sweep_kernel<NT, 0, X_LI, X_LJ, X_RR, X_MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                           (int)(sizeof(double) * warp_smem_doubles(NT > 0 ? NT : XF_MAXN, X_LI, X_RR)));         \
  if (e != cudaSuccess) return XF_ECUDA;
  CALL(0) CALL(1) CALL(2) CALL(3) CALL(4) CALL(10)
#undef CALL
  return XF_OK;
}
