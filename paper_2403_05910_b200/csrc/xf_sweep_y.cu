// xf_sweep_y.cu -- instantiations and launcher of the y-direction sweep (see xf_sweeps.cuh).
#include "xf_sweeps.cuh"

int xf_launch_sweep_y(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      cudaStream_t s) {
  using namespace xf;
  constexpr int DIR = 1, OD = DIR == 1 ? 2 : 1;
  const int groups = (G.n[0] + YZ_LI - 1) / YZ_LI;
  // one warp marches a whole column unless it is very long; each split costs one extra face row
  const int n = G.n[DIR];
  const int max_len = YZ_MAXCH * YZ_LJ - 1;
  const int nseg = (n + max_len - 1) / max_len;
  const int seg_len = (n + nseg - 1) / nseg;
  const dim3 grid(groups, G.n[OD], nseg);
  const size_t smem = sizeof(double) * warp_smem_doubles(N, YZ_LI, YZ_LJ);
#define CALL(NT) sweep_kernel<NT, DIR, YZ_LI, YZ_LJ><<<grid, 32, smem, s>>>(G, N, U, prim, E, status, seg_len)
  XF_DISPATCH_SWEEP_N(N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

int xf_sweep_y_init() {
  using namespace xf;
  cudaError_t e = cudaSuccess;
#define CALL(NT)                                                                                               \
  e = cudaFuncSetAttribute(sweep_kernel<NT, 1, YZ_LI, YZ_LJ>, cudaFuncAttributeMaxDynamicSharedMemorySize,     \
                           (int)(sizeof(double) * warp_smem_doubles(NT > 0 ? NT : XF_MAXN, YZ_LI, YZ_LJ)));   \
  if (e != cudaSuccess) return XF_ECUDA;
  CALL(0) CALL(1) CALL(2) CALL(3) CALL(4) CALL(10)
#undef CALL
  return XF_OK;
}
