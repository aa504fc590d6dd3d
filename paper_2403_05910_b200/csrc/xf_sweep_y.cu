// xf_sweep_y.cu -- instantiations and launcher of the y-direction sweep (see xf_sweeps.cuh).
#include "xf_sweeps.cuh"

static int seg_len_for(const XfGrid &G, int n, long long columns) {
  // split long columns when the grid alone cannot fill 148 SMs x 2 blocks; each split costs one extra face
  int nseg = 1;
  while (columns * nseg < 592 && n / (nseg * 2) >= 16) nseg *= 2;
  return (n + nseg - 1) / nseg;
}

int xf_launch_sweep_y(const XfGrid &G, int N, const double *U, const double *p, const double *c, const double *Gam,
                      const double *chi, const XfEpilogue &E, int *status, cudaStream_t s) {
  using namespace xf;
  constexpr int DIR = 1, OD = DIR == 1 ? 2 : 1;
  const int strips = (G.n[0] + 31) / 32;
  const int seg_len = seg_len_for(G, G.n[DIR], (long long)strips * G.n[OD]);
  const int nseg = (G.n[DIR] + seg_len - 1) / seg_len;
  const dim3 grid(strips, G.n[OD], nseg), block(32, YZ_W);
  const size_t smem = sweep_yz_smem(N);
#define CALL(NT) sweep_yz_kernel<NT, DIR><<<grid, block, smem, s>>>(G, N, U, p, c, Gam, chi, E, status, seg_len)
  XF_DISPATCH_SWEEP_N(N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

int xf_sweep_y_init() {
  using namespace xf;
  cudaError_t e = cudaSuccess;
#define CALL(NT)                                                                                          \
  e = cudaFuncSetAttribute(sweep_yz_kernel<NT, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,         \
                           (int)sweep_yz_smem(NT > 0 ? NT : XF_MAXN));                                    \
  if (e != cudaSuccess) return XF_ECUDA;
  CALL(0) CALL(1) CALL(2) CALL(3) CALL(4) CALL(10)
#undef CALL
  return XF_OK;
}
