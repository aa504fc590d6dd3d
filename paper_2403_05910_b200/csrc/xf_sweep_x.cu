// xf_sweep_x.cu -- instantiations and launcher of the x-direction sweep (see xf_sweeps.cuh).
#include "xf_sweeps.cuh"

namespace {
using namespace xf;

template <int NT, int RC>
int launch(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
           XfTmapCache *tc, cudaStream_t s) {
  // U [N + 4]; p, c, 1/rho [3]; Gamma, chi_s [N + 1]
  const CUtensorMap *tmU = xf_tmap(tc, G, U, N + 4, 1), *tmP = xf_tmap(tc, G, prim, 3, 1),
                    *tmS = xf_tmap(tc, G, prim + 3 * G.cells, N + 1, 1);
  if (tmU && tmP && tmS) {
    const long long Lf = (long long)G.n[1] * G.np[0];
    const int segc = XW_NCH * XW_CH - 1;
    const int segs = (int)((Lf + segc - 1) / segc);
    const unsigned blocks = (unsigned)(segs * G.n[2]);
    const size_t smem = sizeof(double) * xw_smem_doubles(N);
    sweep_x_ws_kernel<NT, RC><<<blocks, dim3(32, 2 * XW_W), smem, s>>>(G, N, U, E, status, segs, *tmU, *tmP, *tmS);
    return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
  }
  const long long L = (long long)G.n[1] * G.np[0];
  const int SEGC = X_NCH * 32 - 1;
  const int segs = (int)((L + SEGC - 1) / SEGC);
  const unsigned blocks = (unsigned)(segs * G.n[2]);
  constexpr int RR = X_LJ + stencil_cells(RC) - 1;
  const size_t smem = sizeof(double) * warp_smem_doubles(N, X_LI, RR);
  sweep_kernel<NT, 0, X_LI, X_LJ, RR, X_MINB, RC><<<blocks, 32, smem, s>>>(G, N, U, prim, E, status, segs);
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}
}  // namespace

int xf_launch_sweep_x(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      XfTmapCache *tc, cudaStream_t s) {
  const int rc = E.recon == XF_RECON_WENO5 && E.pp ? 3 : E.recon;   // see xf_sweep_y.cu
#define CALL(NT)                                                            \
  switch (rc) {                                                             \
    case 1: return launch<NT, 1>(G, N, U, prim, E, status, tc, s);          \
    case 2: return launch<NT, 2>(G, N, U, prim, E, status, tc, s);          \
    case 3: return launch<NT, 3>(G, N, U, prim, E, status, tc, s);          \
    default: return launch<NT, 0>(G, N, U, prim, E, status, tc, s);         \
  }
  XF_DISPATCH_SWEEP_N(N, CALL)
#undef CALL
  return XF_EINVAL;
}

int xf_sweep_x_init() {
  cudaError_t e = cudaSuccess;
#define CALL2(NT, RC)                                                                                                  \
  e = cudaFuncSetAttribute(sweep_kernel<NT, 0, X_LI, X_LJ, X_LJ + stencil_cells(RC) - 1, X_MINB, RC>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                           (int)(sizeof(double) * warp_smem_doubles(NT > 0 ? NT : XF_MAXN, X_LI, X_LJ + stencil_cells(RC) - 1)));             \
  if (e != cudaSuccess) return XF_ECUDA;                                                                               \
  e = cudaFuncSetAttribute(sweep_x_ws_kernel<NT, RC>, cudaFuncAttributeMaxDynamicSharedMemorySize,                     \
                           (int)(sizeof(double) * xw_smem_doubles(NT > 0 ? NT : XF_MAXN)));                            \
  if (e != cudaSuccess) return XF_ECUDA;
#define CALL(NT)                                                                                                   \
  CALL2(NT, 0) CALL2(NT, 1) CALL2(NT, 2) CALL2(NT, 3)
  CALL(0) CALL(1) CALL(2) CALL(3) CALL(4) CALL(10)
#undef CALL
#undef CALL2
  return XF_OK;
}
