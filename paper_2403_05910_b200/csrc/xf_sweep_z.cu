// xf_sweep_z.cu -- instantiations and launcher of the z-direction sweep (see xf_sweeps.cuh).
#include <string.h>

#include "xf_sweeps.cuh"

namespace {
constexpr int DIR = 2, OD = DIR == 1 ? 2 : 1;

template <int NT, int RC>
int launch(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
           XfTmapCache *tc, cudaStream_t s) {
  using namespace xf;
  const int strips = (G.n[0] + 31) / 32;
  // one block marches a whole column unless the grid alone cannot fill 148 SMs x 2 blocks a few times over;
  // each split costs one extra face row
  const int n = G.n[DIR];
  int nseg = 1;
  while ((long long)strips * G.n[OD] * nseg < 1184 && n / (nseg * 2) >= 4 * YZ_W) nseg *= 2;
  const int seg_len = (n + nseg - 1) / nseg;
  nseg = (n + seg_len - 1) / seg_len;
  const dim3 grid(strips, G.n[OD], nseg), block(32, 2 * YZ_W);
  const size_t smem = sizeof(double) * yz_smem_doubles(N, YZ_W, stencil_cells(RC));
  // U [N + 4]; p, c, 1/rho [3]; Gamma, chi_s [N + 1]
  const CUtensorMap *tmU = nullptr, *tmP = nullptr, *tmS = nullptr;
  if (G.g[0] > 0) {
    tmU = xf_tmap(tc, G, U, N + 4, 0);
    tmP = xf_tmap(tc, G, prim, 3, 0);
    tmS = xf_tmap(tc, G, prim + 3 * G.cells, N + 1, 0);
  }
  if (tmU && tmP && tmS) {
    sweep_yz_ws_kernel<NT, DIR, YZ_W, true, RC><<<grid, block, smem, s>>>(G, N, U, prim, E, status, seg_len, *tmU, *tmP, *tmS);
  } else {
    CUtensorMap none;   // not read by the cp.async instantiation
    memset(&none, 0, sizeof(none));
    sweep_yz_ws_kernel<NT, DIR, YZ_W, false, RC><<<grid, block, smem, s>>>(G, N, U, prim, E, status, seg_len, none, none, none);
  }
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}
}  // namespace

int xf_launch_sweep_z(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      XfTmapCache *tc, cudaStream_t s) {
  // kernel instantiation: the reconstruction, with WENO5 in its relative-accuracy form when the limiter is on
  const int rc = E.recon == XF_RECON_WENO5 && E.pp ? 3 : E.recon;
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

int xf_sweep_z_init() {
  using namespace xf;
  cudaError_t e = cudaSuccess;
#define CALL2(NT, TM, RC)                                                                                        \
  e = cudaFuncSetAttribute(sweep_yz_ws_kernel<NT, DIR, YZ_W, TM, RC>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                           (int)(sizeof(double) * yz_smem_doubles(NT > 0 ? NT : XF_MAXN, YZ_W, stencil_cells(RC))));                    \
  if (e != cudaSuccess) return XF_ECUDA;
#define CALL(NT) CALL2(NT, true, 0) CALL2(NT, false, 0) CALL2(NT, true, 1) CALL2(NT, false, 1) \
  CALL2(NT, true, 2) CALL2(NT, false, 2) CALL2(NT, true, 3) CALL2(NT, false, 3)
  CALL(0) CALL(1) CALL(2) CALL(3) CALL(4) CALL(10)
#undef CALL
#undef CALL2
  return XF_OK;
}
