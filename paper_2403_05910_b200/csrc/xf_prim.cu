// xf_prim.cu -- primitive recovery (Eq. 21) and the CFL max-wave-speed reduction
// (Eq. 17) for sm_100a, one kernel.  One thread per cell; the species table sits in the
// kernel-parameter constant bank, so every coefficient read is a uniform constant load.
#include "xf_common.cuh"

namespace {

// The Newton iteration runs on the MIXTURE polynomials: with y_s = Y_s R_s fixed in a cell,
//   sum_s y_s cp_s(T)/R_s = A0 + A1 T + ... + A4 T^4,   sum_s y_s h_s(T)/R_s = T (A0 + B1 T + ... + B4 T^4) + A5,
// A_k = sum_s y_s a_{s,k}, B_k = sum_s y_s b_{s,k}: ten sums over the species once per cell, after which an iteration
// costs two Horner chains instead of two per species.  Only the final e_s(T) (for chi_s) is evaluated per species.
template <int N_T>
__global__ void __launch_bounds__(128, 6)
prim_kernel(const XfGrid G, const __grid_constant__ XfThermo th, const double *__restrict__ U, double *__restrict__ T,
            double *__restrict__ prim, double *__restrict__ p_out, double *__restrict__ c_out,
            int *__restrict__ status, unsigned long long *__restrict__ itersum, double *__restrict__ S_out,
            double *__restrict__ lam_glob) {
  constexpr int NS = N_T > 0 ? N_T : XF_MAXN;
  const int N = N_T > 0 ? N_T : th.N;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int it = 0;
  double lg[9] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  double smax = 0.0;   // this cell's sum_d (|u_d| + c)/dx_d if it is an interior cell and S_out is wanted
  bool interior = true;
  if (S_out && idx < G.cells) {
    const int i = (int)(idx % G.np[0]);
    const long long r = idx / G.np[0];
    const int j = (int)(r % G.np[1]), k = (int)(r / G.np[1]);
    interior = i >= G.g[0] && i < G.g[0] + G.n[0] && j >= G.g[1] && j < G.g[1] + G.n[1] && k >= G.g[2] &&
               k < G.g[2] + G.n[2];
  }
  // xf_max_wavespeed (S_out without the workspace fields) looks at interior cells only: ghosts may be unfilled
  if (idx < G.cells && (interior || prim)) {
    const double rho = U[idx];
    const double rinv = xf_rcp(rho);
    double k2 = 0.0, va[3], vs[3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const double v = U[(1 + q) * G.cells + idx] * rinv;
      k2 = fma(v, v, k2);
      va[q] = fabs(v);
      vs[q] = v;
    }
    const double e = fma(U[4 * G.cells + idx], rinv, -0.5 * k2);
    double yr[NS];  // Y_s R_s
    double sum = 0.0, Rbar = 0.0;
#pragma unroll
    for (int i = 0; i < NS - 1; ++i) {
      if (i < N - 1) {
        const double Y = U[(5 + i) * G.cells + idx] * rinv;
        sum += Y;
        yr[i] = Y * th.Rs[i];
        Rbar += yr[i];
      }
    }
#pragma unroll
    for (int i = 0; i < NS; ++i)
      if (i == N - 1) {  // closure: no clipping, no renormalisation (reading R12)
        yr[i] = (1.0 - sum) * th.Rs[i];
        Rbar += yr[i];
      }
    double A[6], B[4];  // mixture coefficients (a5 = enthalpy constant)
#pragma unroll
    for (int q = 0; q < 6; ++q) A[q] = 0.0;
#pragma unroll
    for (int q = 0; q < 4; ++q) B[q] = 0.0;
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      if (s < N) {
#pragma unroll
        for (int q = 0; q < 6; ++q) A[q] = fma(yr[s], th.a[s][q], A[q]);
#pragma unroll
        for (int q = 0; q < 4; ++q) B[q] = fma(yr[s], th.b[s][q], B[q]);
      }
    }
    double Tk = T[idx];
    double cpm, Tc;
    bool fin = false, conv = false;
#pragma unroll 1
    for (;;) {
      Tc = fmin(fmax(Tk, th.Tlo), th.Thi);
      cpm = fma(Tc, fma(Tc, fma(Tc, fma(Tc, A[4], A[3]), A[2]), A[1]), A[0]);
      if (fin) break;
      const double hp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, B[3], B[2]), B[1]), B[0]), A[0]);
      const double hm = fma(cpm, Tk - Tc, fma(Tc, hp, A[5]));   // constant-cp continuation outside [Tlo, Thi] (R3)
      // Eq. 21: T <- T + (e - e(T)) / C_v(T)
      const double Tn = fma(e - fma(-Rbar, Tk, hm), xf_rcp(cpm - Rbar), Tk);
      ++it;
      conv = fabs(Tn - Tk) <= th.rtol * fabs(Tn);
      fin = conv || it >= th.maxit || !(Tn == Tn);
      Tk = Tn;
    }
    const double iCv = xf_rcp(cpm - Rbar);
    const double pr = rho * Rbar * Tk;  // Eq. 7
    const double Gam = Rbar * iCv;
    const double cs = sqrt((1.0 + Gam) * pr * rinv);
    T[idx] = Tk;
    if (S_out) {   // Eq. 17 / reading R9, interior cells only
      double sc = 0.0;
#pragma unroll
      for (int q = 0; q < 3; ++q)
        if (G.n[q] > 1) sc = fma(va[q] + cs, G.inv_d[q], sc);
      if (interior && sc == sc) smax = sc;
    }
    if (lam_glob) {   // GLF (include/xf.h): this cell's |u_d - c|, |u_d|, |u_d + c|
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        lg[3 * q] = fabs(vs[q] - cs);
        lg[3 * q + 1] = va[q];
        lg[3 * q + 2] = fabs(vs[q] + cs);
      }
    }
    if (p_out) p_out[idx] = pr;
    if (c_out) c_out[idx] = cs;
    if (prim) {  // what the sweeps stage per cell: p, c, 1/rho, Gamma, chi_s
      prim[idx] = pr;
      prim[G.cells + idx] = cs;
      prim[2 * G.cells + idx] = rinv;
      prim[3 * G.cells + idx] = Gam;
      const double dTc = Tk - Tc;
      const bool outside = __any_sync(__activemask(), dTc != 0.0);   // warp-uniform: cp_s only where it is needed
#pragma unroll
      for (int s = 0; s < NS; ++s) {
        if (s < N) {   // chi_s = R_s T - Gamma e_s,  e_s/R_s = h_s/R_s - T
          const double *a = th.a[s];
          const double *b = th.b[s];
          const double hp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, b[3], b[2]), b[1]), b[0]), a[0]);
          double hR = fma(Tc, hp, a[5]);
          if (outside) hR = fma(fma(Tc, fma(Tc, fma(Tc, fma(Tc, a[4], a[3]), a[2]), a[1]), a[0]), dTc, hR);
          prim[(4 + s) * G.cells + idx] = th.Rs[s] * fma(-Gam, hR - Tk, Tk);
        }
      }
    }
    int flag = 0;
    if (!(rho > 0.0) || !(Tk > 0.0) || !(pr > 0.0)) flag |= XF_FLAG_NONPHYSICAL;
    if (!conv) flag |= XF_FLAG_NOCONV;
    if (flag) atomicOr(status, flag);
  }
  if (itersum) {
    unsigned v = (unsigned)it;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(itersum, (unsigned long long)v);
  }
  if (lam_glob) {   // uniform branch; same idea as S below for nine values: lane q of a warp ends up owning maximum q,
                    // so a warp costs one load of the nine running maxima and, rarely, an atomic
    double mine = 0.0;
#pragma unroll
    for (int q = 0; q < 9; ++q) {
      double v = lg[q] == lg[q] ? lg[q] : 0.0;
      for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
      if ((threadIdx.x & 31) == q) mine = v;
    }
    const int q = threadIdx.x & 31;
    if (q < 9 && mine > *reinterpret_cast<volatile double *>(lam_glob + q))
      atomicMax(reinterpret_cast<unsigned long long *>(lam_glob + q), (unsigned long long)__double_as_longlong(mine));
  }
  if (S_out) {   // non-negative doubles order like their bit patterns: one 64-bit atomicMax per warp
    for (int o = 16; o > 0; o >>= 1) smax = fmax(smax, __shfl_down_sync(0xffffffffu, smax, o));
    // the running maximum only grows: a warp whose own maximum is not above it has nothing to add (a million
    // atomics on one address would serialise in L2)
    if ((threadIdx.x & 31) == 0 && smax > *reinterpret_cast<volatile double *>(S_out))
      atomicMax(reinterpret_cast<unsigned long long *>(S_out), (unsigned long long)__double_as_longlong(smax));
  }
}

}  // namespace

#define XF_DISPATCH_N(N, CALL)        \
  switch (N) {                        \
    case 1: { CALL(1); break; }       \
    case 2: { CALL(2); break; }       \
    case 3: { CALL(3); break; }       \
    case 4: { CALL(4); break; }       \
    case 10: { CALL(10); break; }     \
    default: { CALL(0); break; }      \
  }

int xf_launch_prim(const XfGrid &G, const XfThermo &Th, const double *U, double *T, double *prim, double *p,
                   double *c, int *status, unsigned long long *itersum, double *S_out, double *lam_glob,
                   cudaStream_t s) {
  if (S_out && cudaMemsetAsync(S_out, 0, sizeof(double), s) != cudaSuccess) return XF_ECUDA;
  if (lam_glob && cudaMemsetAsync(lam_glob, 0, 9 * sizeof(double), s) != cudaSuccess) return XF_ECUDA;
  const int threads = 128;
  const unsigned blocks = (unsigned)((G.cells + threads - 1) / threads);
#define CALL(NT) prim_kernel<NT><<<blocks, threads, 0, s>>>(G, Th, U, T, prim, p, c, status, itersum, S_out, lam_glob)
  XF_DISPATCH_N(Th.N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

int xf_launch_wavespeed(const XfGrid &G, const XfThermo &Th, const double *U, double *T, double *S_dev, int *status,
                        cudaStream_t s) {
  return xf_launch_prim(G, Th, U, T, nullptr, nullptr, nullptr, status, nullptr, S_dev, nullptr, s);
}
