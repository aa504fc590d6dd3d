// xf_prim.cu -- primitive recovery (Eq. 21) and the CFL max-wave-speed reduction
// (Eq. 17) for sm_100a.  One thread per cell; the species table sits in the
// kernel-parameter constant bank, so every coefficient read is a uniform constant load.
#include "xf_common.cuh"

namespace {

template <int N_T>
struct CellState {
  static constexpr int NS = N_T > 0 ? N_T : XF_MAXN;
  double Y[NS];
  double rho, rinv, vel[3], e, E;
};

// cp_s/R_s and e_s/R_s... at temperature T with the constant-cp continuation outside [Tlo, Thi] (reading R3)
__device__ __forceinline__ void species_cp_h(const XfThermo &th, int s, double T, double Tc, double &cpR, double &hR) {
  const double *a = th.a[s];
  const double *b = th.b[s];
  cpR = fma(Tc, fma(Tc, fma(Tc, fma(Tc, a[4], a[3]), a[2]), a[1]), a[0]);
  const double hp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, b[3], b[2]), b[1]), b[0]), a[0]);
  hR = fma(Tc, hp, a[5]);
  hR = fma(cpR, T - Tc, hR);
}

template <int N_T>
__device__ __forceinline__ void load_cell(const XfGrid &G, int N, const double *__restrict__ U, long long idx,
                                          CellState<N_T> &S) {
  S.rho = U[idx];
  S.rinv = 1.0 / S.rho;
  double k = 0.0;
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    S.vel[q] = U[(1 + q) * G.cells + idx] * S.rinv;
    k = fma(S.vel[q], S.vel[q], k);
  }
  S.E = U[4 * G.cells + idx];
  S.e = fma(S.E, S.rinv, -0.5 * k);
  double sum = 0.0;
#pragma unroll
  for (int i = 0; i < CellState<N_T>::NS - 1; ++i) {
    if (i < N - 1) {
      S.Y[i] = U[(5 + i) * G.cells + idx] * S.rinv;
      sum += S.Y[i];
    }
  }
#pragma unroll
  for (int i = 0; i < CellState<N_T>::NS; ++i)
    if (i == N - 1) S.Y[i] = 1.0 - sum;  // closure: no clipping, no renormalisation (reading R12)
}

// Newton iteration T^{k+1} = T^k + (e - e(T^k))/Cv(T^k) (Eq. 21); returns T, Rbar, Cv at the final T is recomputed
// by the caller.  Stops when |dT| <= rtol |T| or after maxit steps.
template <int N_T>
__device__ __forceinline__ double newton_T(const XfThermo &th, int N, const CellState<N_T> &S, double T, int &iters,
                                           bool &converged) {
  double Rbar = 0.0;
#pragma unroll
  for (int s = 0; s < CellState<N_T>::NS; ++s)
    if (s < N) Rbar = fma(S.Y[s], th.Rs[s], Rbar);
  int k = 0;
  converged = false;
  while (k < th.maxit) {
    const double Tc = fmin(fmax(T, th.Tlo), th.Thi);
    double hm = 0.0, cpm = 0.0;  // sum Y_s h_s, sum Y_s cp_s
#pragma unroll
    for (int s = 0; s < CellState<N_T>::NS; ++s) {
      if (s < N) {
        double cpR, hR;
        species_cp_h(th, s, T, Tc, cpR, hR);
        const double yr = S.Y[s] * th.Rs[s];
        hm = fma(yr, hR, hm);
        cpm = fma(yr, cpR, cpm);
      }
    }
    const double eT = fma(-Rbar, T, hm);
    const double Cv = cpm - Rbar;
    const double Tn = T + (S.e - eT) / Cv;
    ++k;
    const double dT = fabs(Tn - T);
    T = Tn;
    if (dT <= th.rtol * fabs(Tn)) {
      converged = true;
      break;
    }
    if (!(Tn == Tn)) break;
  }
  iters = k;
  return T;
}

// One evaluation site for the species polynomials: the loop body evaluates sum Y_s h_s, sum Y_s cp_s and e_s/R_s at
// the current T; a Newton update follows unless the previous update already converged, in which case the values
// just computed ARE the final ones (C_v, e_s at the converged T, as the problem statement asks: p, Gamma, c, chi_s
// follow from the final T).  One code copy instead of two keeps the kernel at 128 registers = 16 warps per SM.
template <int N_T>
__global__ void __launch_bounds__(128, 4)
prim_kernel(const XfGrid G, const __grid_constant__ XfThermo th, const double *__restrict__ U, double *__restrict__ T,
            double *__restrict__ prim, double *__restrict__ p_out, double *__restrict__ c_out,
            int *__restrict__ status, unsigned long long *__restrict__ itersum) {
  constexpr int NS = CellState<N_T>::NS;
  const int N = N_T > 0 ? N_T : th.N;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int it = 0;
  if (idx < G.cells) {
    const double rho = U[idx];
    const double rinv = xf_rcp(rho);
    double k2 = 0.0;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const double v = U[(1 + q) * G.cells + idx] * rinv;
      k2 = fma(v, v, k2);
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
    double Tk = T[idx];
    double esR[NS], cpm;
    bool fin = false, conv = false;
#pragma unroll 1
    for (;;) {
      const double Tc = fmin(fmax(Tk, th.Tlo), th.Thi);
      double hm = 0.0;
      cpm = 0.0;
#pragma unroll
      for (int s = 0; s < NS; ++s) {
        if (s < N) {
          double cpR, hR;
          species_cp_h(th, s, Tk, Tc, cpR, hR);
          hm = fma(yr[s], hR, hm);
          cpm = fma(yr[s], cpR, cpm);
          esR[s] = hR - Tk;  // e_s / R_s
        }
      }
      if (fin) break;
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
    if (p_out) p_out[idx] = pr;
    if (c_out) c_out[idx] = cs;
    if (prim) {  // what the sweeps stage per cell: p, c, 1/rho, Gamma, chi_s
      prim[idx] = pr;
      prim[G.cells + idx] = cs;
      prim[2 * G.cells + idx] = rinv;
      prim[3 * G.cells + idx] = Gam;
#pragma unroll
      for (int s = 0; s < NS; ++s)
        if (s < N) prim[(4 + s) * G.cells + idx] = th.Rs[s] * fma(-Gam, esR[s], Tk);  // chi_s = R_s T - Gamma e_s
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
}

// S = max over interior cells of sum_d (|u_d| + c)/dx_d.  Non-negative doubles order like their bit patterns,
// so the grid-wide maximum is one 64-bit atomicMax per block.
template <int N_T>
__global__ void __launch_bounds__(256)
wavespeed_kernel(const XfGrid G, const __grid_constant__ XfThermo th, const double *__restrict__ U,
                 double *__restrict__ T, double *__restrict__ S_dev, int *__restrict__ status) {
  const int N = N_T > 0 ? N_T : th.N;
  const long long interior = (long long)G.n[0] * G.n[1] * G.n[2];
  double smax = 0.0;
  for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < interior;
       q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % G.n[0]);
    const long long r = q / G.n[0];
    const int j = (int)(r % G.n[1]);
    const int k = (int)(r / G.n[1]);
    const long long idx = (long long)(k + G.g[2]) * G.st[2] + (long long)(j + G.g[1]) * G.st[1] + (i + G.g[0]);
    CellState<N_T> S;
    load_cell<N_T>(G, N, U, idx, S);
    int it;
    bool conv;
    const double Tn = newton_T<N_T>(th, N, S, T[idx], it, conv);
    const double Tc = fmin(fmax(Tn, th.Tlo), th.Thi);
    double Rbar = 0.0, cpm = 0.0;
#pragma unroll
    for (int s = 0; s < CellState<N_T>::NS; ++s) {
      if (s < N) {
        double cpR, hR;
        species_cp_h(th, s, Tn, Tc, cpR, hR);
        const double yr = S.Y[s] * th.Rs[s];
        Rbar += yr;
        cpm = fma(yr, cpR, cpm);
      }
    }
    const double Cv = cpm - Rbar;
    const double pr = S.rho * Rbar * Tn;
    const double Gam = Rbar / Cv;
    const double cs = sqrt((1.0 + Gam) * pr * S.rinv);
    T[idx] = Tn;
    double s = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d)
      if (G.n[d] > 1) s = fma(fabs(S.vel[d]) + cs, G.inv_d[d], s);
    int flag = 0;
    if (!(S.rho > 0.0) || !(Tn > 0.0) || !(pr > 0.0)) flag |= XF_FLAG_NONPHYSICAL;
    if (!conv) flag |= XF_FLAG_NOCONV;
    if (flag) atomicOr(status, flag);
    if (s == s) smax = fmax(smax, s);
  }
  for (int o = 16; o > 0; o >>= 1) smax = fmax(smax, __shfl_down_sync(0xffffffffu, smax, o));
  __shared__ double wmax[8];
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = smax;
  __syncthreads();
  if (threadIdx.x == 0) {
    double m = wmax[0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, wmax[w]);
    atomicMax(reinterpret_cast<unsigned long long *>(S_dev), (unsigned long long)__double_as_longlong(m));
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
                   double *c, int *status, unsigned long long *itersum, cudaStream_t s) {
  const int threads = 128;
  const unsigned blocks = (unsigned)((G.cells + threads - 1) / threads);
#define CALL(NT) prim_kernel<NT><<<blocks, threads, 0, s>>>(G, Th, U, T, prim, p, c, status, itersum)
  XF_DISPATCH_N(Th.N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

int xf_launch_wavespeed(const XfGrid &G, const XfThermo &Th, const double *U, double *T, double *S_dev, int *status,
                        cudaStream_t s) {
  if (cudaMemsetAsync(S_dev, 0, sizeof(double), s) != cudaSuccess) return XF_ECUDA;
  const int threads = 256;
  const long long interior = (long long)G.n[0] * G.n[1] * G.n[2];
  long long want = (interior + threads - 1) / threads;
  const unsigned blocks = (unsigned)(want < 148 * 8 ? want : 148 * 8);
#define CALL(NT) wavespeed_kernel<NT><<<blocks, threads, 0, s>>>(G, Th, U, T, S_dev, status)
  XF_DISPATCH_N(Th.N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}
