// xf_react.cu -- the reaction step for sm_100a (Eq. 8-12
// Eq. 27-28: the alpha-QSS predictor-corrector of CHEMEQ2 inside a Lie-Trotter / Strang splitting; readings R24-R30 of
// DESIGN.md).  One thread per interior cell, cells are independent: rho, rho u and E stay fixed, the species are advanced
// over dt in n_sub sub-steps of one predictor and n_corr correctors, the temperature follows from the fixed internal
// energy by the Newton iteration of Eq. 21 after every update.  Per-thread arrays (mass fractions, concentrations, rates)
// live in shared memory as [species][thread] so that the reaction loop can index them by species number; the mechanism
// is a kernel parameter in a compiled form (reactant / product species lists, at most three of each per reaction): all
// threads of a warp walk the same reaction, so every access to it is a uniform constant-bank load.
// ALU-bound by construction (a handful of exponentials per reaction per rate evaluation); no code shared with oracle/.
#include "xf_common.cuh"

namespace {

constexpr int RT = 64;   // threads per block
static_assert(sizeof(XfMechDev) + sizeof(XfThermo) + sizeof(XfGrid) + 64 < 32 * 1024, "kernel parameters: 32 KB on sm_100a");

__device__ __forceinline__ double qss_alpha(double r) {   // reading R26
  if (r < 0.1) {
    const double r2 = r * r;
    return fma(r, fma(-r2, fma(-r2, fma(-r2, 1.0 / 1209600.0, 1.0 / 30240.0), 1.0 / 720.0), 1.0 / 12.0), 0.5);
  }
  const double em = 1.0 - exp(-r);
  return (1.0 - em / r) / em;
}

struct Cell {            // what a thread keeps in registers
  double rho, e, T;
};

// T from the fixed internal energy and the composition Y[s * RT] (Eq. 21); returns false if not converged
__device__ bool newton_T(const XfThermo &th, const int N, const double *Y, const double e, double &T) {
  double Tk = T;
  for (int it = 0; it < th.maxit; ++it) {
    const double Tc = fmin(fmax(Tk, th.Tlo), th.Thi);
    double Rbar = 0.0, em = 0.0, cpm = 0.0;
    for (int s = 0; s < N; ++s) {
      const double *a = th.a[s], *b = th.b[s];
      const double cp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, a[4], a[3]), a[2]), a[1]), a[0]);
      const double hp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, b[3], b[2]), b[1]), b[0]), a[0]);
      const double hR = fma(cp, Tk - Tc, fma(Tc, hp, a[5]));        // h_s / R_s with the constant-cp continuation (R3)
      const double yr = Y[s * RT] * th.Rs[s];
      Rbar += yr;
      em = fma(yr, hR - Tk, em);                                     // e_s = h_s - R_s T
      cpm = fma(yr, cp, cpm);
    }
    const double Tn = Tk + (e - em) / (cpm - Rbar);
    const bool conv = fabs(Tn - Tk) <= th.rtol * fabs(Tn);
    Tk = Tn;
    if (conv) { T = Tk; return true; }
    if (!(Tn == Tn)) break;
  }
  T = Tk;
  return false;
}

// q[s], d[s] (production and destruction rates of Y_s, 1/time) at (rho, Y, T); conc and g are scratch  (Eq. 9-12)
// The reaction loop accumulates MOLAR rates (sum of R_f, R_b per species); the factor W_s / rho of Eq. 9 is applied once
// per species afterwards instead of once per reaction and species (those divisions were 11 % of the warp samples).
__device__ void rates(const XfThermo &th, const XfMechDev &mm, const int N, const double rho, const double *Y,
                      const double T, double *conc, double *g, double *q, double *d) {
  const XfMechDev *m = &mm;
  const double Tc = fmin(fmax(T, th.Tlo), th.Thi), lnTc = log(Tc), lnr = log(T / Tc), iT = 1.0 / T;
  for (int s = 0; s < N; ++s) {
    const double *a = th.a[s], *b = th.b[s];
    conc[s * RT] = rho * Y[s * RT] * m->iW[s];
    const double cp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, a[4], a[3]), a[2]), a[1]), a[0]);
    const double hp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, b[3], b[2]), b[1]), b[0]), a[0]);
    const double hR = fma(cp, T - Tc, fma(Tc, hp, a[5]));
    // S_s/R_s = a1 ln T + a2 T + a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7 (+ cp ln(T/Tc) outside the fit range)
    const double SR = fma(a[0], lnTc, fma(Tc, fma(Tc, fma(Tc, fma(Tc, a[4] * 0.25, a[3] * (1.0 / 3.0)), a[2] * 0.5), a[1]), m->a7[s])) +
                      cp * lnr;
    g[s * RT] = SR - hR * iT;
    q[s * RT] = 0.0;
    d[s * RT] = 0.0;
  }
  const double lnT = log(T), iRT = 1.0 / (m->Ru * T), lnp = log(m->p_atm * iRT);
  for (int r = 0; r < m->NR; ++r) {
    // three reactant and three product slots, the unused ones (index 0, a valid species) switched off by a warp-uniform
    // predicate: fixed trip counts, so all index loads and shared-memory reads of a reaction are in flight together
    // (as loops over n_r, n_p their control flow and dependent loads were 28 % of the warp samples)
    const int nr = m->n_r[r], np = m->n_p[r];
    int sr[3], sp[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      sr[k] = m->re[r][k] * RT;
      sp[k] = m->pr[r][k] * RT;
    }
    double dg = 0.0, Rf = 1.0, Rb = 1.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const double gr = g[sr[k]], cr = conc[sr[k]], gp = g[sp[k]], cp = conc[sp[k]];
      if (k < nr) {
        dg -= gr;
        Rf *= cr;
      }
      if (k < np) {
        dg += gp;
        Rb *= cp;
      }
    }
    const double kf = m->A[r] * exp(fma(m->B[r], lnT, -m->E[r] * iRT));               // Eq. 11 (reading R24)
    const double kb = kf * exp(-fma((double)(np - nr), lnp, dg));                      // k_f / K_c, Eq. 12
    double tb = 1.0;
    if (m->third[r]) {
      double t0 = 0.0, t1 = 0.0;                                  // two chains: the sum was one dependent FMA per species
      int s = 0;
      for (; s + 1 < N; s += 2) {
        t0 = fma(m->eff[r][s], conc[s * RT], t0);
        t1 = fma(m->eff[r][s + 1], conc[(s + 1) * RT], t1);
      }
      if (s < N) t0 = fma(m->eff[r][s], conc[s * RT], t0);
      tb = t0 + t1;
    }
    Rf *= tb * kf;
    Rb *= tb * kb;
#pragma unroll
    for (int k = 0; k < 3; ++k) {                                                       // Eq. 9 split as Eq. 27 (R25)
      if (k < nr) {
        d[sr[k]] += Rf;
        q[sr[k]] += Rb;
      }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      if (k < np) {
        q[sp[k]] += Rf;
        d[sp[k]] += Rb;
      }
    }
  }
  const double rinv = 1.0 / rho;
  for (int s = 0; s < N; ++s) {
    const double w = m->W[s] * rinv;
    q[s * RT] *= w;
    d[s * RT] *= w;
  }
}

__global__ void __launch_bounds__(RT)
react_kernel(const XfGrid G, const __grid_constant__ XfThermo th, const __grid_constant__ XfMechDev m, double *__restrict__ U,
             double *__restrict__ T, const double dt, const int n_sub, const int n_corr, int *__restrict__ status) {
  const int N = th.N;
  extern __shared__ double sh[];                                   // 8 arrays [N][RT]
  double *Y0 = sh + threadIdx.x, *Yp = Y0 + N * RT, *q0 = Yp + N * RT, *p0 = q0 + N * RT, *conc = p0 + N * RT,
         *g = conc + N * RT, *q = g + N * RT, *d = q + N * RT;
  // interior cell of this thread
  const long long t = (long long)blockIdx.x * RT + threadIdx.x;
  const long long ncell = (long long)G.n[0] * G.n[1] * G.n[2];
  if (t >= ncell) return;
  const int i = (int)(t % G.n[0]);
  const long long r2 = t / G.n[0];
  const int j = (int)(r2 % G.n[1]), k = (int)(r2 / G.n[1]);
  const long long idx = (i + G.g[0]) + (long long)(j + G.g[1]) * G.st[1] + (long long)(k + G.g[2]) * G.st[2];
  const long long C = G.cells;
  const double rho = U[idx], rinv = 1.0 / rho;
  double k2 = 0.0, sum = 0.0;
  for (int c = 0; c < 3; ++c) {
    const double v = U[(1 + c) * C + idx] * rinv;
    k2 = fma(v, v, k2);
  }
  const double e = fma(U[4 * C + idx], rinv, -0.5 * k2);           // fixed over the step (reading R29)
  for (int s = 0; s < N - 1; ++s) {
    const double y = U[(5 + s) * C + idx] * rinv;
    Y0[s * RT] = y;
    sum += y;
  }
  Y0[(N - 1) * RT] = 1.0 - sum;
  double Tk = T[idx];
  bool ok = newton_T(th, N, Y0, e, Tk);
  const double h = dt / n_sub;
  for (int sub = 0; sub < n_sub; ++sub) {
    rates(th, m, N, rho, Y0, Tk, conc, g, q0, d);
    sum = 0.0;
    for (int s = 0; s < N - 1; ++s) {                              // predictor, Eq. 28
      const double y = Y0[s * RT];
      const double p = y > 0.0 ? d[s * RT] / y : 0.0;
      p0[s * RT] = p;
      const double yp = y + h * (q0[s * RT] - p * y) / fma(qss_alpha(p * h), p * h, 1.0);
      Yp[s * RT] = yp;
      sum += yp;
    }
    Yp[(N - 1) * RT] = 1.0 - sum;
    double Tp = Tk;
    for (int it = 0; it < n_corr; ++it) {                          // corrector(s) (reading R27)
      ok = newton_T(th, N, Yp, e, Tp) && ok;
      rates(th, m, N, rho, Yp, Tp, conc, g, q, d);
      sum = 0.0;
      for (int s = 0; s < N - 1; ++s) {
        const double y0 = Y0[s * RT], yp = Yp[s * RT];
        const double pp = yp > 0.0 ? d[s * RT] / yp : 0.0;
        const double pb = 0.5 * (p0[s * RT] + pp);
        const double ab = qss_alpha(pb * h);
        const double qb = fma(ab, q[s * RT], (1.0 - ab) * q0[s * RT]);
        const double yc = y0 + h * (qb - pb * y0) / fma(ab, pb * h, 1.0);
        Yp[s * RT] = yc;                                           // Yp[s] is not read again in this loop
        sum += yc;
      }
      Yp[(N - 1) * RT] = 1.0 - sum;
    }
    for (int s = 0; s < N; ++s) Y0[s * RT] = Yp[s * RT];
    Tk = Tp;
    ok = newton_T(th, N, Y0, e, Tk) && ok;
  }
  for (int s = 0; s < N - 1; ++s) U[(5 + s) * C + idx] = rho * Y0[s * RT];
  T[idx] = Tk;
  int flag = 0;
  if (!ok) flag |= XF_FLAG_NOCONV;
  if (!(Tk > 0.0)) flag |= XF_FLAG_NONPHYSICAL;
  if (flag) atomicOr(status, flag);
}

}  // namespace

int xf_launch_react(const XfGrid &G, const XfThermo &Th, const XfMechDev &mech, double *U, double *T, double dt,
                    int n_sub, int n_corr, int *status, cudaStream_t s) {
  const long long ncell = (long long)G.n[0] * G.n[1] * G.n[2];
  const unsigned blocks = (unsigned)((ncell + RT - 1) / RT);
  const size_t smem = sizeof(double) * 8 * (size_t)Th.N * RT;
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(react_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(double) * 8 * XF_MAXN * RT));
    attr_done = true;
  }
  react_kernel<<<blocks, RT, smem, s>>>(G, Th, mech, U, T, dt, n_sub, n_corr, status);
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}
