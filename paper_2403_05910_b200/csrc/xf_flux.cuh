// xf_flux.cuh -- the per-face numerical flux of the directional sweeps for sm_100a (the hot loop: PAPER.md:98-107,
// Eq. 13-15).
//
// One thread computes one face flux Fhat_{i+1/2} = R (F+ + F-) from the six stencil cells staged in shared memory:
//   * Roe-type average of the two adjacent cells (reading R5), c~^2 from the identity that makes L R = I;
//   * the eigenvector matrices are never formed: L V needs one dense functional pi.V (Nv FMAs) plus sparse rows,
//     and because F_m = u_m U_m + p_m (e_n + u_m e_E), the projected flux L F_m is u_m (L U_m) plus a pressure term
//     that is non-zero only for the two acoustic fields and the entropy field -- so the flux is never projected;
//   * local Lax-Friedrichs splitting (Eq. 14; reading R8), WENO5-JS in a common-denominator form with a single
//     reciprocal per reconstruction (reading R7), back-projection with the structure of R (Eq. 15);
//   * every component of Fhat is handed to `emit` the moment it is final, so the caller can difference it against
//     the neighbouring face (Eq. 13) and write it out without holding all Nv components in registers.
// The fp64 pipe bounds this path, so the code minimises fp64 instructions, not bytes.
#pragma once
#include "xf_common.cuh"

namespace xf {

// WENO5-JS value at +1/2 from point values v0..v4 = v_{-2}..v_{+2} (Jiang & Shu; eps = 1e-6, exponent 2).
// Written on first differences D_k; smoothness indicators scaled by 4 (cancels in the weights);
//   result = v2 + (D2 + 2 D3)/6 + [ (2/3) P0 (d0 - d1) + P2 (d1 - d2) ] / [ 2 (P0 + 6 P1 + 3 P2) ],
// with P0 = (s1 s2)^2, P1 = (s0 s2)^2, P2 = (s0 s1)^2, s_k = 4 (eps + beta_k): the Jiang-Shu weights
// d_k/(eps+beta_k)^2 brought to a common denominator, so one reciprocal instead of four divisions.
#ifndef XF_SPECIES_UNROLL
#define XF_SPECIES_UNROLL 3   // measured: 1 (nothing to overlap) and 9 (instruction cache) are both slower
#endif
#define XF_PRAGMA(x) _Pragma(#x)
#define XF_UNROLL(n) XF_PRAGMA(unroll n)

// the nonlinear part of one reconstruction as a fraction num/den and the linear part `base`, from the centre value v2
// and the four first differences D_k = v_k - v_{k-1}
__device__ __forceinline__ void weno5_core(double v2, double D1, double D2, double D3, double D4, double &num,
                                           double &den, double &base) {
  const double d0 = D2 - D1, d1 = D3 - D2, d2 = D4 - D3;
  const double e0 = fma(3.0, D2, -D1);   // v0 - 4 v1 + 3 v2
  const double e1 = D2 + D3;             // v3 - v1
  const double e2 = fma(-3.0, D3, D4);   // 3 v2 - 4 v3 + v4
  const double k133 = 13.0 / 3.0, eps4 = 4.0e-6;
  const double s0 = fma(e0, e0, fma(k133 * d0, d0, eps4));
  const double s1 = fma(e1, e1, fma(k133 * d1, d1, eps4));
  const double s2 = fma(e2, e2, fma(k133 * d2, d2, eps4));
  const double p12 = s1 * s2, p02 = s0 * s2, p01 = s0 * s1;
  const double P0 = p12 * p12, P1 = p02 * p02, P2 = p01 * p01;
  num = fma(P0 * (d0 - d1), 2.0 / 3.0, P2 * (d1 - d2));
  den = fma(6.0, P1, fma(3.0, P2, P0));   // HALF the common denominator: the caller halves the reciprocal (exponent - 1)
  base = fma(fma(2.0, D3, D2), 1.0 / 6.0, v2);
}

__device__ __forceinline__ double weno5_finish(double num, double den, double base) {
  // 1/(2 den): the factor 1/2 is ONE integer subtraction on the exponent field (high word), not an fp64-pipe instruction
  const double rc = xf_rcp(den);
  const double rh = __hiloint2double(__double2hiint(rc) - 0x00100000, __double2loint(rc));
  return fma(num, rh, base);
}

__device__ __forceinline__ double weno5(double v0, double v1, double v2, double v3, double v4) {
  double num, den, base;
  weno5_core(v2, v1 - v0, v2 - v1, v3 - v2, v4 - v3, num, den, base);
  return weno5_finish(num, den, base);
}

// WENO-CU6 (include/xf.h XF_RECON_WENOCU6; PAPER.md:107 ref 34) value at +1/2 from v0..v5 = v_{-2}..v_{+3}.
// Candidates on first differences: q_k = v2 + c_k/6 with c_0 = 5 D2 - 2 D1, c_1 = D2 + 2 D3, c_2 = 4 D3 - D4,
// c_3 = 6 D3 - 5 D4 + 2 D5; beta_0..2 as Jiang-Shu; beta_6 is the six-point measure, a quadratic form of the five
// first differences (translation invariant: no cancellation of large terms; coefficients over 120960, derived exactly
// from the form in tests/golden/wenocu6_beta6_form.txt); tau = beta_6 - (beta_0 + 4 beta_1 + beta_2)/6 and
// alpha_k = d_k (C + tau/(beta_k + eps)), C = 20, eps = 1e-40, brought to the common denominator prod (beta_j + eps):
// one reciprocal per reconstruction.
__device__ __forceinline__ double wenocu6(double v0, double v1, double v2, double v3, double v4, double v5) {
  const double D1 = v1 - v0, D2 = v2 - v1, D3 = v3 - v2, D4 = v4 - v3, D5 = v5 - v4;
  const double d0 = D2 - D1, d1 = D3 - D2, d2 = D4 - D3;
  const double e0 = fma(3.0, D2, -D1), e1 = D2 + D3, e2 = fma(-3.0, D3, D4);
  const double k1312 = 13.0 / 12.0, eps = 1e-40;
  const double b0 = fma(0.25 * e0, e0, fma(k1312 * d0, d0, eps));   // beta_k + eps
  const double b1 = fma(0.25 * e1, e1, fma(k1312 * d1, d1, eps));
  const double b2 = fma(0.25 * e2, e2, fma(k1312 * d2, d2, eps));
  constexpr double s = 1.0 / 120960.0;
  const double t1 = fma(271779.0 * s, D1, fma(-1837242.0 * s, D2, fma(2249110.0 * s, D3, fma(-1213142.0 * s, D4, 245620.0 * s * D5))));
  const double t2 = fma(3544296.0 * s, D2, fma(-9252940.0 * s, D3, fma(5189840.0 * s, D4, -1079386.0 * s * D5)));
  const double t3 = fma(6713736.0 * s, D3, fma(-7947412.0 * s, D4, 1713274.0 * s * D5));
  const double t4 = fma(2534504.0 * s, D4, -1150710.0 * s * D5);
  const double beta6 = fma(D1, t1, fma(D2, t2, fma(D3, t3, fma(D4, t4, 139633.0 * s * D5 * D5))));
  const double tau = beta6 - (b0 + fma(4.0, b1, b2) - 6.0 * eps) * (1.0 / 6.0);
  const double b3 = beta6 + eps;
  // A_k = d_k (20 b_k + tau) prod_{j != k} b_j,  d = (1, 9, 9, 1)/20
  const double p01 = b0 * b1, p23 = b2 * b3;
  const double A0 = fma(20.0, b0, tau) * (b1 * p23);
  const double A1 = 9.0 * fma(20.0, b1, tau) * (b0 * p23);
  const double A2 = 9.0 * fma(20.0, b2, tau) * (p01 * b3);
  const double A3 = fma(20.0, b3, tau) * (p01 * b2);
  const double c0 = fma(5.0, D2, -2.0 * D1), c1 = fma(2.0, D3, D2), c2 = fma(4.0, D3, -D4);
  const double c3 = fma(6.0, D3, fma(-5.0, D4, 2.0 * D5));
  const double num = fma(A0, c0, fma(A1, c1, fma(A2, c2, A3 * c3)));
  const double den = 6.0 * ((A0 + A1) + (A2 + A3));
  return fma(num, xf_rcp(den), v2);
}

// g = R(f+ at i-2..) + R(f- mirrored)  (Eq. 15); RECON: 0 WENO5-JS (five points each), 1 WENO-CU6 (all six)
template <int RECON>
__device__ __forceinline__ double weno_pair(const double (&fp)[6], const double (&fm)[6]) {
  if (RECON == 1)
    return wenocu6(fp[0], fp[1], fp[2], fp[3], fp[4], fp[5]) + wenocu6(fm[5], fm[4], fm[3], fm[2], fm[1], fm[0]);
  return weno5(fp[0], fp[1], fp[2], fp[3], fp[4]) + weno5(fm[5], fm[4], fm[3], fm[2], fm[1]);
}

template <int DIR> struct Axes;
template <> struct Axes<0> { static constexpr int nd = 0, t1 = 1, t2 = 2; };
template <> struct Axes<1> { static constexpr int nd = 1, t1 = 0, t2 = 2; };
template <> struct Axes<2> { static constexpr int nd = 2, t1 = 1, t2 = 0; };

// Staged cell fields, in this order: the Nv conserved variables, then the N + 4 fields the primitives kernel leaves
// in the workspace: p, c, 1/rho, Gamma, chi_1..chi_N.
__host__ __device__ constexpr int nstaged(int N) { return 2 * N + 8; }
__host__ __device__ constexpr int nprimfields(int N) { return N + 4; }

// Numerical flux at one face.  sm: staged fields, field f of stencil cell m at sm[f*FS + o[m]] (m = 0..5 <-> i-2..i+3;
// the face lies between m = 2 and m = 3).  emit(v, Fhat_v, vnext) is called once per component, in the order
// 0, 1+nd, 1+t1, 1+t2, 5, ..., Nv-1, 4 (vnext = the component that follows, -1 after the last).
// visc: XF_VISC_* (include/xf.h); lamg: this direction's three global maxima (GLF only).
// Returns false if the Roe-averaged c~^2 is not positive.
// The fields needed only at the two cells next to the face (Gamma, chi_1..chi_N) are read through a second
// accessor: field g (0 = Gamma, 1 + s = chi_s) of the cell below / above the face at ss[g*SS + s2] / ss[g*SS + s3],
// so a sweep may keep them in a shallower ring than the six-deep stencil fields.
// p, c, 1/rho (six-deep like U) are read through their own base pointer sp (field g at sp[g*FS + o[m]]) so that a
// sweep may place them in a separately aligned box of the same ring row.
template <int DIR, int RECON, class Emit>
__device__ __forceinline__ bool face_flux(const int N, const double *sm, const double *sp, const int FS,
                                          const int (&o)[6], const double *ss, const int SS, const int s2,
                                          const int s3, const int visc, const double *__restrict__ lamg, Emit &emit) {
  constexpr int nd = Axes<DIR>::nd, t1 = Axes<DIR>::t1, t2 = Axes<DIR>::t2;
  
#define XS(f, m) sm[(f) * FS + o[m]]
#define XP(m) sp[o[m]]
#define XC(m) sp[FS + o[m]]
#define XRI(m) sp[2 * FS + o[m]]
#define XA(g) ss[(g) * SS + s2]
#define XB(g) ss[(g) * SS + s3]

  // ---- Roe-type average (reading R5): q~ = (w_a q_a + w_b q_b)/(w_a + w_b), w = sqrt(rho); with
  //      r = w_b/w_a = sqrt(rho_b/rho_a) the weights are 1/(1+r) and r/(1+r)
  const double ria = XRI(2), rib = XRI(3);
  const double r = sqrt(XS(0, 3) * ria);
  const double oa = xf_rcp(1.0 + r), ob = r * oa;
  const double oma = oa * ria, omb = ob * rib;                // weights acting on conserved quantities
  double ut[3];
#pragma unroll
  for (int q = 0; q < 3; ++q) ut[q] = fma(oma, XS(1 + q, 2), omb * XS(1 + q, 3));
  const double Ht = fma(oma, XS(4, 2) + XP(2), omb * (XS(4, 3) + XP(3)));
  const double Gt = fma(oa, XA(0), ob * XB(0));
  const double kt = 0.5 * fma(ut[0], ut[0], fma(ut[1], ut[1], ut[2] * ut[2]));
  const double chiN = fma(oa, XA(N), ob * XB(N));

  // ---- the dense functional pi.U_m for the six stencil cells; species part first
  double rho[6], piU[6];
#pragma unroll
  for (int m = 0; m < 6; ++m) {
    rho[m] = XS(0, m);
    piU[m] = 0.0;
  }
  double c2acc = 0.0;
#pragma unroll 3
  for (int i = 0; i < N - 1; ++i) {
    const double zeta = fma(oa, XA(1 + i), ob * XB(1 + i)) - chiN;
    double y[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) y[m] = XS(5 + i, m);
    const double Yt = fma(oma, y[2], omb * y[3]);
    c2acc = fma(Yt, zeta, c2acc);
#pragma unroll
    for (int m = 0; m < 6; ++m) piU[m] = fma(zeta, y[m], piU[m]);
  }
  // c~^2 = sum_s Y~_s chi~_s + Gamma~ (H~ - k~), with Y~_N = 1 - sum_{i<N} Y~_i
  const double c2 = chiN + c2acc + Gt * (Ht - kt);
  const double ct = sqrt(c2);
  const double h = 0.5 * xf_rcp(c2);  // 1/(2 c~^2)
  const double Prho = fma(Gt, kt, chiN);

  const double hh = 0.5 * h, ghh = Gt * hh, chh = ct * hh;
  double nuU[6], ud[6], qp[6], rp[6];
  double lam_m = 0.0, lam_0 = 0.0, lam_p = 0.0;  // LLF: max over the stencil of |u-c|, |u|, |u+c| (reading R8)
#pragma unroll
  for (int m = 0; m < 6; ++m) {
    const double mn = XS(1 + nd, m);
    const double mdot = fma(ut[nd], mn, fma(ut[t1], XS(1 + t1, m), ut[t2] * XS(1 + t2, m)));
    piU[m] += fma(Prho, rho[m], Gt * (XS(4, m) - mdot));
    nuU[m] = fma(-ut[nd], rho[m], mn);
    ud[m] = mn * XRI(m);
    const double cm = XC(m);
    if (visc == XF_VISC_LLF) {   // max by compare + select: fmax() drags IEEE NaN handling along (a dozen integer
                                 // instructions each); a NaN state is caught by the status flag anyway
      const double tm = fabs(ud[m] - cm), t0 = fabs(ud[m]), tp = fabs(ud[m] + cm);
      lam_m = tm > lam_m ? tm : lam_m;
      lam_0 = t0 > lam_0 ? t0 : lam_0;
      lam_p = tp > lam_p ? tp : lam_p;
    }
    const double pm = XP(m);                           // pressure terms of L F_m, with p_m / (4 c~^2) = hh p_m:
    qp[m] = (ghh * pm) * (ud[m] - ut[nd]);             //   Gamma~ (u_m - u~) p_m / (4 c~^2)
    rp[m] = chh * pm;                                  //   c~ p_m / (4 c~^2)
  }
  if (visc == XF_VISC_ROE) {          // |lambda_n| of the Roe-averaged state (warp-uniform branch)
    lam_m = fabs(ut[nd] - ct);
    lam_0 = fabs(ut[nd]);
    lam_p = fabs(ut[nd] + ct);
  } else if (visc == XF_VISC_GLF) {   // global maxima of this direction, left by the primitives kernel
    lam_m = lamg[0];
    lam_0 = lamg[1];
    lam_p = lamg[2];
  }

  double hud[6];
#pragma unroll
  for (int m = 0; m < 6; ++m) hud[m] = 0.5 * ud[m];
  const double hlm = 0.5 * lam_m, hl0 = 0.5 * lam_0, hlp = 0.5 * lam_p;

  // ---- acoustic (u-c), entropy (u) and acoustic (u+c) fields
  double g0, g1, gL;
  {
    double fp[6], fm[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
      const double a = h * fma(-ct, nuU[m], piU[m]);
      const double pt = qp[m] - rp[m];
      fp[m] = fma(hud[m] + hlm, a, pt);   // (u_m + Lambda)/2: halving is exact, so the halves are formed once
      fm[m] = fma(hud[m] - hlm, a, pt);
    }
    g0 = weno_pair<RECON>(fp, fm);
#pragma unroll
    for (int m = 0; m < 6; ++m) {
      const double a = h * fma(ct, nuU[m], piU[m]);
      const double pt = qp[m] + rp[m];
      fp[m] = fma(hud[m] + hlp, a, pt);
      fm[m] = fma(hud[m] - hlp, a, pt);
    }
    gL = weno_pair<RECON>(fp, fm);
  }
  double ap[6], am[6];  // (u_m +- Lambda_u)/2 for all fields that travel with u
#pragma unroll
  for (int m = 0; m < 6; ++m) {
    ap[m] = hud[m] + hl0;
    am[m] = hud[m] - hl0;
  }
  {
    double fp[6], fm[6];
#pragma unroll
    for (int m = 0; m < 6; ++m) {
      const double a = fma(-2.0 * h, piU[m], rho[m]);
      const double pt = -2.0 * qp[m];
      fp[m] = fma(ap[m], a, pt);
      fm[m] = fma(am[m], a, pt);
    }
    g1 = weno_pair<RECON>(fp, fm);
  }

  // ---- back-projection Fhat = R g (Eq. 15), structured
  const double s = g0 + g1 + gL;
  const double delta = ct * (gL - g0);
  const double invG = xf_rcp(Gt);
  double F4 = fma(Ht, s, fma(ut[nd], delta, -(c2 * invG) * g1));
  emit(0, s, 1 + nd);
  emit(1 + nd, fma(ut[nd], s, delta), 1 + t1);

  // ---- fields travelling with u: two shear fields, N-1 species fields.  alpha_m = V_m - C rho_m with
  //      C = Roe average of V/rho; L F_m = u_m alpha_m, so f+-_m = (u_m +- Lambda)/2 * alpha_m.
  //      The stencil values of the NEXT field are loaded before the current one is reconstructed (software
  //      pipeline): the emit is a store, no later load may be moved above it, and a warp issues in order.
#define XF_LOAD_FIELD(VIDX, V) _Pragma("unroll") for (int m = 0; m < 6; ++m) V[m] = XS(VIDX, m);
#define XF_LINEAR_FIELD(VIDX, V, DEXPR, VNEXT)                                                         \
  {                                                                                                    \
    double fp[6], fm[6];                                                                               \
    const double C = fma(oma, V[2], omb * V[3]);                                                       \
    _Pragma("unroll") for (int m = 0; m < 6; ++m) {                                                    \
      const double a = fma(-C, rho[m], V[m]);                                                          \
      fp[m] = ap[m] * a;                                                                               \
      fm[m] = am[m] * a;                                                                               \
    }                                                                                                  \
    const double g = weno_pair<RECON>(fp, fm);                                                         \
    F4 = fma((DEXPR), g, F4);                                                                          \
    emit(VIDX, fma(C, s, g), VNEXT);                                                                   \
  }
  {
    double Va[6], Vb[6];
    XF_LOAD_FIELD(1 + t1, Va)
    XF_LOAD_FIELD(1 + t2, Vb)
    XF_LINEAR_FIELD(1 + t1, Va, C, 1 + t2)
    double zn = 0.0;
    if (N > 1) {
      XF_LOAD_FIELD(5, Va)
      zn = fma(oa, XA(1), ob * XB(1)) - chiN;
    }
    XF_LINEAR_FIELD(1 + t2, Vb, C, N > 1 ? 5 : 4)
XF_UNROLL(XF_SPECIES_UNROLL)
    for (int i = 0; i < N - 1; ++i) {
      double V[6];
      _Pragma("unroll") for (int m = 0; m < 6; ++m) V[m] = Va[m];
      const double zeta = zn;
      if (i + 2 < N) {
        XF_LOAD_FIELD(6 + i, Va)
        zn = fma(oa, XA(2 + i), ob * XB(2 + i)) - chiN;
      }
      XF_LINEAR_FIELD(5 + i, V, -zeta * invG, i + 2 < N ? 6 + i : 4)
    }
  }
#undef XF_LINEAR_FIELD
#undef XF_LOAD_FIELD
  emit(4, F4, -1);
#undef XS
#undef XA
#undef XP
#undef XC
#undef XRI
#undef XB
  return c2 > 0.0;
}

}  // namespace xf
