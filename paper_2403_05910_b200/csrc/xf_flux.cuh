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

// The same reconstruction as v2 + sum_k A_k c_k / (6 sum_k A_k), A = (P0, 6 P1, 3 P2), 6 (q_k - v2) = c_k = 5 D2 - 2 D1 |
// D2 + 2 D3 | 4 D3 - D4.  weno5() above is q_1 + [weighted (q_k - q_1)]: when the stencil that carries the weight is
// NOT the central one and holds values many orders below its neighbours' (a trace species next to a cell where it is
// abundant), an O(max |v|) candidate is cancelled by the correction and the result has the ABSOLUTE error eps max|v|.
// That is far below the 1e-12-of-the-row tolerance of a residual, but the positivity limiter divides by such a flux:
// theta = (q^LF - eps)/(q^LF - q) amplifies it by max|v|/|q^LF - q|.  In this form every term is either small or carries
// a small weight, so the result keeps its RELATIVE accuracy; two fp64 instructions more per reconstruction.  Used by
// the sweeps when the limiter is on (kernel instantiation RECON = 3).
__device__ __forceinline__ double weno5_rel(double v0, double v1, double v2, double v3, double v4) {
  const double D1 = v1 - v0, D2 = v2 - v1, D3 = v3 - v2, D4 = v4 - v3;
  const double d0 = D2 - D1, d1 = D3 - D2, d2 = D4 - D3;
  const double e0 = fma(3.0, D2, -D1), e1 = D2 + D3, e2 = fma(-3.0, D3, D4);
  const double k133 = 13.0 / 3.0, eps4 = 4.0e-6;
  const double s0 = fma(e0, e0, fma(k133 * d0, d0, eps4));
  const double s1 = fma(e1, e1, fma(k133 * d1, d1, eps4));
  const double s2 = fma(e2, e2, fma(k133 * d2, d2, eps4));
  const double p12 = s1 * s2, p02 = s0 * s2, p01 = s0 * s1;
  const double A0 = p12 * p12, A1 = 6.0 * (p02 * p02), A2 = 3.0 * (p01 * p01);
  const double c0 = fma(5.0, D2, -2.0 * D1), c1 = fma(2.0, D3, D2), c2 = fma(4.0, D3, -D4);
  const double num = fma(A0, c0, fma(A1, c1, A2 * c2));
  const double den = 6.0 * (A0 + (A1 + A2));
  return fma(num, xf_rcp(den), v2);
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

// WENO7 (include/xf.h XF_RECON_WENO7; PAPER.md:107 ref 36; reading R18) value at +1/2 from v0..v6 = v_{-3}..v_{+3}.
// Four cubic candidates on cells (k-3..k), linear weights (1, 12, 18, 4)/35, alpha_k = d_k/(eps + beta_k)^2, eps = 1e-6.
// On first differences D_j = v_j - v_{j-1} and second differences E_j = D_{j+1} - D_j:
//   12 (q_k - v3) = 3 D1 - 10 D2 + 13 D3 | -D2 + 4 D3 + 3 D4 | D3 + 6 D4 - D5 | 9 D4 - 4 D5 + D6
// and the Jiang-Shu measure of a cubic p over its target cell is a sum of three squares (Legendre expansion of dp/dx):
//   beta = A^2 + (13/12) S^2 + (781/720) T^2,  A = p(+1/2) - p(-1/2), S = dx^2 d2p/dx2 (0), T = dx^3 d3p/dx3
//   6 A_k = 2 D1 - 7 D2 + 11 D3 | -D2 + 5 D3 + 2 D4 | 2 D3 + 5 D4 - D5 | 11 D4 - 7 D5 + 2 D6
//   S_k   = 2 E2 - E1 | E3 | E3 | 2 E4 - E5;   T_k = E_{k+2} - E_{k+1}
// (the oracle evaluates the same measure as a quadratic form of the first differences with an integer table; the two
// forms are equal polynomials).  The four weights are brought to the common denominator prod (eps + beta_j)^2: one
// reciprocal per reconstruction; indicators scaled by 36 (cancels in the weights).
__device__ __forceinline__ double weno7(double v0, double v1, double v2, double v3, double v4, double v5, double v6) {
  const double D1 = v1 - v0, D2 = v2 - v1, D3 = v3 - v2, D4 = v4 - v3, D5 = v5 - v4, D6 = v6 - v5;
  const double E1 = D2 - D1, E2 = D3 - D2, E3 = D4 - D3, E4 = D5 - D4, E5 = D6 - D5;
  const double A0 = fma(11.0, D3, fma(-7.0, D2, 2.0 * D1));
  const double A1 = fma(5.0, D3, fma(2.0, D4, -D2));
  const double A2 = fma(5.0, D4, fma(2.0, D3, -D5));
  const double A3 = fma(11.0, D4, fma(-7.0, D5, 2.0 * D6));
  const double S0 = fma(2.0, E2, -E1), S3 = fma(2.0, E4, -E5);
  const double T0 = E2 - E1, T1 = E3 - E2, T2 = E4 - E3, T3 = E5 - E4;
  constexpr double cS = 39.0, cT = 781.0 / 20.0, eps36 = 36.0e-6;
  const double s0 = fma(A0, A0, fma(cS * S0, S0, fma(cT * T0, T0, eps36)));   // 36 (eps + beta_k)
  const double s1 = fma(A1, A1, fma(cS * E3, E3, fma(cT * T1, T1, eps36)));
  const double s2 = fma(A2, A2, fma(cS * E3, E3, fma(cT * T2, T2, eps36)));
  const double s3 = fma(A3, A3, fma(cS * S3, S3, fma(cT * T3, T3, eps36)));
  const double t0 = s0 * s0, t1 = s1 * s1, t2 = s2 * s2, t3 = s3 * s3;
  const double t01 = t0 * t1, t23 = t2 * t3;
  const double w0 = t1 * t23, w1 = 12.0 * (t0 * t23), w2 = 18.0 * (t01 * t3), w3 = 4.0 * (t01 * t2);
  const double c0 = fma(13.0, D3, fma(-10.0, D2, 3.0 * D1));
  const double c1 = fma(4.0, D3, fma(3.0, D4, -D2));
  const double c2 = fma(6.0, D4, D3 - D5);
  const double c3 = fma(9.0, D4, fma(-4.0, D5, D6));
  const double num = fma(w0, c0, fma(w1, c1, fma(w2, c2, w3 * c3)));
  const double den = 12.0 * ((w0 + w1) + (w2 + w3));
  return fma(num, xf_rcp(den), v3);
}

// stencil cells of a face: i-2..i+3, or i-3..i+4 for WENO7; the face lies between m = S/2 - 1 and m = S/2
__host__ __device__ constexpr int stencil_cells(int recon) { return recon == 2 ? 8 : 6; }

// g = R(f+ at i-2..) + R(f- mirrored)  (Eq. 15); RECON: 0 WENO5-JS (five points each), 1 WENO-CU6 (all six),
// 2 WENO7 (seven of the eight), 3 WENO5-JS in the relative-accuracy form (positivity limiter on)
template <int RECON>
__device__ __forceinline__ double weno_pair(const double (&fp)[stencil_cells(RECON)], const double (&fm)[stencil_cells(RECON)]) {
  if constexpr (RECON == 2) {
    return weno7(fp[0], fp[1], fp[2], fp[3], fp[4], fp[5], fp[6]) + weno7(fm[7], fm[6], fm[5], fm[4], fm[3], fm[2], fm[1]);
  } else if constexpr (RECON == 1) {
    return wenocu6(fp[0], fp[1], fp[2], fp[3], fp[4], fp[5]) + wenocu6(fm[5], fm[4], fm[3], fm[2], fm[1], fm[0]);
  } else if constexpr (RECON == 3) {
    return weno5_rel(fp[0], fp[1], fp[2], fp[3], fp[4]) + weno5_rel(fm[5], fm[4], fm[3], fm[2], fm[1]);
  } else {
    return weno5(fp[0], fp[1], fp[2], fp[3], fp[4]) + weno5(fm[5], fm[4], fm[3], fm[2], fm[1]);
  }
}

template <int DIR> struct Axes;
template <> struct Axes<0> { static constexpr int nd = 0, t1 = 1, t2 = 2; };
template <> struct Axes<1> { static constexpr int nd = 1, t1 = 0, t2 = 2; };
template <> struct Axes<2> { static constexpr int nd = 2, t1 = 1, t2 = 0; };

// Staged cell fields, in this order: the Nv conserved variables, then the N + 4 fields the primitives kernel leaves
// in the workspace: p, c, 1/rho, Gamma, chi_1..chi_N.
__host__ __device__ constexpr int nstaged(int N) { return 2 * N + 8; }
__host__ __device__ constexpr int nprimfields(int N) { return N + 4; }

// Numerical flux at one face.  sm: staged fields, field f of stencil cell m at sm[f*FS + o[m]] (m = 0..S-1 <-> i-S/2+1..i+S/2,
// S = 6 or, for WENO7, 8; the face lies between m = S/2 - 1 and m = S/2).  emit(v, Fhat_v, vnext) is called once per component, in the order
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
                                          const int (&o)[stencil_cells(RECON)], const double *ss, const int SS, const int s2,
                                          const int s3, const int visc, const double *__restrict__ lamg, Emit &emit) {
  constexpr int nd = Axes<DIR>::nd, t1 = Axes<DIR>::t1, t2 = Axes<DIR>::t2;
  constexpr int S = stencil_cells(RECON), MA = S / 2 - 1, MB = S / 2;   // cells below / above the face

#define XS(f, m) sm[(f) * FS + o[m]]
#define XP(m) sp[o[m]]
#define XC(m) sp[FS + o[m]]
#define XRI(m) sp[2 * FS + o[m]]
#define XA(g) ss[(g) * SS + s2]
#define XB(g) ss[(g) * SS + s3]

  // ---- Roe-type average (reading R5): q~ = (w_a q_a + w_b q_b)/(w_a + w_b), w = sqrt(rho); with
  //      r = w_b/w_a = sqrt(rho_b/rho_a) the weights are 1/(1+r) and r/(1+r)
  const double ria = XRI(MA), rib = XRI(MB);
  const double r = sqrt(XS(0, MB) * ria);
  const double oa = xf_rcp(1.0 + r), ob = r * oa;
  const double oma = oa * ria, omb = ob * rib;                // weights acting on conserved quantities
  double ut[3];
#pragma unroll
  for (int q = 0; q < 3; ++q) ut[q] = fma(oma, XS(1 + q, MA), omb * XS(1 + q, MB));
  const double Ht = fma(oma, XS(4, MA) + XP(MA), omb * (XS(4, MB) + XP(MB)));
  const double Gt = fma(oa, XA(0), ob * XB(0));
  const double kt = 0.5 * fma(ut[0], ut[0], fma(ut[1], ut[1], ut[2] * ut[2]));
  const double chiN = fma(oa, XA(N), ob * XB(N));

  // ---- the dense functional pi.U_m for the six stencil cells; species part first
  double rho[S], piU[S];
#pragma unroll
  for (int m = 0; m < S; ++m) {
    rho[m] = XS(0, m);
    piU[m] = 0.0;
  }
  double c2acc = 0.0;
#pragma unroll 3
  for (int i = 0; i < N - 1; ++i) {
    const double zeta = fma(oa, XA(1 + i), ob * XB(1 + i)) - chiN;
    double y[S];
#pragma unroll
    for (int m = 0; m < S; ++m) y[m] = XS(5 + i, m);
    const double Yt = fma(oma, y[MA], omb * y[MB]);
    c2acc = fma(Yt, zeta, c2acc);
#pragma unroll
    for (int m = 0; m < S; ++m) piU[m] = fma(zeta, y[m], piU[m]);
  }
  // c~^2 = sum_s Y~_s chi~_s + Gamma~ (H~ - k~), with Y~_N = 1 - sum_{i<N} Y~_i
  const double c2 = chiN + c2acc + Gt * (Ht - kt);
  const double ct = sqrt(c2);
  const double h = 0.5 * xf_rcp(c2);  // 1/(2 c~^2)
  const double Prho = fma(Gt, kt, chiN);

  const double hh = 0.5 * h, ghh = Gt * hh, chh = ct * hh;
  double nuU[S], ud[S], qp[S], rp[S];
  double lam_m = 0.0, lam_0 = 0.0, lam_p = 0.0;  // LLF: max over the stencil of |u-c|, |u|, |u+c| (reading R8)
#pragma unroll
  for (int m = 0; m < S; ++m) {
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

  double hud[S];
#pragma unroll
  for (int m = 0; m < S; ++m) hud[m] = 0.5 * ud[m];
  const double hlm = 0.5 * lam_m, hl0 = 0.5 * lam_0, hlp = 0.5 * lam_p;

  // ---- acoustic (u-c), entropy (u) and acoustic (u+c) fields
  double g0, g1, gL;
  {
    double fp[S], fm[S];
#pragma unroll
    for (int m = 0; m < S; ++m) {
      const double a = h * fma(-ct, nuU[m], piU[m]);
      const double pt = qp[m] - rp[m];
      fp[m] = fma(hud[m] + hlm, a, pt);   // (u_m + Lambda)/2: halving is exact, so the halves are formed once
      fm[m] = fma(hud[m] - hlm, a, pt);
    }
    g0 = weno_pair<RECON>(fp, fm);
#pragma unroll
    for (int m = 0; m < S; ++m) {
      const double a = h * fma(ct, nuU[m], piU[m]);
      const double pt = qp[m] + rp[m];
      fp[m] = fma(hud[m] + hlp, a, pt);
      fm[m] = fma(hud[m] - hlp, a, pt);
    }
    gL = weno_pair<RECON>(fp, fm);
  }
  double ap[S], am[S];  // (u_m +- Lambda_u)/2 for all fields that travel with u
#pragma unroll
  for (int m = 0; m < S; ++m) {
    ap[m] = hud[m] + hl0;
    am[m] = hud[m] - hl0;
  }
  {
    double fp[S], fm[S];
#pragma unroll
    for (int m = 0; m < S; ++m) {
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
#define XF_LOAD_FIELD(VIDX, V) _Pragma("unroll") for (int m = 0; m < S; ++m) V[m] = XS(VIDX, m);
#define XF_LINEAR_FIELD(VIDX, V, DEXPR, VNEXT)                                                         \
  {                                                                                                    \
    double fp[S], fm[S];                                                                               \
    const double C = fma(oma, V[MA], omb * V[MB]);                                                     \
    _Pragma("unroll") for (int m = 0; m < S; ++m) {                                                    \
      const double a = fma(-C, rho[m], V[m]);                                                          \
      fp[m] = ap[m] * a;                                                                               \
      fm[m] = am[m] * a;                                                                               \
    }                                                                                                  \
    const double g = weno_pair<RECON>(fp, fm);                                                         \
    F4 = fma((DEXPR), g, F4);                                                                          \
    emit(VIDX, fma(C, s, g), VNEXT);                                                                   \
  }
  {
    double Va[S], Vb[S];
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
      double V[S];
      _Pragma("unroll") for (int m = 0; m < S; ++m) V[m] = Va[m];
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

// ---------------------------------------------------------------------------------------------------------------
// Positivity-preserving flux blending (Eq. 17-20; theta: DESIGN.md reading R17) of one face flux
// that already sits in memory as F[v * stride] (the flux buffer of the sweep, written by this same lane).
// Cells a, b next to the face at staged offsets oa, ob.  Guarded quantities q in {rho, rho Y_1..rho Y_{N-1}, rho Y_N by
// closure}, all linear in U, so q(F) is the same functional of a flux.  With kappa = 2 D dt/dx_d (Eq. 18 split over D
// directions):  q+ = q(U_a) - kappa q(F), q- = q(U_b) + kappa q(F), the same with the first-order Lax-Friedrichs flux
// F^LF = (F_a + F_b + Lambda~ (U_a - U_b))/2 (Eq. 19), Lambda~ = max(|u_d| + c) of the two cells; floor eps =
// min(1e-13, q^LF); theta = min over q and sides of (q^LF - eps)/(q^LF - q) where q < eps; F* = (1 - theta) F^LF +
// theta F (Eq. 20), one factor for the whole vector.  theta = 1 almost everywhere: the flux is then left untouched
// (bit-identical residual) and only the N + 1 guards are paid for.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double pp_kappa(const XfEpilogue &E, const XfGrid &G, const int dir) {
  const double dt = E.pp_S ? E.pp_cfl / *E.pp_S : E.pp_dt;
  const int D = (G.n[0] > 1) + (G.n[1] > 1) + (G.n[2] > 1);
  return 2.0 * D * dt * G.inv_d[dir];
}

template <int DIR>
__device__ __noinline__ void positivity_blend(const int N, const double *sm, const double *sp, const int FS,
                                              const int oa, const int ob, const double kappa, double *F,
                                              const int stride) {
  constexpr int nd = Axes<DIR>::nd;
  const int Nv = N + 4;
  const double ua = sm[(1 + nd) * FS + oa] * sp[2 * FS + oa], ub = sm[(1 + nd) * FS + ob] * sp[2 * FS + ob];
  const double la = fabs(ua) + sp[FS + oa], lb = fabs(ub) + sp[FS + ob];
  const double Lam = la > lb ? la : lb;
  double theta = 1.0;
  auto lf = [&](double qa, double qb) { return 0.5 * (fma(qa, ua, qb * ub) + Lam * (qa - qb)); };
  auto guard = [&](double qa, double qb, double qF, double qL) {
    const double qp = fma(-kappa, qF, qa), qpL = fma(-kappa, qL, qa);   // Eq. 18: U+ of cell a
    const double qm = fma(kappa, qF, qb), qmL = fma(kappa, qL, qb);     //         U- of cell b
    const double ep = fmin(1e-13, qpL), em = fmin(1e-13, qmL);
    if (qp < ep) theta = fmin(theta, (qpL - ep) / (qpL - qp));
    if (qm < em) theta = fmin(theta, (qmL - em) / (qmL - qm));
  };
  double sa = sm[oa], sb = sm[ob], sF = F[0];
  double sL = lf(sa, sb);
  guard(sa, sb, sF, sL);
  for (int i = 0; i < N - 1; ++i) {
    const double qa = sm[(5 + i) * FS + oa], qb = sm[(5 + i) * FS + ob], qF = F[(5 + i) * stride];
    const double qL = lf(qa, qb);
    guard(qa, qb, qF, qL);
    sa -= qa;   // rho Y_N = rho - sum_{s<N} rho Y_s, of the states and of both fluxes
    sb -= qb;
    sF -= qF;
    sL -= qL;
  }
  if (N > 1) guard(sa, sb, sF, sL);
  if (theta < 1.0) {
    const double pa = sp[oa], pb = sp[ob], omt = 1.0 - theta;
    for (int v = 0; v < Nv; ++v) {
      double qa = sm[v * FS + oa], qb = sm[v * FS + ob];
      double extra = 0.0;                              // pressure terms of the physical flux (Eq. 2)
      if (v == 1 + nd) extra = pa + pb;
      if (v == 4) extra = fma(pa, ua, pb * ub);
      const double FLF = 0.5 * (fma(qa, ua, qb * ub) + extra + Lam * (qa - qb));
      F[v * stride] = fma(omt, FLF, theta * F[v * stride]);
    }
  }
}

}  // namespace xf
