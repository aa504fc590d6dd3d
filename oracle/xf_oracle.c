/*
 * xf_oracle.c -- plain CPU oracle (TEST INFRASTRUCTURE ONLY; see xf_oracle.h for scope, pins and build flags).
 *
 * Layout: SoA, U[v][k][j][i], i fastest; v = 0: rho, 1..3: rho u, rho v, rho w, 4: E, 5..Nv-1: rho Y_1..rho Y_{N-1}
 * (Eq. 2, "s = 1..N-1"; reading R1).  A direction with one interior cell carries no ghosts.
 */
#include "xf_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------------------------ */
/* grid helpers                                                                                                 */
/* ------------------------------------------------------------------------------------------------------------ */
int xo_nv(const xo_config *c) { return c->N + 4; }

void xo_padded_dims(const xo_config *c, int *nxp, int *nyp, int *nzp) {
  *nxp = c->nx > 1 ? c->nx + 2 * c->ng : 1;
  *nyp = c->ny > 1 ? c->ny + 2 * c->ng : 1;
  *nzp = c->nz > 1 ? c->nz + 2 * c->ng : 1;
}

long xo_padded_cells(const xo_config *c) {
  int a, b, d;
  xo_padded_dims(c, &a, &b, &d);
  return (long)a * b * d;
}

static void grid(const xo_config *c, int np[3], int n[3], int g[3], long stride[3]) {
  xo_padded_dims(c, &np[0], &np[1], &np[2]);
  n[0] = c->nx; n[1] = c->ny; n[2] = c->nz;
  for (int d = 0; d < 3; ++d) g[d] = n[d] > 1 ? c->ng : 0;
  stride[0] = 1; stride[1] = np[0]; stride[2] = (long)np[0] * np[1];
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C1. Thermodynamics (Eq. 7; Eq. 21; NASA polynomials PAPER.md:153)            */
/*     T_c = min(max(T, Tlo), Thi); outside the fit range cp is frozen and h continues linearly (reading R3).   */
/* ------------------------------------------------------------------------------------------------------------ */
void xo_species_thermo(const xo_config *c, int s, double T, double *cp, double *h, double *e) {
  const double *a = c->a[s];
  const double Rs = c->Ru / c->W[s];
  double Tc = T;
  if (Tc < c->Tlo) Tc = c->Tlo;
  if (Tc > c->Thi) Tc = c->Thi;
  const double cpR = a[0] + Tc * (a[1] + Tc * (a[2] + Tc * (a[3] + Tc * a[4])));
  const double hR = Tc * (a[0] + Tc * (a[1] / 2.0 + Tc * (a[2] / 3.0 + Tc * (a[3] / 4.0 + Tc * (a[4] / 5.0))))) + a[5];
  *cp = Rs * cpR;
  *h = Rs * hR + (*cp) * (T - Tc);
  *e = *h - Rs * T;
}

/* mixture: Rbar = sum Y_s R_s (Eq. 7); e(T) = sum Y_s e_s(T); Cv = sum Y_s cp_s - Rbar (Eq. 21); s ascending */
void xo_mixture(const xo_config *c, const double *Y, double T, double *Rbar, double *e, double *Cv) {
  double R = 0.0, em = 0.0, cpm = 0.0;
  for (int s = 0; s < c->N; ++s) {
    double cp, h, es;
    xo_species_thermo(c, s, T, &cp, &h, &es);
    R += Y[s] * (c->Ru / c->W[s]);
    em += Y[s] * es;
    cpm += Y[s] * cp;
  }
  *Rbar = R;
  *e = em;
  *Cv = cpm - R;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C2. Primitive recovery.  Newton: T^{k+1} = T^k + (e - e(T^k))/Cv(T^k)  (Eq. 21)           */
/* ------------------------------------------------------------------------------------------------------------ */
static void cell_basic(const xo_config *c, const double *Ucell, xo_prim *P) {
  const int N = c->N;
  P->rho = Ucell[0];
  for (int d = 0; d < 3; ++d) P->vel[d] = Ucell[1 + d] / P->rho;
  double sumY = 0.0;
  for (int i = 0; i < N - 1; ++i) {
    P->Y[i] = Ucell[5 + i] / P->rho;
    sumY += P->Y[i];
  }
  P->Y[N - 1] = 1.0 - sumY; /* closure, no clipping, no renormalisation (reading R12) */
  P->e = Ucell[4] / P->rho - 0.5 * (P->vel[0] * P->vel[0] + P->vel[1] * P->vel[1] + P->vel[2] * P->vel[2]);
}

/* everything that follows from a given temperature */
static void cell_from_T(const xo_config *c, const double *Ucell, double T, xo_prim *P) {
  const int N = c->N;
  double Rbar, em, Cv;
  xo_mixture(c, P->Y, T, &Rbar, &em, &Cv);
  P->T = T;
  P->Rbar = Rbar;
  P->Cv = Cv;
  P->p = P->rho * Rbar * T;              /* Eq. 7 */
  P->Gamma = Rbar / Cv;                  /* Gamma = (dp/de)_rho / rho = gamma - 1 */
  P->c = sqrt((1.0 + P->Gamma) * P->p / P->rho);
  P->H = (Ucell[4] + P->p) / P->rho;
  for (int s = 0; s < N; ++s) {
    double cp, h, es;
    xo_species_thermo(c, s, T, &cp, &h, &es);
    P->chi[s] = (c->Ru / c->W[s]) * T - P->Gamma * es;   /* chi_s = (dp/d(rho Y_s)) at fixed rho e */
  }
  if (!(P->rho > 0.0) || !(P->T > 0.0) || !(P->p > 0.0)) P->status |= XO_ENONPHYSICAL;
}

void xo_cell_primitives(const xo_config *c, const double *Ucell, double Tguess, xo_prim *P) {
  memset(P, 0, sizeof(*P));
  cell_basic(c, Ucell, P);
  double T = Tguess;
  int k = 0, converged = 0;
  while (k < c->maxit) {
    double Rbar, eT, Cv;
    xo_mixture(c, P->Y, T, &Rbar, &eT, &Cv);
    const double Tn = T + (P->e - eT) / Cv;
    ++k;
    const double dT = fabs(Tn - T);
    T = Tn;
    if (dT <= c->rtol * fabs(Tn)) { converged = 1; break; }
    if (!(Tn == Tn)) break; /* NaN */
  }
  P->iters = k;
  if (!converged) P->status |= XO_ENOCONV;
  cell_from_T(c, Ucell, T, P);
}

static void gather_cell(const xo_config *c, const double *U, long cells, long idx, double *Ucell) {
  const int Nv = c->N + 4;
  for (int v = 0; v < Nv; ++v) Ucell[v] = U[v * cells + idx];
}

int xo_primitives(const xo_config *c, const double *U, double *T, double *p, double *cs, double *iters_mean) {
  const long cells = xo_padded_cells(c);
  int status = 0;
  double itsum = 0.0;
#pragma omp parallel for reduction(| : status) reduction(+ : itsum) schedule(static) if (cells > 16384)
  for (long idx = 0; idx < cells; ++idx) {
    double Uc[XO_MAXNV];
    xo_prim P;
    gather_cell(c, U, cells, idx, Uc);
    xo_cell_primitives(c, Uc, T[idx], &P);
    T[idx] = P.T;
    if (p) p[idx] = P.p;
    if (cs) cs[idx] = P.c;
    status |= P.status;
    itsum += P.iters;
  }
  if (iters_mean) *iters_mean = itsum / (double)cells;
  return status;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C3. Physical flux in direction d (Eq. 2)                                                         */
/* ------------------------------------------------------------------------------------------------------------ */
void xo_phys_flux(const xo_config *c, const double *Uc, const xo_prim *P, int d, double *F) {
  const int Nv = c->N + 4;
  const double ud = P->vel[d];
  F[0] = Uc[0] * ud;
  for (int q = 0; q < 3; ++q) F[1 + q] = Uc[1 + q] * ud + (q == d ? P->p : 0.0);
  F[4] = (Uc[4] + P->p) * ud;
  for (int v = 5; v < Nv; ++v) F[v] = Uc[v] * ud;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C4. Dense face eigensystem (Lambda = L A R with the Roe-averaged Jacobian, refs 32/33/37;    */
/*     the matrices are not printed in the paper -> readings R5, R6)                                            */
/* ------------------------------------------------------------------------------------------------------------ */
static void tangentials(int d, int *t1, int *t2) {
  /* x: (v, w); y: roles of (u, index 1) and (v, index 2) swapped -> (u, w); z: u <-> w swapped -> (v, u) */
  if (d == 0) { *t1 = 1; *t2 = 2; }
  else if (d == 1) { *t1 = 0; *t2 = 2; }
  else { *t1 = 1; *t2 = 0; }
}

int xo_eigensystem(const xo_config *c, const xo_prim *A, const xo_prim *B, int d, double *L, double *R, double *roe) {
  const int N = c->N, Nv = N + 4;
  int status = 0;
  /* Roe-type average (reading R5): q~ = (w_a q_a + w_b q_b)/(w_a + w_b), w = sqrt(rho) */
  const double wa = sqrt(A->rho), wb = sqrt(B->rho);
#define AVG(qa, qb) ((wa * (qa) + wb * (qb)) / (wa + wb))
  double vt[3], Yt[XO_MAXN], chit[XO_MAXN];
  for (int q = 0; q < 3; ++q) vt[q] = AVG(A->vel[q], B->vel[q]);
  const double Ht = AVG(A->H, B->H);
  const double Gt = AVG(A->Gamma, B->Gamma);
  for (int s = 0; s < N; ++s) {
    Yt[s] = AVG(A->Y[s], B->Y[s]);
    chit[s] = AVG(A->chi[s], B->chi[s]);
  }
#undef AVG
  const double kt = 0.5 * (vt[0] * vt[0] + vt[1] * vt[1] + vt[2] * vt[2]);
  double c2 = 0.0;
  for (int s = 0; s < N; ++s) c2 += Yt[s] * chit[s];
  c2 += Gt * (Ht - kt);
  if (!(c2 > 0.0)) status |= XO_ENONPHYSICAL;
  const double ct = sqrt(c2);
  double zeta[XO_MAXN];
  for (int i = 0; i < N - 1; ++i) zeta[i] = chit[i] - chit[N - 1];
  const double Prho = chit[N - 1] + Gt * kt;

  double pi[XO_MAXNV], nu[XO_MAXNV], b[XO_MAXNV];
  memset(nu, 0, sizeof(nu));
  pi[0] = Prho;
  for (int q = 0; q < 3; ++q) pi[1 + q] = -Gt * vt[q];
  pi[4] = Gt;
  for (int i = 0; i < N - 1; ++i) pi[5 + i] = zeta[i];
  nu[0] = -vt[d];
  nu[1 + d] = 1.0;
  b[0] = 1.0;
  for (int q = 0; q < 3; ++q) b[1 + q] = vt[q];
  b[4] = Ht;
  for (int i = 0; i < N - 1; ++i) b[5 + i] = Yt[i];

  int t1, t2;
  tangentials(d, &t1, &t2);
  memset(L, 0, sizeof(double) * Nv * Nv);
  memset(R, 0, sizeof(double) * Nv * Nv);
#define LL(n, j) L[(n) * Nv + (j)]
#define RR(j, n) R[(j) * Nv + (n)]
  for (int j = 0; j < Nv; ++j) {
    LL(0, j) = (pi[j] - ct * nu[j]) / (2.0 * c2);
    LL(Nv - 1, j) = (pi[j] + ct * nu[j]) / (2.0 * c2);
    LL(1, j) = (j == 0 ? 1.0 : 0.0) - pi[j] / c2;
    RR(j, 0) = b[j];
    RR(j, 1) = b[j];
    RR(j, Nv - 1) = b[j];
  }
  RR(1 + d, 0) -= ct;
  RR(4, 0) -= vt[d] * ct;
  RR(1 + d, Nv - 1) += ct;
  RR(4, Nv - 1) += vt[d] * ct;
  RR(4, 1) = Ht - c2 / Gt;
  LL(2, 0) = -vt[t1]; LL(2, 1 + t1) = 1.0;
  LL(3, 0) = -vt[t2]; LL(3, 1 + t2) = 1.0;
  RR(1 + t1, 2) = 1.0; RR(4, 2) = vt[t1];
  RR(1 + t2, 3) = 1.0; RR(4, 3) = vt[t2];
  for (int i = 0; i < N - 1; ++i) {
    LL(4 + i, 0) = -Yt[i];
    LL(4 + i, 5 + i) = 1.0;
    RR(5 + i, 4 + i) = 1.0;
    RR(4, 4 + i) = -zeta[i] / Gt;
  }
#undef LL
#undef RR
  if (roe) { /* exposed for the pins: u~ v~ w~ H~ Gamma~ c~ */
    roe[0] = vt[0]; roe[1] = vt[1]; roe[2] = vt[2]; roe[3] = Ht; roe[4] = Gt; roe[5] = ct;
  }
  return status;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C6. WENO5-JS (ref 35; eps = 1e-6, exponent 2, linear weights 0.1 0.6 0.3: reading R7)          */
/* ------------------------------------------------------------------------------------------------------------ */
double xo_weno5(const double v[5], int ideal_weights) {
  const double q0 = (2.0 * v[0] - 7.0 * v[1] + 11.0 * v[2]) / 6.0;
  const double q1 = (-v[1] + 5.0 * v[2] + 2.0 * v[3]) / 6.0;
  const double q2 = (2.0 * v[2] + 5.0 * v[3] - v[4]) / 6.0;
  double a0, a1, a2;
  if (ideal_weights) {
    a0 = 0.1; a1 = 0.6; a2 = 0.3;
  } else {
    const double eps = 1e-6;
    const double t0 = v[0] - 2.0 * v[1] + v[2], s0 = v[0] - 4.0 * v[1] + 3.0 * v[2];
    const double t1 = v[1] - 2.0 * v[2] + v[3], s1 = v[1] - v[3];
    const double t2 = v[2] - 2.0 * v[3] + v[4], s2 = 3.0 * v[2] - 4.0 * v[3] + v[4];
    const double b0 = 13.0 / 12.0 * t0 * t0 + 0.25 * s0 * s0;
    const double b1 = 13.0 / 12.0 * t1 * t1 + 0.25 * s1 * s1;
    const double b2 = 13.0 / 12.0 * t2 * t2 + 0.25 * s2 * s2;
    a0 = 0.1 / ((eps + b0) * (eps + b0));
    a1 = 0.6 / ((eps + b1) * (eps + b1));
    a2 = 0.3 / ((eps + b2) * (eps + b2));
  }
  return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C6'. WENO-CU6 (PAPER.md:107 names it, ref 34, and prints no formula: reading R16).  Six-point stencil v_{-2}..v_{+3};   */
/* candidates q_0..q_2 as in WENO5 plus the downwind q_3; linear weights 1/20, 9/20, 9/20, 1/20 (the sixth-order        */
/* central scheme); beta_0..beta_2 as Jiang-Shu; the fourth indicator is beta_6, the Jiang-Shu measure                 */
/*   sum_{l=1..5} dx^(2l-1) int (d^l p/dx^l)^2 dx  of the degree-5 polynomial over all six cells (its quadratic form,  */
/* over 120960, is derived exactly in tests/golden/make_golden.py and pinned against quadrature in the tests);          */
/* tau_6 = beta_6 - (beta_0 + 4 beta_1 + beta_2)/6;  alpha_k = d_k (C + tau_6/(beta_k + eps)), C = 20, eps = 1e-40.    */
/* ------------------------------------------------------------------------------------------------------------ */
double xo_wenocu6(const double v[6], int ideal_weights, double *beta_out, double *w_out) {
  static const double d[4] = {1.0 / 20.0, 9.0 / 20.0, 9.0 / 20.0, 1.0 / 20.0};
  /* beta_6 * 120960 as a quadratic form of the five first differences D_k = v_{k+1} - v_k (the measure is translation
   * invariant; in terms of the values themselves the form has coefficients up to 3.6e7 that cancel to round-off on
   * smooth data).  Entry [k][l], l >= k, multiplies D_k D_l; obtained from the value form of
   * tests/golden/wenocu6_beta6_form.txt by v_j = v_0 + sum_{k<j} D_k. */
  static const double G6[5][5] = {
      {271779.0, -1837242.0, 2249110.0, -1213142.0, 245620.0},
      {0.0, 3544296.0, -9252940.0, 5189840.0, -1079386.0},
      {0.0, 0.0, 6713736.0, -7947412.0, 1713274.0},
      {0.0, 0.0, 0.0, 2534504.0, -1150710.0},
      {0.0, 0.0, 0.0, 0.0, 139633.0}};
  double q[4], a[4], beta[4];
  q[0] = (2.0 * v[0] - 7.0 * v[1] + 11.0 * v[2]) / 6.0;
  q[1] = (-v[1] + 5.0 * v[2] + 2.0 * v[3]) / 6.0;
  q[2] = (2.0 * v[2] + 5.0 * v[3] - v[4]) / 6.0;
  q[3] = (11.0 * v[3] - 7.0 * v[4] + 2.0 * v[5]) / 6.0;
  for (int k = 0; k < 3; ++k) {
    const double t = v[k] - 2.0 * v[k + 1] + v[k + 2];
    const double s = k == 0 ? v[0] - 4.0 * v[1] + 3.0 * v[2] : (k == 1 ? v[1] - v[3] : 3.0 * v[2] - 4.0 * v[3] + v[4]);
    beta[k] = 13.0 / 12.0 * t * t + 0.25 * s * s;
  }
  double D[5], b6 = 0.0;
  for (int k = 0; k < 5; ++k) D[k] = v[k + 1] - v[k];
  for (int k = 0; k < 5; ++k)
    for (int l = k; l < 5; ++l) b6 += G6[k][l] * D[k] * D[l];
  beta[3] = b6 / 120960.0;
  if (ideal_weights) {
    for (int k = 0; k < 4; ++k) a[k] = d[k];
  } else {
    const double tau = beta[3] - (beta[0] + 4.0 * beta[1] + beta[2]) / 6.0;
    for (int k = 0; k < 4; ++k) a[k] = d[k] * (20.0 + tau / (beta[k] + 1e-40));
  }
  const double sum = a[0] + a[1] + a[2] + a[3];
  if (beta_out) for (int k = 0; k < 4; ++k) beta_out[k] = beta[k];
  if (w_out) for (int k = 0; k < 4; ++k) w_out[k] = a[k] / sum;
  return (a[0] * q[0] + a[1] * q[1] + a[2] * q[2] + a[3] * q[3]) / sum;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C6''. WENO7 (PAPER.md:107 names it, ref 36, and prints no formula: reading R18).  Seven-point stencil v_{-3}..v_{+3}; */
/* four cubic candidates on cells (k-3..k), k = 0..3; linear weights 1/35, 12/35, 18/35, 4/35 (together the 7-point     */
/* interpolation (-3, 25, -101, 319, 214, -38, 4)/420); beta_k = sum_{l=1..3} dx^(2l-1) int (d^l p_k/dx^l)^2 dx of the   */
/* candidate polynomial over cell i -- the Jiang-Shu measure; its quadratic form in the three FIRST DIFFERENCES of the   */
/* sub-stencil, times 240, is derived exactly in tests/golden/make_golden.py (weno7_coefficients.txt);                   */
/* alpha_k = d_k/(eps + beta_k)^2 with eps = 1e-6 and exponent 2 as for WENO5 (reading R7).                             */
/* ------------------------------------------------------------------------------------------------------------ */
double xo_weno7(const double v[7], int ideal_weights, double *beta_out, double *w_out) {
  static const double d[4] = {1.0 / 35.0, 12.0 / 35.0, 18.0 / 35.0, 4.0 / 35.0};
  static const double C[4][4] = {{-3.0, 13.0, -23.0, 25.0}, {1.0, -5.0, 13.0, 3.0}, {-1.0, 7.0, 7.0, -1.0}, {3.0, 13.0, -5.0, 1.0}};
  /* 240 beta_k = G[k][0] D0^2 + G[k][1] D0 D1 + G[k][2] D0 D2 + G[k][3] D1^2 + G[k][4] D1 D2 + G[k][5] D2^2,
   * D_m = v_{k+m+1} - v_{k+m} the first differences of sub-stencil k */
  static const double G[4][6] = {{547.0, -2788.0, 1854.0, 3708.0, -5188.0, 2107.0},
                                 {267.0, -1108.0, 494.0, 1468.0, -1428.0, 547.0},
                                 {547.0, -1428.0, 494.0, 1468.0, -1108.0, 267.0},
                                 {2107.0, -5188.0, 1854.0, 3708.0, -2788.0, 547.0}};
  double q[4], a[4], beta[4];
  for (int k = 0; k < 4; ++k) {
    q[k] = (C[k][0] * v[k] + C[k][1] * v[k + 1] + C[k][2] * v[k + 2] + C[k][3] * v[k + 3]) / 12.0;
    const double D0 = v[k + 1] - v[k], D1 = v[k + 2] - v[k + 1], D2 = v[k + 3] - v[k + 2];
    beta[k] = (G[k][0] * D0 * D0 + G[k][1] * D0 * D1 + G[k][2] * D0 * D2 + G[k][3] * D1 * D1 + G[k][4] * D1 * D2 +
               G[k][5] * D2 * D2) / 240.0;
  }
  if (ideal_weights) {
    for (int k = 0; k < 4; ++k) a[k] = d[k];
  } else {
    const double eps = 1e-6;
    for (int k = 0; k < 4; ++k) a[k] = d[k] / ((eps + beta[k]) * (eps + beta[k]));
  }
  const double sum = a[0] + a[1] + a[2] + a[3];
  if (beta_out) for (int k = 0; k < 4; ++k) beta_out[k] = beta[k];
  if (w_out) for (int k = 0; k < 4; ++k) w_out[k] = a[k] / sum;
  return (a[0] * q[0] + a[1] * q[1] + a[2] * q[2] + a[3] * q[3]) / sum;
}

int xo_stencil_cells(const xo_config *c) { return c->recon == XO_RECON_WENO7 ? 8 : 6; }

/* ------------------------------------------------------------------------------------------------------------ */
/* C5 + C6 + C7. Numerical flux at one face (Eq. 14-15; LLF: PAPER.md:374, reading R8)        */
/* Ust[m][v], Pst[m], m = 0..S-1 <-> cells i-S/2+1..i+S/2 (S = 6: i-2..i+3; WENO7, S = 8: i-3..i+4); the face lies      */
/* between m = S/2-1 and m = S/2.                                                                                */
/* ------------------------------------------------------------------------------------------------------------ */
int xo_face_flux(const xo_config *c, int d, const double *Ust, const xo_prim *Pst, double *Fhat) {
  const int Nv = c->N + 4;
  const int S = xo_stencil_cells(c), ma = S / 2 - 1;
  double L[XO_MAXNV * XO_MAXNV], R[XO_MAXNV * XO_MAXNV], roe[6];
  int status = xo_eigensystem(c, &Pst[ma], &Pst[ma + 1], d, L, R, roe);

  double aF[8][XO_MAXNV], aU[8][XO_MAXNV], lam[8][3];
  for (int m = 0; m < S; ++m) {
    double F[XO_MAXNV];
    xo_phys_flux(c, Ust + m * Nv, &Pst[m], d, F);
    for (int n = 0; n < Nv; ++n) {          /* alpha^F_m = L F_m, alpha^U_m = L U_m (face-frozen L) */
      double sF = 0.0, sU = 0.0;
      for (int j = 0; j < Nv; ++j) {
        sF += L[n * Nv + j] * F[j];
        sU += L[n * Nv + j] * Ust[m * Nv + j];
      }
      aF[m][n] = sF;
      aU[m][n] = sU;
    }
    lam[m][0] = Pst[m].vel[d] - Pst[m].c;   /* the cell's own eigenvalues */
    lam[m][1] = Pst[m].vel[d];
    lam[m][2] = Pst[m].vel[d] + Pst[m].c;
  }
  double g[XO_MAXNV];
  for (int n = 0; n < Nv; ++n) {
    const int kind = n == 0 ? 0 : (n == Nv - 1 ? 2 : 1);
    double Lam = 0.0;
    if (c->viscosity == XO_VISC_ROE) {       /* |lambda_n| of the Roe-averaged state: u~_d -+ c~ (roe[5] = c~) */
      Lam = fabs(roe[d] + (kind - 1) * roe[5]);
    } else if (c->viscosity == XO_VISC_GLF) {
      Lam = c->lam_glob[d][kind];            /* global maximum, set by the caller */
    } else {                                 /* LLF: max over the S stencil cells, factor 1 */
      for (int m = 0; m < S; ++m) Lam = fmax(Lam, fabs(lam[m][kind]));
    }
    double fp[8], fm[8];
    for (int m = 0; m < S; ++m) {            /* Eq. 14 */
      fp[m] = 0.5 * (aF[m][n] + Lam * aU[m][n]);
      fm[m] = 0.5 * (aF[m][n] - Lam * aU[m][n]);
    }
    if (c->recon == XO_RECON_WENO7) {        /* seven points each: i-3..i+3 for f+, i+4..i-2 for f- */
      const double vp[7] = {fp[0], fp[1], fp[2], fp[3], fp[4], fp[5], fp[6]};
      const double vm[7] = {fm[7], fm[6], fm[5], fm[4], fm[3], fm[2], fm[1]};
      g[n] = xo_weno7(vp, c->ideal_weights, NULL, NULL) + xo_weno7(vm, c->ideal_weights, NULL, NULL);
    } else if (c->recon == XO_RECON_WENOCU6) {      /* six points: i-2..i+3 for f+, mirrored for f- */
      const double vp[6] = {fp[0], fp[1], fp[2], fp[3], fp[4], fp[5]};
      const double vm[6] = {fm[5], fm[4], fm[3], fm[2], fm[1], fm[0]};
      g[n] = xo_wenocu6(vp, c->ideal_weights, NULL, NULL) + xo_wenocu6(vm, c->ideal_weights, NULL, NULL);
    } else {
      const double vp[5] = {fp[0], fp[1], fp[2], fp[3], fp[4]};
      const double vm[5] = {fm[5], fm[4], fm[3], fm[2], fm[1]};
      g[n] = xo_weno5(vp, c->ideal_weights) + xo_weno5(vm, c->ideal_weights);
    }
  }
  for (int j = 0; j < Nv; ++j) {             /* Eq. 15: Fhat = R (F+ + F-) */
    double s = 0.0;
    for (int n = 0; n < Nv; ++n) s += R[j * Nv + n] * g[n];
    Fhat[j] = s;
  }
  return status;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* Positivity-preserving flux blending (Eq. 17-20).  The paper gives the convex splitting      */
/* U^{n+1}_i = (U^-_i + U^+_i)/2, U^+- = U_i -+ 2 lambda Fhat_{i+-1/2} (Eq. 18), the first-order Lax-Friedrichs  */
/* flux (Eq. 19) and the blend F* = (1 - theta) F^LF + theta Fhat (Eq. 20), and defers theta to its ref 41.     */
/* Reading R17: the guarded quantities are q in {rho, rho Y_1, ..., rho Y_N} ("extended to both the  */
/* density and mass fractions"), rho Y_N = rho - sum_{s<N} rho Y_s; all are linear in U, so q(F)   */
/* is the same functional of a flux.  For the face between cells a = i and b = i+1, with kappa = 2 D dt/dx_d     */
/* (each of the D active directions carries the weight 1/D of the splitting):                                   */
/*   q^+  = q(U_a) - kappa q(Fhat),  q^+LF = q(U_a) - kappa q(F^LF)     (cell a, its upper face)                 */
/*   q^-  = q(U_b) + kappa q(Fhat),  q^-LF = q(U_b) + kappa q(F^LF)     (cell b, its lower face)                 */
/*   eps  = min(1e-13, q^LF);  theta^+- = 1 if q^+- >= eps, else (q^LF - eps)/(q^LF - q^+-)                       */
/*   theta = min over q and over the two sides -- ONE factor for the whole flux vector (Eq. 20).                 */
/* Lambda~ of Eq. 19 = max(|u_d| + c) of the two cells.  Whenever the LF states are non-negative (they are for  */
/* kappa Lambda~ <= 1, i.e. D dt Lambda~/dx_d <= 1/2: "CFL <= 0.5"), the blended states satisfy   */
/* q^+-* >= eps >= 0, and the updated cell value, their average over directions and sides, is non-negative.     */
/* ------------------------------------------------------------------------------------------------------------ */
double xo_positivity_blend(const xo_config *c, int d, const double *Ua, const xo_prim *Pa, const double *Ub,
                           const xo_prim *Pb, double kappa, double *Fhat) {
  const int N = c->N, Nv = N + 4;
  double Fa[XO_MAXNV], Fb[XO_MAXNV], FLF[XO_MAXNV];
  xo_phys_flux(c, Ua, Pa, d, Fa);
  xo_phys_flux(c, Ub, Pb, d, Fb);
  const double Lam = fmax(fabs(Pa->vel[d]) + Pa->c, fabs(Pb->vel[d]) + Pb->c);
  for (int v = 0; v < Nv; ++v) FLF[v] = 0.5 * (Fa[v] + Fb[v] + Lam * (Ua[v] - Ub[v]));   /* Eq. 19 */
  double theta = 1.0;
  for (int k = 0; k <= N; ++k) {             /* k = 0: rho; k = 1..N-1: rho Y_k; k = N: rho Y_N by closure */
    double qa, qb, qF, qL;
    if (k == 0) { qa = Ua[0]; qb = Ub[0]; qF = Fhat[0]; qL = FLF[0]; }
    else if (k < N) { qa = Ua[4 + k]; qb = Ub[4 + k]; qF = Fhat[4 + k]; qL = FLF[4 + k]; }
    else {
      qa = Ua[0]; qb = Ub[0]; qF = Fhat[0]; qL = FLF[0];
      for (int s = 1; s < N; ++s) { qa -= Ua[4 + s]; qb -= Ub[4 + s]; qF -= Fhat[4 + s]; qL -= FLF[4 + s]; }
    }
    const double qp = qa - kappa * qF, qpL = qa - kappa * qL;     /* Eq. 18: U^+ of cell a */
    const double qm = qb + kappa * qF, qmL = qb + kappa * qL;     /*         U^- of cell b */
    const double epsp = fmin(1e-13, qpL), epsm = fmin(1e-13, qmL);
    if (qp < epsp) theta = fmin(theta, (qpL - epsp) / (qpL - qp));
    if (qm < epsm) theta = fmin(theta, (qmL - epsm) / (qmL - qm));
  }
  if (theta < 1.0)
    for (int v = 0; v < Nv; ++v) Fhat[v] = (1.0 - theta) * FLF[v] + theta * Fhat[v];     /* Eq. 20 */
  return theta;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C8. Ghost fill ("specific boundary conditions", 433; formulas: reading R10), x then y then z    */
/* ------------------------------------------------------------------------------------------------------------ */
void xo_fill_ghosts(const xo_config *c, double *U) {
  const int Nv = c->N + 4;
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  const long cells = xo_padded_cells(c);
  for (int d = 0; d < 3; ++d) {
    if (n[d] == 1) continue;
    /* extent of the two other axes: padded if that direction was already filled, interior otherwise */
    int lo[3], hi[3];
    for (int q = 0; q < 3; ++q) {
      if (q < d) { lo[q] = 0; hi[q] = np[q]; }
      else { lo[q] = g[q]; hi[q] = g[q] + n[q]; }
    }
    const int a1 = (d + 1) % 3, a2 = (d + 2) % 3;
    for (int side = 0; side < 2; ++side) {
      const int bc = c->bc[2 * d + side];
      for (int l = 0; l < g[d]; ++l) {
        const int ighost = side == 0 ? g[d] - 1 - l : g[d] + n[d] + l;
        int isrc = ighost;
        if (bc == XO_BC_PERIODIC) isrc = side == 0 ? ighost + n[d] : ighost - n[d];
        else if (bc == XO_BC_TRANSMISSIVE) isrc = side == 0 ? g[d] : g[d] + n[d] - 1;
        else if (bc == XO_BC_REFLECTIVE) isrc = side == 0 ? g[d] + l : g[d] + n[d] - 1 - l;
        for (int p = lo[a1]; p < hi[a1]; ++p)
          for (int q = lo[a2]; q < hi[a2]; ++q) {
            const long base = (long)p * st[a1] + (long)q * st[a2];
            const long ig = base + (long)ighost * st[d], is = base + (long)isrc * st[d];
            for (int v = 0; v < Nv; ++v) {
              double val;
              if (bc == XO_BC_DIRICHLET) val = c->bc_state[2 * d + side][v];
              else {
                val = U[v * cells + is];
                if (bc == XO_BC_REFLECTIVE && v == 1 + d) val = -val; /* wall-normal momentum negated */
              }
              U[v * cells + ig] = val;
            }
          }
      }
    }
  }
}

/* ------------------------------------------------------------------------------------------------------------ */
/* C7. rhs = - sum_d (Fhat_{i+1/2} - Fhat_{i-1/2})/dx_d  (Eq. 13; faces per PAPER.md:271-273)       */
/* ------------------------------------------------------------------------------------------------------------ */
static void pencil_prims(const xo_config *c, const double *U, const double *T, long cells, long base, long stride,
                         int count, double *Ust, xo_prim *Pst) {
  const int Nv = c->N + 4;
  for (int m = 0; m < count; ++m) {
    const long idx = base + m * stride;
    gather_cell(c, U, cells, idx, Ust + m * Nv);
    memset(&Pst[m], 0, sizeof(xo_prim));
    cell_basic(c, Ust + m * Nv, &Pst[m]);
    cell_from_T(c, Ust + m * Nv, T[idx], &Pst[m]);
  }
}

/* U must have its ghosts filled; T: in guess, out converged temperature (whole padded field) */
/* GLF: max over all padded cells (ghosts filled) of |u_d - c|, |u_d|, |u_d + c| per direction, from each cell's own
 * primitives at the T guess given */
static void global_wavespeeds(const xo_config *c, const double *U, const double *T, double lam[3][3]) {
  const long cells = xo_padded_cells(c);
  const int Nv = c->N + 4;
  for (int d = 0; d < 3; ++d)
    for (int k = 0; k < 3; ++k) lam[d][k] = 0.0;
  for (long id = 0; id < cells; ++id) {
    double Uc[XO_MAXNV];
    xo_prim P;
    for (int v = 0; v < Nv; ++v) Uc[v] = U[(long)v * cells + id];
    xo_cell_primitives(c, Uc, T[id], &P);
    for (int d = 0; d < 3; ++d) {
      lam[d][0] = fmax(lam[d][0], fabs(P.vel[d] - P.c));
      lam[d][1] = fmax(lam[d][1], fabs(P.vel[d]));
      lam[d][2] = fmax(lam[d][2], fabs(P.vel[d] + P.c));
    }
  }
}

int xo_rhs_nofill(const xo_config *c_in, const double *U, double *T, double *rhs) {
  xo_config cc = *c_in;
  const xo_config *c = &cc;
  const int Nv = c->N + 4;
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  const long cells = xo_padded_cells(c);
  int status = xo_primitives(c, U, T, NULL, NULL, NULL);   /* "after updating the primitive variables" PAPER.md:411 */
  if (c->viscosity == XO_VISC_GLF) global_wavespeeds(c, U, T, cc.lam_glob);
  memset(rhs, 0, sizeof(double) * Nv * cells);
  const double dxs[3] = {c->dx, c->dy, c->dz};
  const int ma = xo_stencil_cells(c) / 2 - 1;                /* stencil cell index of the cell below the face */
  const int D = (n[0] > 1) + (n[1] > 1) + (n[2] > 1);
  const double kappa[3] = {2.0 * D * c->pp_dt / c->dx, 2.0 * D * c->pp_dt / c->dy, 2.0 * D * c->pp_dt / c->dz};
  for (int d = 0; d < 3; ++d) {
    if (n[d] == 1) continue;
    const int a1 = (d + 1) % 3, a2 = (d + 2) % 3;
    const long npen = (long)n[a1] * n[a2];
    const int len = np[d];
#pragma omp parallel reduction(| : status) if (npen > 16)
    {
      double *Ust = (double *)malloc(sizeof(double) * len * Nv);
      xo_prim *Pst = (xo_prim *)malloc(sizeof(xo_prim) * len);
      double *Fh = (double *)malloc(sizeof(double) * (n[d] + 1) * Nv);
#pragma omp for schedule(dynamic, 4)
      for (long pen = 0; pen < npen; ++pen) {
        const int p = g[a1] + (int)(pen / n[a2]), q = g[a2] + (int)(pen % n[a2]);
        const long base = (long)p * st[a1] + (long)q * st[a2];
        pencil_prims(c, U, T, cells, base, st[d], len, Ust, Pst);
        /* faces i = g-1 .. g+n-1 (face i+1/2 between cells i and i+1): n+1 faces */
        for (int f = 0; f <= n[d]; ++f) {
          const int i = g[d] - 1 + f;
          status |= xo_face_flux(c, d, Ust + (i - ma) * Nv, Pst + (i - ma), Fh + f * Nv);
          if (c->positivity)                 /* Eq. 20: "the blended flux is used to update Eq. (13)" */
            xo_positivity_blend(c, d, Ust + i * Nv, Pst + i, Ust + (i + 1) * Nv, Pst + (i + 1), kappa[d], Fh + f * Nv);
        }
        for (int f = 0; f < n[d]; ++f) {
          const long idx = base + (long)(g[d] + f) * st[d];
          for (int v = 0; v < Nv; ++v) rhs[v * cells + idx] -= (Fh[(f + 1) * Nv + v] - Fh[f * Nv + v]) / dxs[d];
        }
      }
      free(Ust); free(Pst); free(Fh);
    }
  }
  return status;
}

int xo_rhs(const xo_config *c, double *U, double *T, double *rhs) {
  xo_fill_ghosts(c, U);                /* "with specific boundary conditions" before each residual: R11 */
  return xo_rhs_nofill(c, U, T, rhs);
}

/* rhs at a list of sampled interior cells, each computed on its own from U (ghosts filled) and the T guess:
 * primitives by Newton for the (S+1)-cell cross of every direction (S = 6 or 8 stencil cells), two faces per direction.
 * Used for parity at sizes where the whole-field oracle would take too long. rhs_out[q][v]. */
int xo_rhs_cells(const xo_config *c_in, const double *U, const double *Tguess, long ncells, const long *idx,
                 double *rhs_out) {
  xo_config cc = *c_in;
  const xo_config *c = &cc;
  if (c->viscosity == XO_VISC_GLF) global_wavespeeds(c, U, Tguess, cc.lam_glob);
  const int Nv = c->N + 4;
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  const long cells = xo_padded_cells(c);
  const double dxs[3] = {c->dx, c->dy, c->dz};
  const int S = xo_stencil_cells(c), h = S / 2;              /* cells i-h .. i+h */
  const int D = (n[0] > 1) + (n[1] > 1) + (n[2] > 1);
  int status = 0;
#pragma omp parallel for reduction(| : status) schedule(dynamic, 8) if (ncells > 64)
  for (long q = 0; q < ncells; ++q) {
    double acc[XO_MAXNV];
    for (int v = 0; v < Nv; ++v) acc[v] = 0.0;
    for (int d = 0; d < 3; ++d) {
      if (n[d] == 1) continue;
      double Ust[9 * XO_MAXNV];
      xo_prim Pst[9];
      for (int m = 0; m <= 2 * h; ++m) {
        const long id = idx[q] + (long)(m - h) * st[d];
        gather_cell(c, U, cells, id, Ust + m * Nv);
        xo_cell_primitives(c, Ust + m * Nv, Tguess[id], &Pst[m]);
        status |= Pst[m].status;
      }
      double Fl[XO_MAXNV], Fr[XO_MAXNV];
      status |= xo_face_flux(c, d, Ust, Pst, Fl);            /* face i-1/2: cells i-h..i+h-1 */
      status |= xo_face_flux(c, d, Ust + Nv, Pst + 1, Fr);   /* face i+1/2: cells i-h+1..i+h */
      if (c->positivity) {
        const double kappa = 2.0 * D * c->pp_dt / dxs[d];
        xo_positivity_blend(c, d, Ust + (h - 1) * Nv, Pst + h - 1, Ust + h * Nv, Pst + h, kappa, Fl);
        xo_positivity_blend(c, d, Ust + h * Nv, Pst + h, Ust + (h + 1) * Nv, Pst + h + 1, kappa, Fr);
      }
      for (int v = 0; v < Nv; ++v) acc[v] -= (Fr[v] - Fl[v]) / dxs[d];
    }
    for (int v = 0; v < Nv; ++v) rhs_out[q * Nv + v] = acc[v];
  }
  return status;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* SSP-RK3 (Eq. 16); ghosts + primitives before each of the three residuals     */
/* ------------------------------------------------------------------------------------------------------------ */
/* ------------------------------------------------------------------------------------------------------------ */
/* Viscous / diffusive right-hand side (Eq. 1-6; 155-178 Eq. 22, 26; 505-513 Eq. 29; readings R19-R23) */
/* ------------------------------------------------------------------------------------------------------------ */
static double fit_eval(const double a[4], double lnT) {           /* Eq. 29: ln eta = sum_n a_n (ln T)^n */
  return exp(a[0] + lnT * (a[1] + lnT * (a[2] + lnT * a[3])));
}

void xo_transport_cell(const xo_config *c, const xo_transport *tr, double rho, const double *Y, double T, double *mu,
                       double *kappa, double *rhoD, double *h) {
  const int N = c->N;
  const double lnT = log(T);
  double X[XO_MAXN], ms[XO_MAXN], ks[XO_MAXN];
  double sum = 0.0, Rbar = 0.0;
  for (int s = 0; s < N; ++s) sum += Y[s] / c->W[s];
  for (int s = 0; s < N; ++s) {
    X[s] = (Y[s] / c->W[s]) / sum;                                /* mole fractions */
    ms[s] = fit_eval(tr->mu[s], lnT);
    ks[s] = fit_eval(tr->kappa[s], lnT);
    Rbar += Y[s] * (c->Ru / c->W[s]);
    double cp, es;
    xo_species_thermo(c, s, T, &cp, &h[s], &es);
  }
  const double p = rho * Rbar * T;                                /* Eq. 7 */
  /* Eq. 22 (Wilke), for mu and for kappa with the ratio of the respective property */
  double m = 0.0, k = 0.0;
  for (int s = 0; s < N; ++s) {
    double dm = 0.0, dk = 0.0;
    for (int t = 0; t < N; ++t) {
      const double w = 1.0 / sqrt(8.0) / sqrt(1.0 + c->W[s] / c->W[t]);
      const double q4 = sqrt(sqrt(c->W[t] / c->W[s]));
      const double bm = 1.0 + sqrt(ms[s] / ms[t]) * q4, bk = 1.0 + sqrt(ks[s] / ks[t]) * q4;
      dm += X[t] * w * bm * bm;
      dk += X[t] * w * bk * bk;
    }
    m += X[s] * ms[s] / dm;
    k += X[s] * ks[s] / dk;
  }
  *mu = m;
  *kappa = k;
  /* Eq. 26 with X_t + 1e-12 (reading R20); D_st(T, p) = D_st(T, p_ref) p_ref / p (reading R19) */
  double Wbar = 0.0;
  for (int s = 0; s < N; ++s) Wbar += X[s] * c->W[s];
  for (int s = 0; s < N; ++s) {
    double num = 0.0, den = 0.0;
    for (int t = 0; t < N; ++t) {
      if (t == s) continue;
      const double Dst = fit_eval(tr->D[s][t], lnT) * tr->p_ref / p;
      num += (X[t] + 1e-12) * c->W[t];
      den += (X[t] + 1e-12) / Dst;
    }
    rhoD[s] = N > 1 ? rho * num / (Wbar * den) : 0.0;
  }
}

typedef struct { double u[3], T, Y[XO_MAXN], h[XO_MAXN], mu, kappa, rD[XO_MAXN]; } vcell;

static void vcell_at(const xo_config *c, const xo_transport *tr, const double *U, const double *T, long cells, long id,
                     vcell *V) {
  const int N = c->N;
  const double rho = U[id];
  for (int q = 0; q < 3; ++q) V->u[q] = U[(1 + q) * cells + id] / rho;
  double sum = 0.0;
  for (int i = 0; i < N - 1; ++i) {
    V->Y[i] = U[(5 + i) * cells + id] / rho;
    sum += V->Y[i];
  }
  V->Y[N - 1] = 1.0 - sum;
  V->T = T[id];
  xo_transport_cell(c, tr, rho, V->Y, V->T, &V->mu, &V->kappa, V->rD, V->h);
}

static double interp4(double m1, double a, double b, double p2) { return (9.0 * (a + b) - (m1 + p2)) / 16.0; }
static double dnorm4(double m1, double a, double b, double p2, double dx) { return (27.0 * (b - a) - (p2 - m1)) / (24.0 * dx); }
static double dctr4(double mm, double m, double p, double pp, double dx) { return (mm - 8.0 * m + 8.0 * p - pp) / (12.0 * dx); }

/* face above padded cell ia in direction d, from the per-cell table V (all padded cells) */
static void vface(const xo_config *c, const vcell *V, const long st[3], const int n[3], long ia, int d, double *F,
                  double *J_out) {
  const int N = c->N, Nv = N + 4;
  const double dxs[3] = {c->dx, c->dy, c->dz};
  const vcell *q[4];
  for (int k = 0; k < 4; ++k) q[k] = V + ia + (long)(k - 1) * st[d];
#define FACE(field) interp4(q[0]->field, q[1]->field, q[2]->field, q[3]->field)
#define DN(field) dnorm4(q[0]->field, q[1]->field, q[2]->field, q[3]->field, dxs[d])
  double G[3][3];                                                 /* G[p][e] = d u_p / d x_e at the face */
  for (int p = 0; p < 3; ++p)
    for (int e = 0; e < 3; ++e) {
      if (e == d) G[p][e] = DN(u[p]);
      else if (n[e] == 1) G[p][e] = 0.0;
      else {
        double t[4];
        for (int k = 0; k < 4; ++k) {
          const vcell *z = q[k];
          t[k] = dctr4((z - 2 * st[e])->u[p], (z - st[e])->u[p], (z + st[e])->u[p], (z + 2 * st[e])->u[p], dxs[e]);
        }
        G[p][e] = interp4(t[0], t[1], t[2], t[3]);
      }
    }
  const double mu = FACE(mu), kappa = FACE(kappa);
  const double div = G[0][0] + G[1][1] + G[2][2];
  double tau[3];                                                  /* tau_{p d}, Eq. 3 */
  for (int p = 0; p < 3; ++p) tau[p] = mu * (G[p][d] + G[d][p]) - (p == d ? 2.0 / 3.0 * mu * div : 0.0);
  double J[XO_MAXN], dY[XO_MAXN], corr = 0.0;
  for (int s = 0; s < N; ++s) {
    dY[s] = DN(Y[s]);
    corr += FACE(rD[s]) * dY[s];
  }
  double qd = 0.0;
  for (int s = 0; s < N; ++s) {                                   /* Eq. 6 (reading R21), Eq. 5 */
    J[s] = -(FACE(rD[s]) * dY[s] - FACE(Y[s]) * corr);
    qd += FACE(h[s]) * J[s];
  }
  for (int v = 0; v < Nv; ++v) F[v] = 0.0;
  double work = 0.0;
  for (int p = 0; p < 3; ++p) {
    F[1 + p] = tau[p];
    work += tau[p] * FACE(u[p]);
  }
  F[4] = work + kappa * DN(T) - qd;                               /* tau.u - q_c - q_d, q_c = -kappa grad T (Eq. 4) */
  for (int s = 0; s < N - 1; ++s) F[5 + s] = -J[s];
  if (J_out) for (int s = 0; s < N; ++s) J_out[s] = J[s];
#undef FACE
#undef DN
}

static vcell *vcell_table(const xo_config *c, const xo_transport *tr, const double *U, const double *T) {
  const long cells = xo_padded_cells(c);
  vcell *V = (vcell *)malloc(sizeof(vcell) * cells);
#pragma omp parallel for schedule(static) if (cells > 16384)
  for (long id = 0; id < cells; ++id) vcell_at(c, tr, U, T, cells, id, &V[id]);
  return V;
}

void xo_viscous_face_flux(const xo_config *c, const xo_transport *tr, const double *U, const double *T, long ia, int d,
                          double *F, double *J_out) {
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  vcell *V = vcell_table(c, tr, U, T);
  vface(c, V, st, n, ia, d, F, J_out);
  free(V);
}

int xo_viscous_rhs(const xo_config *c, const xo_transport *tr, const double *U, const double *T, double *rhs) {
  const int Nv = c->N + 4;
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  const long cells = xo_padded_cells(c);
  const double dxs[3] = {c->dx, c->dy, c->dz};
  vcell *V = vcell_table(c, tr, U, T);
  memset(rhs, 0, sizeof(double) * Nv * cells);
  for (int d = 0; d < 3; ++d) {
    if (n[d] == 1) continue;
    const int a1 = (d + 1) % 3, a2 = (d + 2) % 3;
    const long npen = (long)n[a1] * n[a2];
#pragma omp parallel if (npen > 16)
    {
      double *Fv = (double *)malloc(sizeof(double) * (n[d] + 3) * Nv);
#pragma omp for schedule(dynamic, 4)
      for (long pen = 0; pen < npen; ++pen) {
        const int p = g[a1] + (int)(pen / n[a2]), q = g[a2] + (int)(pen % n[a2]);
        const long base = (long)p * st[a1] + (long)q * st[a2];
        /* faces above cells g-2 .. g+n: the n+1 faces of the interior cells and one more on either side */
        for (int f = 0; f < n[d] + 3; ++f) vface(c, V, st, n, base + (long)(g[d] - 2 + f) * st[d], d, Fv + f * Nv, NULL);
        for (int i = 0; i < n[d]; ++i) {                          /* cell g+i: faces f = i+1 (below), i+2 (above) */
          const long idx = base + (long)(g[d] + i) * st[d];
          for (int v = 0; v < Nv; ++v)
            rhs[v * cells + idx] += (27.0 * (Fv[(i + 2) * Nv + v] - Fv[(i + 1) * Nv + v]) -
                                     (Fv[(i + 3) * Nv + v] - Fv[i * Nv + v])) / (24.0 * dxs[d]);
        }
      }
      free(Fv);
    }
  }
  free(V);
  return 0;
}

int xo_rhs_ns(const xo_config *c, const xo_transport *tr, double *U, double *T, double *rhs) {
  int status = xo_rhs(c, U, T, rhs);                    /* ghosts filled, T converged on every padded cell */
  if (tr) {
    const int Nv = c->N + 4;
    const long cells = xo_padded_cells(c);
    double *rv = (double *)malloc(sizeof(double) * Nv * cells);
    status |= xo_viscous_rhs(c, tr, U, T, rv);
    for (long q = 0; q < Nv * cells; ++q) rhs[q] += rv[q];
    free(rv);
  }
  return status;
}

static int rk3_step(const xo_config *c_in, const xo_transport *tr, double *U, double *T, double dt) {
  xo_config cc = *c_in;
  cc.pp_dt = dt;                                          /* every stage is a forward-Euler step of size dt (Eq. 16, 17) */
  const xo_config *c = &cc;
  const int Nv = c->N + 4;
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  const long cells = xo_padded_cells(c);
  const size_t bytes = sizeof(double) * Nv * cells;
  double *U1 = (double *)malloc(bytes), *U2 = (double *)malloc(bytes), *Lr = (double *)malloc(bytes);
  int status = 0;
  status |= xo_rhs_ns(c, tr, U, T, Lr);                       /* L(U^n) */
  memcpy(U1, U, bytes);
  memcpy(U2, U, bytes);
#define FOR_INTERIOR                                                                  \
  for (int v = 0; v < Nv; ++v)                                                        \
    for (int k = g[2]; k < g[2] + n[2]; ++k)                                          \
      for (int j = g[1]; j < g[1] + n[1]; ++j)                                        \
        for (int i = g[0]; i < g[0] + n[0]; ++i)
  FOR_INTERIOR {
    const long id = v * cells + (long)k * st[2] + (long)j * st[1] + i;
    U1[id] = U[id] + dt * Lr[id];
  }
  status |= xo_rhs_ns(c, tr, U1, T, Lr);                       /* L(U^1) */
  FOR_INTERIOR {
    const long id = v * cells + (long)k * st[2] + (long)j * st[1] + i;
    U2[id] = 0.75 * U[id] + 0.25 * (U1[id] + dt * Lr[id]);
  }
  status |= xo_rhs_ns(c, tr, U2, T, Lr);                       /* L(U^2) */
  FOR_INTERIOR {
    const long id = v * cells + (long)k * st[2] + (long)j * st[1] + i;
    U[id] = 1.0 / 3.0 * U[id] + 2.0 / 3.0 * (U2[id] + dt * Lr[id]);
  }
#undef FOR_INTERIOR
  free(U1); free(U2); free(Lr);
  return status;
}

int xo_rk3_step(const xo_config *c, double *U, double *T, double dt) { return rk3_step(c, NULL, U, T, dt); }
int xo_rk3_step_ns(const xo_config *c, const xo_transport *tr, double *U, double *T, double dt) {
  return rk3_step(c, tr, U, T, dt);
}

/* ------------------------------------------------------------------------------------------------------------ */
/* Max wave speed for the CFL time step: S = max_cells sum_d (|u_d| + c)/dx_d; dt = CFL/S                       */
/* (Eq. 17 lambda = dt/dx = CFL/Lambda~ in 1-D; PAPER.md:429 global minimum step; reading R9)      */
/* ------------------------------------------------------------------------------------------------------------ */
double xo_max_wavespeed(const xo_config *c, const double *U, double *T, int *status_out) {
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  const long cells = xo_padded_cells(c);
  const double dxs[3] = {c->dx, c->dy, c->dz};
  double S = 0.0;
  int status = 0;
#pragma omp parallel for reduction(max : S) reduction(| : status) collapse(2) if (cells > 16384)
  for (int k = g[2]; k < g[2] + n[2]; ++k)
    for (int j = g[1]; j < g[1] + n[1]; ++j)
      for (int i = g[0]; i < g[0] + n[0]; ++i) {
        const long idx = (long)k * st[2] + (long)j * st[1] + i;
        double Uc[XO_MAXNV];
        xo_prim P;
        gather_cell(c, U, cells, idx, Uc);
        xo_cell_primitives(c, Uc, T[idx], &P);
        T[idx] = P.T;
        status |= P.status;
        double s = 0.0;
        for (int d = 0; d < 3; ++d)
          if (n[d] > 1) s += (fabs(P.vel[d]) + P.c) / dxs[d];
        if (s > S) S = s;
      }
  if (status_out) *status_out = status;
  return S;
}

/* ------------------------------------------------------------------------------------------------------------ */
/* Reaction step: alpha-QSS predictor-corrector (Eq. 8-12; 180-198 Eq. 27-28; readings R24-R30)      */
/* ------------------------------------------------------------------------------------------------------------ */
double xo_qss_alpha(double r) {
  if (r < 0.1) {   /* alpha = 1/(1 - e^-r) - 1/r = 1/2 + r/12 - r^3/720 + r^5/30240 - r^7/1209600 + O(r^9) */
    const double r2 = r * r;
    return 0.5 + r * (1.0 / 12.0 - r2 * (1.0 / 720.0 - r2 * (1.0 / 30240.0 - r2 / 1209600.0)));
  }
  const double em = 1.0 - exp(-r);
  return (1.0 - em / r) / em;
}

static double ipow(double x, int n) {
  double y = 1.0;
  for (int k = 0; k < n; ++k) y *= x;
  return y;
}

void xo_reaction_rates(const xo_config *c, const xo_mechanism *m, double rho, const double *Y, double T, double *q,
                       double *d) {
  const int N = c->N;
  double conc[XO_MAXN], g0[XO_MAXN];              /* [X_s]; S_s/R_s - h_s/(R_s T) */
  double Tc = T;
  if (Tc < c->Tlo) Tc = c->Tlo;
  if (Tc > c->Thi) Tc = c->Thi;
  for (int s = 0; s < N; ++s) {
    conc[s] = rho * Y[s] / c->W[s];
    const double *a = c->a[s];
    double cp, h, e;
    xo_species_thermo(c, s, T, &cp, &h, &e);
    const double Rs = c->Ru / c->W[s];
    const double SR = a[0] * log(Tc) + Tc * (a[1] + Tc * (a[2] / 2.0 + Tc * (a[3] / 3.0 + Tc * a[4] / 4.0))) + a[6] +
                      (cp / Rs) * log(T / Tc);
    g0[s] = SR - h / (Rs * T);
    q[s] = 0.0;
    d[s] = 0.0;
  }
  for (int r = 0; r < m->NR; ++r) {
    const double kf = m->A[r] * pow(T, m->B[r]) * exp(-m->E[r] / (c->Ru * T));     /* Eq. 11 (reading R24) */
    int dnu = 0;
    double dg = 0.0;
    for (int s = 0; s < N; ++s) {
      const int nu = m->nu_p[r][s] - m->nu_r[r][s];                               /* Eq. 10 */
      dnu += nu;
      dg += nu * g0[s];
    }
    const double Kc = pow(m->p_atm / (c->Ru * T), (double)dnu) * exp(dg);         /* Eq. 12 */
    const double kb = kf / Kc;
    double tb = 1.0;
    if (m->third[r]) {
      tb = 0.0;
      for (int s = 0; s < N; ++s) tb += m->eff[r][s] * conc[s];
    }
    double Rf = tb * kf, Rb = tb * kb;
    for (int s = 0; s < N; ++s) {
      Rf *= ipow(conc[s], m->nu_r[r][s]);
      Rb *= ipow(conc[s], m->nu_p[r][s]);
    }
    for (int s = 0; s < N; ++s) {                                                 /* Eq. 9 split as Eq. 27 (reading R25) */
      const double w = c->W[s] / rho;
      q[s] += w * (m->nu_p[r][s] * Rf + m->nu_r[r][s] * Rb);
      d[s] += w * (m->nu_r[r][s] * Rf + m->nu_p[r][s] * Rb);
    }
  }
}

/* temperature from the fixed internal energy e and the composition Y (C2's Newton iteration) */
static int T_of_e(const xo_config *c, const double *Y, double e, double *T) {
  double Tk = *T;
  for (int k = 0; k < c->maxit; ++k) {
    double Rbar, eT, Cv;
    xo_mixture(c, Y, Tk, &Rbar, &eT, &Cv);
    const double Tn = Tk + (e - eT) / Cv;
    const double dT = fabs(Tn - Tk);
    Tk = Tn;
    if (dT <= c->rtol * fabs(Tn)) { *T = Tk; return 0; }
    if (!(Tn == Tn)) break;
  }
  *T = Tk;
  return XO_ENOCONV;
}

int xo_react_cell(const xo_config *c, const xo_mechanism *m, double *Uc, double *T, double dt, int n_sub, int n_corr) {
  const int N = c->N;
  xo_prim P;
  memset(&P, 0, sizeof(P));
  cell_basic(c, Uc, &P);                           /* rho, Y (closure), e: rho and e stay fixed (reading R29) */
  int status = 0;
  double Y0[XO_MAXN] = {0}, Yp[XO_MAXN] = {0}, q0[XO_MAXN], d0[XO_MAXN], p0[XO_MAXN] = {0}, qp[XO_MAXN], dp[XO_MAXN];
  for (int s = 0; s < N; ++s) Y0[s] = P.Y[s];
  double Tk = *T;
  status |= T_of_e(c, Y0, P.e, &Tk);
  const double h = dt / n_sub;
  for (int sub = 0; sub < n_sub; ++sub) {
    xo_reaction_rates(c, m, P.rho, Y0, Tk, q0, d0);
    double sum = 0.0;
    for (int s = 0; s < N - 1; ++s) {              /* predictor, Eq. 28 */
      p0[s] = Y0[s] > 0.0 ? d0[s] / Y0[s] : 0.0;
      const double a0 = xo_qss_alpha(p0[s] * h);
      Yp[s] = Y0[s] + h * (q0[s] - p0[s] * Y0[s]) / (1.0 + a0 * p0[s] * h);
      sum += Yp[s];
    }
    Yp[N - 1] = 1.0 - sum;
    double Tp = Tk;
    for (int it = 0; it < n_corr; ++it) {          /* corrector(s) (reading R27) */
      status |= T_of_e(c, Yp, P.e, &Tp);
      xo_reaction_rates(c, m, P.rho, Yp, Tp, qp, dp);
      sum = 0.0;
      double Yc[XO_MAXN];
      for (int s = 0; s < N - 1; ++s) {
        const double pp = Yp[s] > 0.0 ? dp[s] / Yp[s] : 0.0;
        const double pb = 0.5 * (p0[s] + pp);
        const double ab = xo_qss_alpha(pb * h);
        const double qb = ab * qp[s] + (1.0 - ab) * q0[s];
        Yc[s] = Y0[s] + h * (qb - pb * Y0[s]) / (1.0 + ab * pb * h);
        sum += Yc[s];
      }
      Yc[N - 1] = 1.0 - sum;
      for (int s = 0; s < N; ++s) Yp[s] = Yc[s];
    }
    for (int s = 0; s < N; ++s) Y0[s] = Yp[s];
    Tk = Tp;
    status |= T_of_e(c, Y0, P.e, &Tk);
  }
  for (int s = 0; s < N - 1; ++s) Uc[5 + s] = P.rho * Y0[s];
  *T = Tk;
  if (!(Tk > 0.0)) status |= XO_ENONPHYSICAL;
  return status;
}

int xo_react(const xo_config *c, const xo_mechanism *m, double *U, double *T, double dt, int n_sub, int n_corr) {
  const int Nv = c->N + 4;
  int np[3], n[3], g[3];
  long st[3];
  grid(c, np, n, g, st);
  const long cells = xo_padded_cells(c);
  int status = 0;
#pragma omp parallel for reduction(| : status) collapse(2) if (cells > 4096)
  for (int k = g[2]; k < g[2] + n[2]; ++k)
    for (int j = g[1]; j < g[1] + n[1]; ++j)
      for (int i = g[0]; i < g[0] + n[0]; ++i) {
        const long idx = (long)k * st[2] + (long)j * st[1] + i;
        double Uc[XO_MAXNV];
        gather_cell(c, U, cells, idx, Uc);
        double Tk = T[idx];
        status |= xo_react_cell(c, m, Uc, &Tk, dt, n_sub, n_corr);
        for (int v = 5; v < Nv; ++v) U[v * cells + idx] = Uc[v];
        T[idx] = Tk;
      }
  return status;
}
