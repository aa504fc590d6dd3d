/*
 * xf_oracle.h -- plain CPU oracle for the convective right-hand side of the multicomponent compressible Euler
 * equations (XFluids, arxiv 2403.05910).  TEST INFRASTRUCTURE ONLY.
 *
 * This is the slow, obviously-correct fp64 restatement of what the hot path computes.  It follows the paper
 * step by step (citations are PAPER.md:<line>, section / equation) and, where the paper prints no formula,
 * the readings R1..R30 listed in DESIGN.md (R1-R15 taken from SURVEY.md 8(c)).  It shares NO code with the CUDA path
 * (paper_2403_05910_b200/csrc): dense Nv x Nv eigenvector matrices and dense mat-vec products here, an expanded
 * structured form there; plain Jiang-Shu weights with three divisions here, a common-denominator form there.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load or
 * call anything in oracle/.  The product path never does.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): closed-form T(e); c^2 identity; L.R = I, L.A.R = diag
 * (finite-difference Jacobian); N = 1 textbook Euler eigenvectors and Roe sound speed; WENO5 exactness on
 * degree-4 polynomials, 5th order on smooth data; uniform-flow preservation; exact Sod Riemann solution; design
 * order on an advected density wave; round-off conservation; interface equilibrium (equal gamma); mirror and
 * permutation symmetry; direction consistency; dense-inverse brute-force face flux.
 * Roe's property U (F_b - F_a = A~ (U_b - U_a)) in the mass, tangential-momentum and species rows for a mixture and
 * in all rows for one perfect gas fixes the sqrt(rho) weights of u~, Y~_s, H~ (tests/test_oracle_pins_definitions.py).
 * Parity unpinned: agreement with XFluids' own code output and with the paper's Fig. 15 curves (neither code,
 * numbers nor reference data are available); the sqrt(rho) weighting of Gamma~ and chi~_s in xo_eigensystem (reading
 * R5: a definition that neither PAPER.md:107 nor the mathematics fixes; written out in the same test file).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared (no -ffast-math).  OpenMP only on outermost loops of
 * independent per-cell / per-face work, so results do not depend on the thread count.
 */
#ifndef XF_ORACLE_H
#define XF_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

#define XO_MAXN 16            /* max species */
#define XO_MAXNV (XO_MAXN + 4)

enum { XO_BC_PERIODIC = 0, XO_BC_TRANSMISSIVE = 1, XO_BC_REFLECTIVE = 2, XO_BC_DIRICHLET = 3 };
enum { XO_OK = 0, XO_ENONPHYSICAL = 4, XO_ENOCONV = 5 };   /* status bits */

typedef struct {
  int nx, ny, nz;             /* interior cells; n == 1 -> direction inactive (no ghosts, no sweep)           */
  int ng;                     /* ghost width: 3 (WENO5, WENO-CU6: stencil i-2..i+3) or 4 (WENO7: i-3..i+4)    */
  double dx, dy, dz;
  int N;                      /* species; Nv = N + 4                                                          */
  double Ru;
  double W[XO_MAXN];
  double a[XO_MAXN][7];       /* NASA-7 single range a1..a7 (a7 unused)                                       */
  double Tlo, Thi;
  int bc[6];                  /* xlo xhi ylo yhi zlo zhi                                                      */
  double bc_state[6][XO_MAXNV];
  double rtol;                /* Newton |dT| <= rtol |T|, 1e-13                                               */
  int maxit;                  /* 50                                                                           */
  int ideal_weights;          /* test switch: WENO5 with the linear weights               */
  int viscosity;              /* artificial viscosity of Eq. 14 (options PAPER.md:374):          */
                              /*   0 LLF: per field, max over the six stencil cells of |lambda_n| (reading R8)  */
                              /*   1 ROE: |lambda_n| of the Roe-averaged face state, no maximum                 */
                              /*   2 GLF: per field and direction, max of |lambda_n| over ALL padded cells      */
  double lam_glob[3][3];      /* GLF maxima [direction][u-c, u, u+c]; filled by the residual routines           */
  int recon;                  /* reconstruction of Eq. 15: 0 WENO5-JS (reading R7), 1 WENO-CU6 ("[34]"),  */
                              /*   2 WENO7 ("[36]"; reading R18; needs ng = 4)                            */
  int positivity;             /* 1: positivity-preserving flux blending for rho and rho Y_s (PAPER.md:120-141,         */
                              /*    Eq. 17-20; the limiting factor theta: reading R17)                                 */
  double pp_dt;               /* the time step the limiter guards (lambda = dt/dx of Eq. 17); xo_rk3_step sets it     */
} xo_config;
enum { XO_RECON_WENO5 = 0, XO_RECON_WENOCU6 = 1, XO_RECON_WENO7 = 2 };
enum { XO_VISC_LLF = 0, XO_VISC_ROE = 1, XO_VISC_GLF = 2 };

/* all primitive quantities of one cell (C2) */
typedef struct {
  double rho, vel[3], Y[XO_MAXN], e, T, p, Rbar, Cv, Gamma, c, H, chi[XO_MAXN];
  int iters, status;
} xo_prim;

/* grid helpers */
int xo_nv(const xo_config *c);
long xo_padded_cells(const xo_config *c);
void xo_padded_dims(const xo_config *c, int *nxp, int *nyp, int *nzp);

/* C1 thermodynamics */
void xo_species_thermo(const xo_config *c, int s, double T, double *cp, double *h, double *e);
void xo_mixture(const xo_config *c, const double *Y, double T, double *Rbar, double *e, double *Cv);

/* C2 primitive recovery of one cell / of the whole padded field */
void xo_cell_primitives(const xo_config *c, const double *Ucell, double Tguess, xo_prim *out);
int xo_primitives(const xo_config *c, const double *U, double *T, double *p, double *cs, double *iters_mean);

/* C3 physical flux of one cell in direction d */
void xo_phys_flux(const xo_config *c, const double *Ucell, const xo_prim *P, int d, double *F);

/* C4 dense face eigensystem from two cells' primitives: L, R are Nv x Nv row-major; returns status bits */
int xo_eigensystem(const xo_config *c, const xo_prim *A, const xo_prim *B, int d, double *L, double *R, double *roe);

/* C6 WENO5-JS: v[0..4] = v_{-2}..v_{+2}, value at +1/2 */
double xo_weno5(const double v[5], int ideal_weights);
/* WENO-CU6 value at +1/2 from v[0..5] = v_{-2}..v_{+3}; beta_out (may be NULL) receives beta_0, beta_1, beta_2, beta_6 and
 * w_out (may be NULL) the four normalised weights */
double xo_wenocu6(const double v[6], int ideal_weights, double *beta_out, double *w_out);

/* WENO7 ("[36]") value at +1/2 from v[0..6] = v_{-3}..v_{+3}; beta_out / w_out (may be NULL): the four
 * smoothness indicators / normalised weights */
double xo_weno7(const double v[7], int ideal_weights, double *beta_out, double *w_out);

/* number of stencil cells of a face flux: 6 (i-2..i+3) for WENO5 / WENO-CU6, 8 (i-3..i+4) for WENO7 */
int xo_stencil_cells(const xo_config *c);

/* C5-C7 numerical flux at one face from the S = xo_stencil_cells stencil cells (Ust[m][v], m = 0..S-1 <-> i-S/2+1..i+S/2;
 * the face lies between m = S/2-1 and m = S/2) */
int xo_face_flux(const xo_config *c, int d, const double *Ust, const xo_prim *Pst, double *Fhat);

/* Positivity-preserving blending at one face (Eq. 17-20; reading R17): cells a = i, b = i+1 (conserved
 * vectors + primitives), kappa = 2 D dt/dx_d (D = number of active directions), Fhat: in the high-order flux, out the
 * blended flux F* = (1-theta) F^LF + theta Fhat.  Returns theta. */
double xo_positivity_blend(const xo_config *c, int d, const double *Ua, const xo_prim *Pa, const double *Ub,
                           const xo_prim *Pb, double kappa, double *Fhat);

/* C8 ghost fill; C7 rhs, rk3, max wave speed.  U is [Nv][padded], T is [padded] (in: guess, out: T) */
void xo_fill_ghosts(const xo_config *c, double *U);
int xo_rhs(const xo_config *c, double *U, double *T, double *rhs);
int xo_rhs_nofill(const xo_config *c, const double *U, double *T, double *rhs);
/* rhs at sampled interior cells (padded linear indices idx[ncells]) straight from ghost-filled U and the T guess */
int xo_rhs_cells(const xo_config *c, const double *U, const double *Tguess, long ncells, const long *idx,
                 double *rhs_out);
int xo_rk3_step(const xo_config *c, double *U, double *T, double dt);
double xo_max_wavespeed(const xo_config *c, const double *U, double *T, int *status);

/* ------------------------------------------------------------------------------------------------------------------
 * Viscous / diffusive right-hand side div F_v (Eq. 1-6, Eq. 22, 26,
 * PAPER.md:505-513 Eq. 29, "central 4th-order accuracy scheme" PAPER.md:107).  Readings R19-R23 of DESIGN.md:
 *   R19 transport fits (Eq. 29): ln eta = a_0 + a_1 ln T + a_2 (ln T)^2 + a_3 (ln T)^3 for mu_s, kappa_s and for the binary
 *       D_st at the reference pressure p_ref; D_st(T, p) = D_st(T, p_ref) p_ref / p (Eq. 25: D ~ 1/p).
 *   R20 mixture rules as printed: Wilke's formula Eq. 22 for BOTH mu and kappa (Phi with the ratio of the respective
 *       property); D_sm by Eq. 26 with X_t + 1e-12 in both sums (the printed form is 0/0 for a pure species).
 *   R21 species diffusion flux, Eq. 6 with its indices repaired: J_s = -rho (D_sm grad Y_s - Y_s sum_i D_im grad Y_i), so
 *       that sum_s J_s = 0; the species row of F_v is -J_s and the energy row tau.u + kappa grad T - sum_s h_s J_s (the
 *       signs that make Eq. 1 a diffusion equation; Eq. 2 prints +J_s).
 *   R22 discretisation: conservative, fourth order.  At the face between cells a and b = a + 1 of direction d, with the
 *       four cells a-1, a, b, b+1: normal derivative (27 (f_b - f_a) - (f_{b+1} - f_{a-1}))/(24 dx_d); face value
 *       (9 (f_a + f_b) - (f_{a-1} + f_{b+1}))/16, used for mu, kappa, rho D_sm, Y_s, h_s, u; transverse derivatives =
 *       that face value of the cell-centred (f_{-2} - 8 f_{-1} + 8 f_{+1} - f_{+2})/(12 dx_e).  Divergence:
 *       (27 (F_{i+1/2} - F_{i-1/2}) - (F_{i+3/2} - F_{i-3/2}))/(24 dx_d).  Reach: three cells, the ghost width of WENO5.
 *   R23 the face-interpolated product rho D_sm (one cell quantity), not rho and D_sm apart.
 * U must have its ghosts filled and T must hold the converged temperature of every padded cell (xo_rhs leaves both so).
 * ------------------------------------------------------------------------------------------------------------------ */
typedef struct {
  double mu[XO_MAXN][4], kappa[XO_MAXN][4];     /* a_0..a_3 of ln mu_s, ln kappa_s in ln T                      */
  double D[XO_MAXN][XO_MAXN][4];                /* a_0..a_3 of ln D_st(T, p_ref); symmetric, diagonal unused    */
  double p_ref;
} xo_transport;

/* mixture transport of one cell: mu (Eq. 22), kappa (Eq. 22), rhoD[s] = rho D_sm (Eq. 26), h[s] (NASA polynomials) */
void xo_transport_cell(const xo_config *c, const xo_transport *tr, double rho, const double *Y, double T, double *mu,
                       double *kappa, double *rhoD, double *h);
/* viscous flux at the face above padded cell ia in direction d (all Nv rows; row 0 is zero); J_out (may be NULL)
 * receives the N diffusion fluxes J_s.n */
void xo_viscous_face_flux(const xo_config *c, const xo_transport *tr, const double *U, const double *T, long ia, int d,
                          double *F, double *J_out);
/* rhs[v][cell] = div F_v at interior cells (other entries zero) */
int xo_viscous_rhs(const xo_config *c, const xo_transport *tr, const double *U, const double *T, double *rhs);
/* convective + viscous residual, and one SSP-RK3 step with it (ghosts and primitives before each residual) */
int xo_rhs_ns(const xo_config *c, const xo_transport *tr, double *U, double *T, double *rhs);
int xo_rk3_step_ns(const xo_config *c, const xo_transport *tr, double *U, double *T, double dt);

/* ------------------------------------------------------------------------------------------------------------------
 * Reaction step (Eq. 8-12, Eq. 27-28: the alpha-QSS solver
 * CHEMEQ2 inside a Lie-Trotter / Strang splitting).  Readings R24-R30 of DESIGN.md:
 *   R24 Arrhenius law k_f = A T^B exp(-E/(Ru T)) (Eq. 11 prints +E/(Ru T)); K_c by Eq. 12 with S_s/R_s = a1 ln T + a2 T +
 *       a3 T^2/2 + a4 T^3/3 + a5 T^4/4 + a7 and h_s of C1 (outside the fit range: cp frozen, S continued with cp ln(T/Tc));
 *       k_b = k_f/K_c; p0 ("1 atm") is an input in the caller's units; molar concentrations [X_s] = rho Y_s / W_s; the
 *       third-body factor of a third-body reaction is sum_s eff_s [X_s], else 1.
 *   R25 Eq. 27: dY_s/dt = q_s - p_s Y_s with q_s = (W_s/rho) sum_r (nu''_sr R_f,r + nu'_sr R_b,r) and the destruction rate
 *       d_s = (W_s/rho) sum_r (nu'_sr R_f,r + nu''_sr R_b,r) = p_s Y_s; p_s = d_s/Y_s (0 where Y_s <= 0).
 *   R26 Eq. 28 with its alpha repaired: alpha(r) = (1 - (1 - e^-r)/r)/(1 - e^-r), r = p dt -- the value for which the update
 *       is exact when q and p are constant; for r < 0.1 its series 1/2 + r/12 - r^3/720 + r^5/30240 - r^7/1209600 (the
 *       closed form cancels there).  Predictor Y^p = Y^0 + dt (q^0 - p^0 Y^0)/(1 + alpha^0 p^0 dt); corrector with pbar = (p^0 + p^p)/2,
 *       abar = alpha(pbar dt), qbar = abar q^p + (1 - abar) q^0: Y^c = Y^0 + dt (qbar - pbar Y^0)/(1 + abar pbar dt).
 *   R27 "multiple corrector steps": n_corr >= 1 of them, each re-evaluating the rates at the last corrected state.
 *   R28 "multiple time steps": n_sub equal sub-steps dt/n_sub (the paper gives no step-size control).
 *   R29 the reaction step holds rho, rho u and E fixed (constant volume, adiabatic); T follows from e(T, Y) = e by the Newton
 *       iteration of C2 after every update of Y -- Eq. 8's heat release is then carried by the formation constants of h_s.
 *   R30 species 1..N-1 are integrated, Y_N = 1 - sum by closure as everywhere else (R1).
 * ------------------------------------------------------------------------------------------------------------------ */
#define XO_MAXR 64
typedef struct {
  int NR;
  int nu_r[XO_MAXR][XO_MAXN], nu_p[XO_MAXR][XO_MAXN];   /* nu' (reactants), nu'' (products): small non-negative integers */
  double A[XO_MAXR], B[XO_MAXR], E[XO_MAXR];            /* Arrhenius parameters of the forward rate                       */
  int third[XO_MAXR];                                   /* 1: third-body reaction                                         */
  double eff[XO_MAXR][XO_MAXN];                         /* third-body efficiencies                                        */
  double p_atm;                                         /* the standard pressure of Eq. 12 in the caller's units          */
} xo_mechanism;

double xo_qss_alpha(double r);
/* q[s], d[s] (1/time) of all N species at (rho, Y, T) */
void xo_reaction_rates(const xo_config *c, const xo_mechanism *m, double rho, const double *Y, double T, double *q,
                       double *d);
/* one cell: Ucell in/out (rho Y_s updated), T in (guess) / out; returns status bits */
int xo_react_cell(const xo_config *c, const xo_mechanism *m, double *Ucell, double *T, double dt, int n_sub, int n_corr);
/* all interior cells */
int xo_react(const xo_config *c, const xo_mechanism *m, double *U, double *T, double dt, int n_sub, int n_corr);

#ifdef __cplusplus
}
#endif
#endif
