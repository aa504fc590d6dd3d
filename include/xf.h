/*
 * xf.h -- C ABI of libxf.so: the convective right-hand side of the multicomponent compressible Euler equations
 * (the per-Runge-Kutta-stage hot path of XFluids, arxiv 2403.05910) as hand-written CUDA for sm_100a.
 *
 * Citations are PAPER.md:<line> (the paper) and DESIGN.md readings R1..R30 where the paper prints no formula.
 *
 * Conventions
 *   Variables   Nv = N + 4 per cell: v = 0 rho, 1..3 rho u, rho v, rho w, 4 E, 5.. rho Y_1 .. rho Y_{N-1}
 *               (Eq. 2; "s = 1..N-1"); Y_N = 1 - sum of the others.
 *   Layout      SoA, fp64, U[v][k][j][i], i fastest.  Every ACTIVE direction (n_d > 1) carries ng ghost cells on both
 *               sides (ng = 3: WENO5 stencil i-2..i+3; ng = 4 for WENO7); an inactive direction
 *               (n_d == 1) has none.  padded extent np_d = n_d + 2 ng (active) or 1; padded cells = npx*npy*npz; field v starts at
 *               U + v*padded_cells.  Scalar fields (T, p, c) are [k][j][i] over the same padded box.
 *   Memory      All field pointers are CALLER-OWNED DEVICE memory (8-byte aligned) unless the name ends in
 *               _host.  The library allocates nothing per call; the context owns the species table, boundary
 *               states, a status word and a few scalars.  `work` must hold xf_workspace_bytes(ctx) bytes
 *               (xf_rhs_workspace_bytes suffices for xf_convective_rhs).
 *   Streams     `stream` is a cudaStream_t passed as void* (NULL = default stream).  Every call is asynchronous
 *               on that stream except xf_create / xf_destroy / xf_status / the *_host calls.
 *   Errors      Every call returns XF_OK or a negative code.  Argument errors are detected on the host before
 *               any launch (XF_EINVAL).  CUDA errors map to XF_ECUDA.  Physics failures (NaN, rho/T/p <= 0,
 *               Newton not converged; the paper's error catcher) set a sticky device flag that
 *               xf_status returns and clears.  No exceptions, no global mutable state: contexts are independent.
 *               There is no CPU fallback: without a CUDA device xf_create fails with XF_ECUDA.
 */
#ifndef XF_H
#define XF_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct xf_ctx xf_ctx; /* opaque, owned by the library */

enum {
  XF_OK = 0,
  XF_EINVAL = -1,
  XF_ECUDA = -2,
  XF_ENOMEM = -3,
  XF_ENONPHYSICAL = -4, /* NaN or rho, p, T <= 0 (or c~^2 <= 0 at a face) seen on the device */
  XF_ENOCONV = -5,      /* Newton iteration hit newton_maxit                                 */
  XF_ETOOBIG = -6       /* problem exceeds the static scratch of xf_convective_rhs_noalloc     */
};

enum { XF_BC_PERIODIC = 0, XF_BC_TRANSMISSIVE = 1, XF_BC_REFLECTIVE = 2, XF_BC_DIRICHLET = 3,
       XF_BC_EXCHANGE = 4 /* the face borders another block: its ghosts come from the halo exchange below */ };

#define XF_MAX_SPECIES 16
#define XF_MAX_REACTIONS 64

typedef struct {
  int nx, ny, nz;          /* interior cells; == 1 -> direction inactive (no ghosts, no sweep)                  */
  int ng;                  /* ghost width = half the stencil: 3 (WENO5, WENO-CU6), 4 for XF_RECON_WENO7         */
  double dx, dy, dz;
  int nspecies;            /* N in 1..XF_MAX_SPECIES; Nv = N + 4                                                */
  double Ru;               /* universal gas constant in the caller's units (Eq. 7)                  */
  const double *W;         /* host [N] molar masses                                                             */
  const double *nasa7;     /* host [N][7] NASA-7 a1..a7, single range (a7, the entropy constant, is used by the
                              reaction step only)                                                   */
  double Tlo, Thi;         /* fit range; constant-cp continuation outside it (reading R3)                       */
  int bc[6];               /* xlo, xhi, ylo, yhi, zlo, zhi: XF_BC_*                                             */
  const double *bc_state;  /* host [6][Nv] conserved states of XF_BC_DIRICHLET faces, or NULL                   */
  double newton_rtol;      /* |dT| <= rtol |T|; 0 -> 1e-13 (reading R4)                                         */
  int newton_maxit;        /* 0 -> 50                                                                           */
  int device;              /* CUDA ordinal                                                                      */
  int viscosity;           /* XF_VISC_*: the artificial viscosity Lambda~ of Eq. 14 (options 374)  */
  int reconstruction;      /* XF_RECON_*: the reconstruction of Eq. 15                            */
  int positivity;          /* != 0: positivity-preserving flux blending of Eq. 17-20, see below */
  const double *transport; /* host: fitted transport coefficients (Eq. 29), or NULL = no viscous /
                              diffusive terms.  ln eta = a_0 + a_1 ln T + a_2 (ln T)^2 + a_3 (ln T)^3, laid out as
                              mu [N][4], kappa [N][4], D [N][N][4] (binary D_st at p_ref, symmetric), then p_ref   */
} xf_config;

/* Positivity-preserving flux blending (theta is deferred by the paper to its ref 41 -> DESIGN.md
 * reading R17).  Every face flux of every sweep becomes F* = (1 - theta) F^LF + theta Fhat (Eq. 20) with the first-order
 * Lax-Friedrichs flux F^LF = (F_a + F_b + Lambda~ (U_a - U_b))/2 of the two adjacent cells (Eq. 19, Lambda~ = max(|u_d| +
 * c)).  Guarded: q in {rho, rho Y_1, .., rho Y_N (by closure)}; with kappa = 2 D dt/dx_d (Eq. 18, D active directions)
 * the half-states q(U_a) - kappa q(F), q(U_b) + kappa q(F) must stay >= eps = min(1e-13, the same half-state under
 * F^LF); theta in [0, 1] is the largest factor for which all 2 (N + 1) of them do; one factor for the whole flux vector.
 * theta = 1 (flux untouched, bit-identical residual) wherever nothing is violated.  dt is the forward-Euler step the
 * limiter guards: the step of xf_rk3_step / xf_rk3_step_cfl / xf_step_cfl in each of their three stages, and for a bare
 * xf_convective_rhs the value set by xf_set_rhs_dt (initially 0: every guard passes when U itself is non-negative).
 * Non-negativity of rho and Y_s after a stage holds if D dt Lambda~/dx_d <= 1/2 in every direction ("CFL <= 0.5",
 * PAPER.md:135). */

/* Reconstruction of the split characteristic fluxes at a face:
 *   WENO5   Jiang-Shu, eps = 1e-6, exponent 2 (reading R7; the default), points i-2..i+2 / mirrored
 *   WENOCU6 the six-point central-upwind scheme of the paper's ref 34 (reading R16: linear weights 1/20, 9/20, 9/20,
 *           1/20; fourth indicator = the six-point Jiang-Shu measure beta_6; tau_6 = beta_6 - (beta_0 + 4 beta_1 +
 *           beta_2)/6; alpha_k = d_k (20 + tau_6/(beta_k + 1e-40))), points i-2..i+3 / mirrored: same ghost width
 *   WENO7   the seventh-order scheme of the paper's ref 36 (reading R18: four cubic candidates, linear weights 1/35,
 *           12/35, 18/35, 4/35, Jiang-Shu indicators of the cubics, alpha_k = d_k/(1e-6 + beta_k)^2), points i-3..i+3 /
 *           mirrored: stencil i-3..i+4, so the context must be created with ng = 4 */
enum { XF_RECON_WENO5 = 0, XF_RECON_WENOCU6 = 1, XF_RECON_WENO7 = 2 };

/* Lambda~_n of the flux splitting f+- = (L F +- Lambda~ L U)/2, per characteristic field n:
 *   LLF  max over the six stencil cells of |lambda_n| of each cell's own state (reading R8; the default)
 *   ROE  |lambda_n| of the Roe-averaged face state (u~_d - c~, u~_d, u~_d + c~), no maximum
 *   GLF  max of |lambda_n| over ALL padded cells, per direction, reduced inside the primitives kernel of the same
 *        residual evaluation (ghosts filled) */
enum { XF_VISC_LLF = 0, XF_VISC_ROE = 1, XF_VISC_GLF = 2 };

/* Create a context: validates cfg, copies every host table, uploads boundary states.  Synchronous. */
int xf_create(xf_ctx **out, const xf_config *cfg);
int xf_destroy(xf_ctx *ctx);

size_t xf_num_vars(const xf_ctx *ctx);            /* Nv                                                        */
size_t xf_padded_cells(const xf_ctx *ctx);        /* product of padded extents                                 */
size_t xf_rhs_workspace_bytes(const xf_ctx *ctx); /* scratch for xf_convective_rhs / xf_viscous_rhs: (N + 4) fields
                                                     (+ 3 N + 5 with a transport table)                        */
size_t xf_workspace_bytes(const xf_ctx *ctx);     /* scratch for the RK3 calls: the above + 3 U-sized buffers  */

/* Ghost-cell fill ("specific boundary conditions"; reading R10): periodic wrap,
 * transmissive copy of the nearest interior cell, reflective mirror with the wall-normal momentum negated, or the
 * stored Dirichlet state; ng layers; x, then y, then z, so that edges and corners are defined.  U in place. */
int xf_fill_ghosts(xf_ctx *ctx, double *U, void *stream);

/* Primitive recovery for every padded cell (Eq. 21): T by Newton iteration on
 * e(T) = sum_s Y_s h_s(T) - Rbar T with Cv = sum_s Y_s cp_s - Rbar; then p = rho Rbar T (Eq. 7) and the frozen
 * sound speed c.  T: in = starting guess, out = temperature.  p and/or c may be NULL.  U must have valid ghosts. */
int xf_primitives(xf_ctx *ctx, const double *U, double *T, double *p, double *c, void *stream);

/* One convective residual L(U) = -sum_d (Fhat_{i+1/2} - Fhat_{i-1/2})/dx_d (Eq. 13) with
 * characteristic-wise WENO5 reconstruction, local Lax-Friedrichs splitting (Eq. 14) on the
 * Roe-averaged eigensystem and back-projection (Eq. 15).  Does: ghost fill (U's ghosts are
 * overwritten, interior read-only), primitives (T in/out), the x, y, z sweeps.  rhs is [Nv][padded]; only interior
 * entries are written.  work: xf_rhs_workspace_bytes. */
int xf_convective_rhs(xf_ctx *ctx, double *U, double *T, double *rhs, void *work, void *stream);

/* xf_convective_rhs WITHOUT a caller-provided workspace, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it): the scratch of the residual evaluation (p, c, 1/rho, Gamma,
 * chi_s per padded cell -- and the cell table of the viscous terms for a context with a transport table) lives in ONE
 * file-scope `static __device__` array of XF_NOALLOC_SCRATCH_BYTES inside the library.  Every GPU that loads the
 * library holds that array until the process exits.  Same arithmetic, same kernels and same result, bit for bit, as
 * xf_convective_rhs; U, T and rhs are the caller's device arrays as there.
 *   - calls no cudaMalloc / cudaFree or allocating library routine (the context was created earlier, by xf_create);
 *   - returns XF_ETOOBIG, launching nothing, when xf_rhs_workspace_bytes(ctx) > XF_NOALLOC_SCRATCH_BYTES
 *     (N = 10: up to 599 186 padded cells, e.g. 78^3);
 *   - the array is shared by every context and every call on that GPU and keeps the last call's contents.  Nothing in
 *     it has to start at zero: the primitives (and transport) kernel writes every field of every padded cell before a
 *     sweep reads it.  Two calls that OVERLAP on the GPU (different streams, or different host threads on different
 *     streams) race on it: serialise them on one stream or with events;
 *   - xf_noalloc_prepare resolves the array's device address for the context's device (cudaGetSymbolAddress, once per
 *     device, cached).  xf_convective_rhs_noalloc does the same on its first call for a device; call xf_noalloc_prepare
 *     beforehand where even that one-time query must stay out of the loop (before a graph capture begins). */
#define XF_NOALLOC_SCRATCH_BYTES (64u << 20)
size_t xf_noalloc_scratch_bytes(void);            /* = XF_NOALLOC_SCRATCH_BYTES of the loaded library */
int xf_noalloc_prepare(xf_ctx *ctx);
int xf_convective_rhs_noalloc(xf_ctx *ctx, double *U, double *T, double *rhs, void *stream);

/* Viscous / diffusive terms (context created with cfg.transport; Eq. 1-6; readings R19-R23):
 * F_v = (0, tau, tau.u + kappa grad T - sum_s h_s J_s, -J_s) with tau of Eq. 3, mu and kappa by Wilke's rule (Eq. 22) from
 * the fitted species values, J_s = -rho (D_sm grad Y_s - Y_s sum_i D_im grad Y_i) (Eq. 6), D_sm by Eq. 26, D_st ~ p_ref / p;
 * conservative fourth-order central discretisation within the three ghost layers of WENO5.
 *   xf_viscous_rhs   rhs = div F_v at interior cells.  U must have its ghosts filled and T must be the converged
 *                    temperature of every padded cell (both are as xf_convective_rhs leaves them).  work:
 *                    xf_rhs_workspace_bytes.
 * With a transport table the three RK3 entry points integrate L = convective + viscous residual (the viscous part is
 * evaluated first, into the partial-residual buffer the sweeps accumulate on); xf_convective_rhs stays convective. */
int xf_viscous_rhs(xf_ctx *ctx, const double *U, const double *T, double *rhs, void *work, void *stream);

/* Reaction step (Eq. 8-12; Eq. 27-28: the alpha-QSS solver CHEMEQ2 inside an operator
 * splitting; readings R24-R30).  xf_set_mechanism copies a mechanism of n_reactions <= XF_MAX_REACTIONS reversible
 * reactions into the context: nu_r, nu_p host [NR][N] non-negative integer coefficients of reactants and products (at most
 * three molecules a side), Arrhenius parameters k_f = A T^B exp(-E/(Ru T)), third[r] != 0 for a third-body reaction with
 * efficiencies eff [NR][N], p_atm the standard pressure of Eq. 12 in the caller's units; backward rates follow from the
 * equilibrium constants (NASA-7 entropies: a7 of the table).  xf_react advances the species of every INTERIOR cell over dt
 * at fixed rho, rho u and E: n_sub equal sub-steps of one predictor and n_corr correctors (Eq. 28), the temperature solved
 * from the internal energy after every update (T: in guess, out T).  Ghost cells are not touched. */
int xf_set_mechanism(xf_ctx *ctx, int n_reactions, const int *nu_r, const int *nu_p, const double *A, const double *B,
                     const double *E, const int *third, const double *eff, double p_atm);
int xf_react(xf_ctx *ctx, double *U, double *T, double dt, int n_sub, int n_corr, void *stream);

/* Domain decomposition (Cartesian blocks, one per GPU, the border layers of a block become the
 * boundary layers of its face neighbour).  A face of kind XF_BC_EXCHANGE is left alone by the ghost fill.  Per residual
 * evaluation the driver (paper_2403_05910_b200/halo.py) goes through the directions in order x, y, z and, for each:
 * xf_fill_ghosts_dir (the physical faces of that direction), xf_pack_halo of its exchange faces, the transfer (NCCL
 * send / recv, or a device copy between blocks of one process), xf_unpack_halo -- each over the padded extent of the
 * directions already done, so edges and corners arrive without diagonal messages.  Then xf_rk3_stage, which evaluates the
 * residual of Uin WITHOUT filling ghosts and writes stage `stage` (0, 1, 2) of Eq. 16: Uout = alpha Un + beta (Uin + dt
 * L(Uin)); stage 0: Uin = Un; the caller owns the stage arrays.  dt comes from the max over blocks of xf_max_wavespeed.
 *   xf_halo_doubles  size of one face buffer of direction dir: (Nv + 1) x ng x (transverse cells, padded for
 *                    directions < dir)
 *   buffers          caller-owned device memory, layout [Nv + 1][ng][transverse]: U and, as the last field, T (the Newton
 *                    guess of a ghost cell is then the one of the cell it mirrors, and a decomposed run reproduces the
 *                    single-block run bit for bit); pack: the ng interior layers next to the face (side 0 = low,
 *                    1 = high); unpack: the ng ghost layers beyond it. */
int xf_fill_ghosts_dir(xf_ctx *ctx, double *U, int dir, void *stream);
size_t xf_halo_doubles(const xf_ctx *ctx, int dir);
int xf_pack_halo(xf_ctx *ctx, const double *U, const double *T, int dir, int side, double *buf, void *stream);
int xf_unpack_halo(xf_ctx *ctx, double *U, double *T, int dir, int side, const double *buf, void *stream);
int xf_rk3_stage(xf_ctx *ctx, int stage, const double *Un, double *Uin, double *Uout, double *T, double dt, void *work,
                 void *stream);

/* The time step assumed by the positivity limiter of a bare xf_convective_rhs (see xf_config.positivity); dt >= 0. */
int xf_set_rhs_dt(xf_ctx *ctx, double dt);

/* One SSP-RK3 step with fixed dt (Eq. 16): three times (ghost fill, primitives, residual,
 * stage combination).  U: in U^n, out U^{n+1} (interior; ghosts are left as filled for the last stage).
 * work: xf_workspace_bytes. */
int xf_rk3_step(xf_ctx *ctx, double *U, double *T, double dt, void *work, void *stream);

/* As xf_rk3_step with dt = cfl / (*S_dev) read on the device (no host round trip); S_dev as written by
 * xf_max_wavespeed on the same stream. */
int xf_rk3_step_cfl(xf_ctx *ctx, double *U, double *T, double cfl, const double *S_dev, void *work, void *stream);

/* One whole time step at a given CFL number: S (as xf_max_wavespeed defines it, of the incoming U^n) is reduced inside
 * the primitives kernel of the first stage and written to *S_dev, and the three stages use dt = cfl / S read on the
 * device -- the same result as xf_max_wavespeed followed by xf_rk3_step_cfl, without recovering the primitives of
 * U^n twice.  S_dev: 1 double, device, written. */
int xf_step_cfl(xf_ctx *ctx, double *U, double *T, double cfl, double *S_dev, void *work, void *stream);

/* S = max over interior cells of sum_{d active} (|u_d| + c)/dx_d, so that dt = CFL / S (Eq. 17,
 * PAPER.md:429; reading R9).  Recovers T of the interior cells on the way (T in/out).  S_dev: 1 double, device. */
int xf_max_wavespeed(xf_ctx *ctx, const double *U, double *T, double *S_dev, void *stream);

/* Synchronises `stream`, returns XF_OK / XF_ENONPHYSICAL / XF_ENOCONV from the sticky device flag and clears it. */
int xf_status(xf_ctx *ctx, void *stream);

/* Mean Newton iteration count of the last xf_primitives launch (debug counter; synchronises the stream). */
int xf_newton_mean_iterations(xf_ctx *ctx, void *stream, double *mean_out);

/* Number of kernel launches issued through this context since xf_create (for bench.py's gpu_launches). */
long xf_launch_count(const xf_ctx *ctx);

/* Per-kernel device timing for the roofline report (bench.py): after xf_timing_enable(ctx, max_records) every
 * kernel the context launches is bracketed by a CUDA event pair on the caller's stream (up to max_records pairs
 * between two reads; further launches go untimed).  xf_timing_read synchronises `stream`, adds up the elapsed
 * milliseconds and the number of records per kernel kind into ms_out[XF_K_COUNT] / count_out[XF_K_COUNT], and
 * resets the record list.  max_records = 0 switches timing off.  The ghost fill (one launch per active direction)
 * is timed as one record. */
enum { XF_K_GHOST = 0, XF_K_PRIM = 1, XF_K_SWEEP_X = 2, XF_K_SWEEP_Y = 3, XF_K_SWEEP_Z = 4, XF_K_WAVESPEED = 5,
       XF_K_TRANSPORT = 6, XF_K_VISCOUS = 7, XF_K_REACT = 8, XF_K_COUNT = 9 };
int xf_timing_enable(xf_ctx *ctx, int max_records);
int xf_timing_read(xf_ctx *ctx, void *stream, double *ms_out, long *count_out);

/* HOST-buffer entry points (end-to-end measurement): copy in, run on the device, copy out.  Device scratch is
 * allocated inside the context on first use and freed by xf_destroy.  Synchronous.
 *   xf_convective_rhs_host: U_host [Nv][padded] in, T_host [padded] in/out, rhs_host [Nv][padded] out.
 *   xf_rk3_steps_host:      nsteps steps with dt = cfl / S recomputed every step on the device; U_host, T_host
 *                           in/out; *t_advanced (may be NULL) receives the sum of the time steps. */
int xf_convective_rhs_host(xf_ctx *ctx, const double *U_host, double *T_host, double *rhs_host);
int xf_rk3_steps_host(xf_ctx *ctx, double *U_host, double *T_host, double cfl, int nsteps, double *t_advanced);

/* Measurement aid for the roofline denominator: runs a register-resident chain of dependent-free fp64 FMAs on
 * every SM for `iters` rounds and returns the achieved TFLOP/s (2 flops per FMA) in *tflops.  Synchronous. */
int xf_probe_fp64_peak(int device, int iters, double *tflops, double *ms);
/* The same probe launched back to back for at least `seconds` (<= 30): the SUSTAINED figure, at the clocks the GPU
 * holds under a long fp64 load (the burst figure above is the best of five short launches). *ms = the timed span. */
int xf_probe_fp64_sustained(int device, double seconds, double *tflops, double *ms);

const char *xf_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* XF_H */
