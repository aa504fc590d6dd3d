// xf_common.cuh -- shared declarations of the CUDA path (sm_100a).  No code is shared with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/xf.h"

#define XF_MAXN XF_MAX_SPECIES
#define XF_MAXNV (XF_MAXN + 4)

// status bits on the device (sticky word owned by the context)
#define XF_FLAG_NONPHYSICAL 1
#define XF_FLAG_NOCONV 2

// Grid geometry handed to every kernel by value (lives in the kernel-parameter constant bank).
struct XfGrid {
  int n[3];        // interior cells per direction
  int np[3];       // padded extents
  int g[3];        // ghost width per direction (0 if inactive)
  long long st[3]; // element strides of i, j, k
  long long cells; // padded cells
  double inv_d[3]; // 1/dx, 1/dy, 1/dz
};

// Species table in evaluation form, handed to the thermo kernels by value (constant bank, <= 4 KB):
//   cp_s/R_s = a0 + a1 T + a2 T^2 + a3 T^3 + a4 T^4            (NASA polynomials; Horner)
//   h_s/R_s  = T (a0 + b1 T + b2 T^2 + b3 T^3 + b4 T^4) + a5,   b_k = a_k/(k+1)
struct XfThermo {
  double Rs[XF_MAXN];
  double a[XF_MAXN][6];  // a0..a4, a5 (enthalpy constant)
  double b[XF_MAXN][4];  // a1/2, a2/3, a3/4, a4/5
  double Tlo, Thi;
  double rtol;
  int maxit;
  int N;
};

// Transport fits of the viscous / diffusive terms in evaluation form, in DEVICE memory (13 KB: too large for the
// kernel-parameter bank): Eq. 29 coefficients and the species-pair constants of Wilke's rule (Eq. 22),
// w8[s][t] = 1 / sqrt(8) / sqrt(1 + W_s/W_t), q4[s][t] = (W_t/W_s)^(1/4).
struct XfTransportDev {
  double mu[XF_MAXN][4], kappa[XF_MAXN][4];
  double D[XF_MAXN][XF_MAXN][4];
  double w8[XF_MAXN][XF_MAXN], q4[XF_MAXN][XF_MAXN];
  double W[XF_MAXN];
  double p_ref;
};

// Reaction mechanism in compiled form, a kernel parameter of xf_react.cu (constant bank: every access is warp-uniform): per reaction the reactant and product species
// lists (a coefficient 2 is the species listed twice; at most three entries a side), the Arrhenius parameters of Eq. 11,
// the third-body flag and efficiencies; a7 = the entropy constants of the NASA-7 table (Eq. 12).
#define XF_MAXR XF_MAX_REACTIONS
struct XfMechDev {
  int NR;
  int n_r[XF_MAXR], n_p[XF_MAXR], re[XF_MAXR][3], pr[XF_MAXR][3], third[XF_MAXR];
  double A[XF_MAXR], B[XF_MAXR], E[XF_MAXR];
  double eff[XF_MAXR][XF_MAXN];
  double a7[XF_MAXN], W[XF_MAXN], iW[XF_MAXN];
  double p_atm, Ru;
};

struct XfBc {
  int kind[6];
};

// How a sweep writes its flux divergence: out = alpha*Un + beta*(Us + dt*(acc + div)).
struct XfEpilogue {
  int mode;           // 0: out = div (first sweep of a plain rhs); 1: out = acc + div; 2: RK stage combine;
                      // 3: out = div + alpha/(beta dt) U^n -- the FIRST sweep of a stage with alpha != 0 carries the
                      //    U^n term in the partial residual, so that the last sweep (mode 2 with alpha = 0: out =
                      //    beta (U^s + dt (acc + div))) need not read U^n: the traffic of the three sweeps is balanced
  int has_acc;        // mode 2: whether a previous sweep left a partial rhs in `acc`
  double alpha, beta; // mode 2: stage weights of Eq. 16
  double dt;          // mode 2: time step, used when S_dev == nullptr
  double cfl;         // mode 2: dt = cfl / *S_dev otherwise
  const double *S_dev;
  const double *acc;  // partial rhs of earlier sweeps [Nv][padded]
  const double *Un;   // U^n  [Nv][padded] (mode 2)
  double *out;        // rhs or U^{s+1} [Nv][padded]
  int visc;           // XF_VISC_*: Lambda~ of Eq. 14
  int recon;          // XF_RECON_*: reconstruction of Eq. 15 (host-side dispatch of the kernel instantiation)
  const double *lam_glob;  // GLF: [direction][u-c, u, u+c] global maxima on the device
  // positivity-preserving flux blending (Eq. 17-20; reading R17), set for EVERY sweep of a
  // residual: the limiter guards a forward-Euler step of size dt, dt = pp_cfl / *pp_S if pp_S else pp_dt
  int pp;
  double pp_dt, pp_cfl;
  const double *pp_S;
};

// Tensor maps of the TMA sweeps depend only on (base pointer, number of fields, grid): encoded once and kept in the
// context (three cuTensorMapEncodeTiled calls per sweep launch showed on the 2 M-cell configuration).
struct XfTmapCache {
  struct Entry {
    const void *base;
    int nf, kind;   // kind 0: rank-4 row map of the y/z sweeps, 1: rank-2 span map of the x sweep
    bool ok;        // false: TMA cannot describe this array (odd extents, unaligned base)
    CUtensorMap tm;
  };
  Entry e[32];
  int n, next;
};

// launch helpers implemented per translation unit
// prim: the N + 4 workspace fields p, c, 1/rho, Gamma, chi_1..chi_N ([field][padded cells]); NULL = do
// not store them (xf_primitives), p_out / c_out: optional separate copies of p and c for the caller.
// S_out (may be NULL): max over INTERIOR cells of sum_d (|u_d| + c)/dx_d, reduced with atomicMax into a zeroed double.
// lam_glob (may be NULL; GLF): [3][3] maxima over ALL cells the launch visits of |u_d - c|, |u_d|, |u_d + c|.
int xf_launch_prim(const XfGrid &G, const XfThermo &Th, const double *U, double *T, double *prim, double *p_out,
                   double *c_out, int *status, unsigned long long *itersum, double *S_out, double *lam_glob,
                   cudaStream_t s);
int xf_launch_wavespeed(const XfGrid &G, const XfThermo &Th, const double *U, double *T, double *S_dev, int *status,
                        cudaStream_t s);
// only_dir >= 0: that direction alone (the halo exchange interleaves fill and exchange direction by direction)
int xf_launch_ghosts(const XfGrid &G, int Nv, const XfBc &bc, const double *bc_state_dev, double *U, cudaStream_t s,
                     long *launches, int only_dir = -1);
// halo exchange (xf_halo.cu): doubles per face buffer of direction d; pack (U -> buf) / unpack (buf -> U) of one face
long long xf_halo_count(const XfGrid &G, int Nv, int d);
int xf_launch_halo(const XfGrid &G, int Nv, int d, int side, bool pack, double *U, double *T, double *buf, cudaStream_t s);
int xf_launch_sweep_x(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      XfTmapCache *tc, cudaStream_t s);
int xf_launch_sweep_y(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      XfTmapCache *tc, cudaStream_t s);
int xf_launch_sweep_z(const XfGrid &G, int N, const double *U, const double *prim, const XfEpilogue &E, int *status,
                      XfTmapCache *tc, cudaStream_t s);

// viscous / diffusive terms (xf_visc.cu): the cell table vtab [3 N + 5][padded] from U, T; then out = base + div F_v with
// base = alpha / (beta dt) U^n if `stage` (an XfEpilogue of mode 2 with alpha != 0) is given, else 0
int xf_launch_transport(const XfGrid &G, const XfThermo &Th, const XfTransportDev *tr_dev, const double *U, const double *T,
                        double *vtab, cudaStream_t s);
int xf_launch_viscous(const XfGrid &G, int N, const double *vtab, const double *T, double *out, const XfEpilogue *stage,
                      cudaStream_t s, long *launches);

// reaction step (xf_react.cu): species of the interior cells advanced over dt at fixed rho, rho u, E; T in / out
int xf_launch_react(const XfGrid &G, const XfThermo &Th, const XfMechDev &mech, double *U, double *T, double dt,
                    int n_sub, int n_corr, int *status, cudaStream_t s);

// fp64 reciprocal: MUFU.RCP64H seed (relative error e <= 1e-6) refined as r (1 + e + e^2), which leaves e^3:
// 3 DFMA, measured max relative error 2.2e-16 over 1e-13 .. 1e13.  The path is bound by the fp64 pipe, and an
// IEEE division costs about four times as many pipe slots.
__device__ __forceinline__ double xf_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  return fma(r, fma(e, e, e), r);
}
