// xf_api.cu -- the C ABI of libxf.so (include/xf.h): context, argument checks, launch sequencing.
// Every step of the path runs in the kernels of this directory; nothing here computes on the host.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>

#include <nvtx3/nvToolsExt.h>

#include "xf_common.cuh"

int xf_sweep_x_init();
int xf_sweep_y_init();
int xf_sweep_z_init();
int xf_probe_fp64_launch(int blocks, int threads, int iters, double *sink, cudaStream_t s);

// Scratch of xf_convective_rhs_noalloc (include/xf.h): one array per GPU that loads the library, held until exit.  In
// host code this NAME is a host-side stand-in, not a device address -- see noalloc_scratch() below.
static __device__ __align__(256) double g_noalloc_scratch[XF_NOALLOC_SCRATCH_BYTES / sizeof(double)];

struct xf_ctx {
  XfGrid G;
  XfThermo Th;
  XfBc bc;
  int N, Nv, device;
  int *status_dev;                    // sticky flag word
  unsigned long long *itersum_dev;    // Newton iteration counter of the last xf_primitives launch
  double *bc_state_dev;               // [6][XF_MAXNV]
  double *S_dev;                      // max wave speed scalar used by the host-buffer entry points
  double *lam_glob_dev;               // GLF: [3][3] global maxima of the current residual evaluation
  int visc, recon;                    // XF_VISC_*, XF_RECON_*
  XfTransportDev *tr_dev;             // transport fits (device), or nullptr: no viscous / diffusive terms
  XfMechDev *mech;                // reaction mechanism: HOST copy, handed to the kernel by value (constant bank), or nullptr
  double a7[XF_MAXN], W[XF_MAXN], Ru; // kept for xf_set_mechanism
  int positivity;                     // positivity-preserving flux blending on (Eq. 17-20)
  double rhs_dt;                      // the step the limiter of a bare xf_convective_rhs guards (xf_set_rhs_dt)
  long launches;
  XfTmapCache tmaps;                  // tensor maps of the TMA sweeps, per (base pointer, fields)
  // lazily allocated device mirrors for the *_host entry points
  double *hU, *hT, *hR;
  void *hW;
  // optional per-kernel timing (xf_timing_enable): event pairs recorded around every launch on the caller's stream
  int timing_cap, timing_n;
  cudaEvent_t *ev0, *ev1;
  int *ev_kind;
};

namespace {

// NVTX range around an ABI call (tracing); free when no profiler is attached
struct Range {
  explicit Range(const char *name) { nvtxRangePushA(name); }
  ~Range() { nvtxRangePop(); }
};

struct DeviceGuard {
  int prev;
  bool ok;
  explicit DeviceGuard(int dev) : prev(-1), ok(false) {
    if (cudaGetDevice(&prev) != cudaSuccess) return;
    ok = prev == dev || cudaSetDevice(dev) == cudaSuccess;
    if (prev == dev) prev = -1;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

// Device address of g_noalloc_scratch on `device`, which must be the CURRENT device: asked of the runtime once per
// device and cached (the query allocates nothing; the array came with the module).
constexpr int NOALLOC_MAX_DEVICES = 64;
int noalloc_scratch(int device, double **out) {
  static std::mutex mu;
  static double *ptr[NOALLOC_MAX_DEVICES];
  if (device < 0 || device >= NOALLOC_MAX_DEVICES) return XF_EINVAL;
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[device]) {
    void *p = nullptr;
    if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) return XF_ECUDA;
    ptr[device] = static_cast<double *>(p);
  }
  *out = ptr[device];
  return XF_OK;
}

inline size_t field_bytes(const xf_ctx *c) { return sizeof(double) * (size_t)c->G.cells; }

// Brackets one kernel (or the ghost-fill group) with an event pair when timing is on; free otherwise.
struct Timed {
  xf_ctx *c;
  cudaStream_t s;
  int slot;
  Timed(xf_ctx *ctx, int kind, cudaStream_t st) : c(ctx), s(st), slot(-1) {
    if (c->timing_cap > 0 && c->timing_n < c->timing_cap) {
      slot = c->timing_n++;
      c->ev_kind[slot] = kind;
      cudaEventRecord(c->ev0[slot], s);
    }
  }
  ~Timed() {
    if (slot >= 0) cudaEventRecord(c->ev1[slot], s);
  }
};

void timing_free(xf_ctx *c) {
  for (int q = 0; q < c->timing_cap; ++q) {
    cudaEventDestroy(c->ev0[q]);
    cudaEventDestroy(c->ev1[q]);
  }
  free(c->ev0);
  free(c->ev1);
  free(c->ev_kind);
  c->ev0 = c->ev1 = nullptr;
  c->ev_kind = nullptr;
  c->timing_cap = c->timing_n = 0;
}

int count_active(const XfGrid &G) { return (G.n[0] > 1) + (G.n[1] > 1) + (G.n[2] > 1); }

// ghosts -> primitives -> sweeps.  E_last describes what the LAST active sweep writes (residual or RK combine);
// earlier sweeps accumulate the partial residual in `acc`.
int residual(xf_ctx *c, double *U, double *T, void *work, double *acc, const XfEpilogue &E_last, cudaStream_t s,
             double *S_out = nullptr, bool with_stage_buffers = false, bool skip_fill = false) {
  int rc = XF_OK;
  if (!skip_fill) {   // xf_rk3_stage: the caller has filled / exchanged the ghosts itself
    Timed t(c, XF_K_GHOST, s);
    rc = xf_launch_ghosts(c->G, c->Nv, c->bc, c->bc_state_dev, U, s, &c->launches);
  }
  if (rc != XF_OK) return rc;
  double *prim = static_cast<double *>(work);  // p, c, 1/rho, Gamma, chi_1..chi_N
  {
    Timed t(c, XF_K_PRIM, s);
    rc = xf_launch_prim(c->G, c->Th, U, T, prim, nullptr, nullptr, c->status_dev, nullptr, S_out,
                        c->visc == XF_VISC_GLF ? c->lam_glob_dev : nullptr, s);
  }
  ++c->launches;
  if (rc != XF_OK) return rc;
  const int nact = count_active(c->G);
  int done = 0;
  // Viscous / diffusive terms (context created with a transport table): div F_v goes into the partial-residual buffer
  // first -- with the alpha / (beta dt) U^n term of the stage, which the first sweep would otherwise carry -- and the
  // sweeps accumulate on top of it, so the fused stage combination of the last sweep stays as it is.
  const bool visc = c->tr_dev != nullptr;
  if (visc) {
    double *vtab = prim + (size_t)(c->N + 4) * (size_t)c->G.cells + (with_stage_buffers ? 3 * (size_t)c->Nv * (size_t)c->G.cells : 0);
    {
      Timed t(c, XF_K_TRANSPORT, s);
      rc = xf_launch_transport(c->G, c->Th, c->tr_dev, U, T, vtab, s);
      ++c->launches;
    }
    if (rc != XF_OK) return rc;
    const bool carry_un = E_last.mode == 2 && E_last.alpha != 0.0;
    Timed t(c, XF_K_VISCOUS, s);
    rc = xf_launch_viscous(c->G, c->N, vtab, T, acc, carry_un ? &E_last : nullptr, s, &c->launches);
    if (rc != XF_OK) return rc;
  }
  for (int dd = 0; dd < 3; ++dd) {
    const int d = dd;
    if (c->G.n[d] == 1) continue;
    XfEpilogue E;
    // a stage with alpha != 0 and more than one sweep: the first sweep adds alpha/(beta dt) U^n to the partial
    // residual and the last one no longer reads U^n (XfEpilogue mode 3)
    const bool un_first = E_last.mode == 2 && E_last.alpha != 0.0 && (nact > 1 || visc);
    const bool have_acc = done > 0 || visc;                 // a partial residual is already in `acc`
    if (done == nact - 1) {
      E = E_last;
      E.has_acc = have_acc;
      if (E.mode != 2) E.mode = have_acc ? 1 : 0;
      if (un_first) E.alpha = 0.0;
      E.acc = acc;
    } else {
      memset(&E, 0, sizeof(E));
      E.mode = have_acc ? 1 : 0;
      if (done == 0 && un_first && !visc) {
        E = E_last;
        E.mode = 3;
      }
      E.acc = acc;
      E.out = acc;
    }
    E.visc = c->visc;
    E.recon = c->recon;
    E.lam_glob = c->lam_glob_dev;
    E.pp = c->positivity;       // the limiter guards the forward-Euler step of this stage (or of xf_set_rhs_dt)
    E.pp_dt = E_last.mode == 2 ? E_last.dt : c->rhs_dt;
    E.pp_cfl = E_last.cfl;
    E.pp_S = E_last.mode == 2 ? E_last.S_dev : nullptr;
    Timed t(c, XF_K_SWEEP_X + d, s);
    if (d == 0) rc = xf_launch_sweep_x(c->G, c->N, U, prim, E, c->status_dev, &c->tmaps, s);
    else if (d == 1) rc = xf_launch_sweep_y(c->G, c->N, U, prim, E, c->status_dev, &c->tmaps, s);
    else rc = xf_launch_sweep_z(c->G, c->N, U, prim, E, c->status_dev, &c->tmaps, s);
    ++c->launches;
    if (rc != XF_OK) return rc;
    ++done;
  }
  return XF_OK;
}

// S_out != nullptr: the first stage's primitives kernel reduces the max wave speed of U^n into it (xf_step_cfl)
int rk3(xf_ctx *c, double *U, double *T, double dt, double cfl, const double *S_dev, void *work, cudaStream_t s,
        double *S_out = nullptr) {
  const size_t n = (size_t)c->G.cells;
  double *w = static_cast<double *>(work);
  double *U1 = w + (size_t)(c->N + 4) * n;
  double *U2 = U1 + (size_t)c->Nv * n;
  double *acc = U2 + (size_t)c->Nv * n;
  XfEpilogue E;
  memset(&E, 0, sizeof(E));
  E.mode = 2;
  E.dt = dt;
  E.cfl = cfl;
  E.S_dev = S_dev;
  E.Un = U;
  // Eq. 16: U1 = Un + dt L(Un); U2 = 3/4 Un + 1/4 (U1 + dt L(U1)); Un+1 = 1/3 Un + 2/3 (U2 + dt L(U2))
  E.alpha = 0.0; E.beta = 1.0; E.out = U1;
  int rc = residual(c, U, T, work, acc, E, s, S_out, true);
  if (rc != XF_OK) return rc;
  E.alpha = 0.75; E.beta = 0.25; E.out = U2;
  rc = residual(c, U1, T, work, acc, E, s, nullptr, true);
  if (rc != XF_OK) return rc;
  E.alpha = 1.0 / 3.0; E.beta = 2.0 / 3.0; E.out = U;
  return residual(c, U2, T, work, acc, E, s, nullptr, true);
}

int ensure_host_mirrors(xf_ctx *c) {
  if (c->hU && c->hT && c->hR && c->hW) return XF_OK;
  const size_t fb = field_bytes(c);
  if (cudaMalloc(&c->hU, fb * c->Nv) == cudaSuccess && cudaMalloc(&c->hT, fb) == cudaSuccess &&
      cudaMalloc(&c->hR, fb * c->Nv) == cudaSuccess && cudaMalloc(&c->hW, xf_workspace_bytes(c)) == cudaSuccess)
    return XF_OK;
  cudaFree(c->hU);   // all or nothing: a later call must not find a partial set
  cudaFree(c->hT);
  cudaFree(c->hR);
  cudaFree(c->hW);
  c->hU = c->hT = c->hR = nullptr;
  c->hW = nullptr;
  cudaGetLastError();
  return XF_ENOMEM;
}

}  // namespace

extern "C" {

int xf_create(xf_ctx **out, const xf_config *cfg) {
  if (!out || !cfg) return XF_EINVAL;
  *out = nullptr;
  const int N = cfg->nspecies;
  if (cfg->reconstruction < XF_RECON_WENO5 || cfg->reconstruction > XF_RECON_WENO7) return XF_EINVAL;
  const int ng = cfg->reconstruction == XF_RECON_WENO7 ? 4 : 3;   // half the stencil: i-2..i+3, or i-3..i+4
  if (cfg->ng != ng || N < 1 || N > XF_MAXN || cfg->nx < 1 || cfg->ny < 1 || cfg->nz < 1) return XF_EINVAL;
  if (!cfg->W || !cfg->nasa7 || !(cfg->Ru > 0.0) || !(cfg->Thi > cfg->Tlo)) return XF_EINVAL;
  const int n[3] = {cfg->nx, cfg->ny, cfg->nz};
  const double dxs[3] = {cfg->dx, cfg->dy, cfg->dz};
  for (int d = 0; d < 3; ++d) {
    if (n[d] == 1) continue;
    if (!(dxs[d] > 0.0)) return XF_EINVAL;
    if (n[d] < ng) return XF_EINVAL;  // ghost layers are copies of interior layers: need >= ng of them
    for (int side = 0; side < 2; ++side) {
      const int b = cfg->bc[2 * d + side];
      if (b < XF_BC_PERIODIC || b > XF_BC_EXCHANGE) return XF_EINVAL;
      if (b == XF_BC_DIRICHLET && !cfg->bc_state) return XF_EINVAL;
    }
    if ((cfg->bc[2 * d] == XF_BC_PERIODIC) != (cfg->bc[2 * d + 1] == XF_BC_PERIODIC)) return XF_EINVAL;
  }
  for (int s = 0; s < N; ++s)
    if (!(cfg->W[s] > 0.0)) return XF_EINVAL;
  if (n[0] == 1 && n[1] == 1 && n[2] == 1) return XF_EINVAL;
  if (cfg->viscosity < XF_VISC_LLF || cfg->viscosity > XF_VISC_GLF) return XF_EINVAL;
  if (n[1] > 65535 || n[2] > 65535) return XF_EINVAL;  // they index the y dimension of the y/z sweep grids

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) return XF_ECUDA;
  DeviceGuard guard(cfg->device);
  if (!guard.ok) return XF_ECUDA;

  xf_ctx *c = new (std::nothrow) xf_ctx;
  if (!c) return XF_ENOMEM;
  memset(c, 0, sizeof(*c));
  c->N = N;
  c->Nv = N + 4;
  c->device = cfg->device;
  c->visc = cfg->viscosity;
  c->recon = cfg->reconstruction;
  c->positivity = cfg->positivity != 0;
  XfGrid &G = c->G;
  for (int d = 0; d < 3; ++d) {
    G.n[d] = n[d];
    G.g[d] = n[d] > 1 ? ng : 0;
    G.np[d] = n[d] + 2 * G.g[d];
    G.inv_d[d] = n[d] > 1 ? 1.0 / dxs[d] : 0.0;
  }
  G.st[0] = 1;
  G.st[1] = G.np[0];
  G.st[2] = (long long)G.np[0] * G.np[1];
  G.cells = (long long)G.np[0] * G.np[1] * G.np[2];

  XfThermo &Th = c->Th;
  Th.N = N;
  Th.Tlo = cfg->Tlo;
  Th.Thi = cfg->Thi;
  Th.rtol = cfg->newton_rtol > 0.0 ? cfg->newton_rtol : 1e-13;
  Th.maxit = cfg->newton_maxit > 0 ? cfg->newton_maxit : 50;
  for (int s = 0; s < N; ++s) {
    const double *a = cfg->nasa7 + 7 * s;
    Th.Rs[s] = cfg->Ru / cfg->W[s];
    for (int q = 0; q < 6; ++q) Th.a[s][q] = a[q];
    for (int q = 0; q < 4; ++q) Th.b[s][q] = a[q + 1] / (double)(q + 2);
  }
  for (int q = 0; q < 6; ++q) c->bc.kind[q] = cfg->bc[q];
  for (int s = 0; s < N; ++s) {
    c->a7[s] = cfg->nasa7[7 * s + 6];
    c->W[s] = cfg->W[s];
  }
  c->Ru = cfg->Ru;

  bool ok = cudaMalloc(&c->status_dev, sizeof(int)) == cudaSuccess &&
            cudaMalloc(&c->itersum_dev, sizeof(unsigned long long)) == cudaSuccess &&
            cudaMalloc(&c->bc_state_dev, sizeof(double) * 6 * XF_MAXNV) == cudaSuccess &&
            cudaMalloc(&c->S_dev, sizeof(double)) == cudaSuccess &&
            cudaMalloc(&c->lam_glob_dev, 9 * sizeof(double)) == cudaSuccess;
  if (ok) {
    double bs[6 * XF_MAXNV];
    memset(bs, 0, sizeof(bs));
    if (cfg->bc_state)
      for (int q = 0; q < 6; ++q)
        for (int v = 0; v < c->Nv; ++v) bs[q * XF_MAXNV + v] = cfg->bc_state[q * c->Nv + v];
    ok = cudaMemcpy(c->bc_state_dev, bs, sizeof(bs), cudaMemcpyHostToDevice) == cudaSuccess &&
         cudaMemset(c->status_dev, 0, sizeof(int)) == cudaSuccess &&
         cudaMemset(c->itersum_dev, 0, sizeof(unsigned long long)) == cudaSuccess;
  }
  if (ok && cfg->transport) {   // Eq. 29 fits [N][4] mu, [N][4] kappa, [N][N][4] D_st, p_ref -> evaluation form on the device
    XfTransportDev *h = new (std::nothrow) XfTransportDev;
    ok = h != nullptr;
    if (ok) {
      memset(h, 0, sizeof(*h));
      const double *t = cfg->transport;
      for (int s = 0; s < N; ++s)
        for (int q = 0; q < 4; ++q) {
          h->mu[s][q] = t[4 * s + q];
          h->kappa[s][q] = t[4 * N + 4 * s + q];
        }
      for (int s = 0; s < N; ++s)
        for (int u = 0; u < N; ++u) {
          for (int q = 0; q < 4; ++q) h->D[s][u][q] = t[8 * N + 4 * (s * N + u) + q];
          h->w8[s][u] = 1.0 / sqrt(8.0) / sqrt(1.0 + cfg->W[s] / cfg->W[u]);
          h->q4[s][u] = sqrt(sqrt(cfg->W[u] / cfg->W[s]));
        }
      for (int s = 0; s < N; ++s) h->W[s] = cfg->W[s];
      h->p_ref = t[8 * N + 4 * N * N];
      ok = h->p_ref > 0.0 && cudaMalloc(&c->tr_dev, sizeof(XfTransportDev)) == cudaSuccess &&
           cudaMemcpy(c->tr_dev, h, sizeof(XfTransportDev), cudaMemcpyHostToDevice) == cudaSuccess;
      delete h;
    }
  }
  if (ok) ok = xf_sweep_x_init() == XF_OK && xf_sweep_y_init() == XF_OK && xf_sweep_z_init() == XF_OK;
  if (!ok) {
    xf_destroy(c);
    return XF_ECUDA;
  }
  *out = c;
  return XF_OK;
}

int xf_destroy(xf_ctx *c) {
  if (!c) return XF_EINVAL;
  DeviceGuard guard(c->device);
  cudaFree(c->status_dev);
  cudaFree(c->itersum_dev);
  cudaFree(c->bc_state_dev);
  cudaFree(c->S_dev);
  cudaFree(c->lam_glob_dev);
  cudaFree(c->tr_dev);
  delete c->mech;
  cudaFree(c->hU);
  cudaFree(c->hT);
  cudaFree(c->hR);
  cudaFree(c->hW);
  timing_free(c);
  delete c;
  return XF_OK;
}

size_t xf_num_vars(const xf_ctx *c) { return c ? (size_t)c->Nv : 0; }
size_t xf_padded_cells(const xf_ctx *c) { return c ? (size_t)c->G.cells : 0; }
// workspace layout: [p, c, 1/rho, Gamma, chi_s: N + 4] ([U1, U2, partial residual: 3 Nv] for the RK3 calls) [cell table of
// the viscous terms: 3 N + 5, only with a transport table]
size_t xf_rhs_workspace_bytes(const xf_ctx *c) {
  return c ? field_bytes(c) * (size_t)(c->N + 4 + (c->tr_dev ? 3 * c->N + 5 : 0)) : 0;
}
size_t xf_workspace_bytes(const xf_ctx *c) {
  return c ? field_bytes(c) * (size_t)(c->N + 4 + 3 * c->Nv + (c->tr_dev ? 3 * c->N + 5 : 0)) : 0;
}

int xf_fill_ghosts(xf_ctx *c, double *U, void *stream) {
  if (!c || !U) return XF_EINVAL;
  Range r("xf_fill_ghosts");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  return xf_launch_ghosts(c->G, c->Nv, c->bc, c->bc_state_dev, U, static_cast<cudaStream_t>(stream), &c->launches);
}

int xf_primitives(xf_ctx *c, const double *U, double *T, double *p, double *cs, void *stream) {
  if (!c || !U || !T) return XF_EINVAL;
  Range r("xf_primitives");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (cudaMemsetAsync(c->itersum_dev, 0, sizeof(unsigned long long), s) != cudaSuccess) return XF_ECUDA;
  ++c->launches;
  return xf_launch_prim(c->G, c->Th, U, T, nullptr, p, cs, c->status_dev, c->itersum_dev, nullptr, nullptr, s);
}

int xf_convective_rhs(xf_ctx *c, double *U, double *T, double *rhs, void *work, void *stream) {
  if (!c || !U || !T || !rhs || !work) return XF_EINVAL;
  Range r("xf_convective_rhs");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  XfEpilogue E;
  memset(&E, 0, sizeof(E));
  E.mode = 0;
  E.out = rhs;
  return residual(c, U, T, work, rhs, E, static_cast<cudaStream_t>(stream));
}

int xf_set_mechanism(xf_ctx *c, int n_reactions, const int *nu_r, const int *nu_p, const double *A, const double *B,
                     const double *E, const int *third, const double *eff, double p_atm) {
  if (!c || n_reactions < 1 || n_reactions > XF_MAXR || !nu_r || !nu_p || !A || !B || !E || !third || !eff || !(p_atm > 0.0))
    return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  XfMechDev *h = new (std::nothrow) XfMechDev;
  if (!h) return XF_ENOMEM;
  memset(h, 0, sizeof(*h));
  h->NR = n_reactions;
  const int N = c->N;
  for (int r = 0; r < n_reactions; ++r) {
    for (int s = 0; s < N; ++s) {
      const int a = nu_r[r * N + s], b = nu_p[r * N + s];
      if (a < 0 || b < 0 || h->n_r[r] + a > 3 || h->n_p[r] + b > 3) {   // at most three reactant and three product molecules
        delete h;
        return XF_EINVAL;
      }
      for (int k = 0; k < a; ++k) h->re[r][h->n_r[r]++] = s;
      for (int k = 0; k < b; ++k) h->pr[r][h->n_p[r]++] = s;
      h->eff[r][s] = eff[r * N + s];
    }
    h->A[r] = A[r];
    h->B[r] = B[r];
    h->E[r] = E[r];
    h->third[r] = third[r] != 0;
  }
  for (int s = 0; s < N; ++s) {
    h->a7[s] = c->a7[s];
    h->W[s] = c->W[s];
    h->iW[s] = 1.0 / c->W[s];
  }
  h->p_atm = p_atm;
  h->Ru = c->Ru;
  delete c->mech;
  c->mech = h;
  return XF_OK;
}

int xf_react(xf_ctx *c, double *U, double *T, double dt, int n_sub, int n_corr, void *stream) {
  if (!c || !U || !T || !c->mech || !(dt >= 0.0) || isinf(dt) || n_sub < 1 || n_corr < 1) return XF_EINVAL;
  Range r("xf_react");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  ++c->launches;
  Timed t(c, XF_K_REACT, static_cast<cudaStream_t>(stream));
  return xf_launch_react(c->G, c->Th, *c->mech, U, T, dt, n_sub, n_corr, c->status_dev, static_cast<cudaStream_t>(stream));
}

int xf_fill_ghosts_dir(xf_ctx *c, double *U, int dir, void *stream) {
  if (!c || !U || dir < 0 || dir > 2) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  return xf_launch_ghosts(c->G, c->Nv, c->bc, c->bc_state_dev, U, static_cast<cudaStream_t>(stream), &c->launches, dir);
}

size_t xf_halo_doubles(const xf_ctx *c, int dir) {
  return c && dir >= 0 && dir <= 2 ? (size_t)xf_halo_count(c->G, c->Nv, dir) : 0;
}

int xf_pack_halo(xf_ctx *c, const double *U, const double *T, int dir, int side, double *buf, void *stream) {
  if (!c || !U || !T || !buf || dir < 0 || dir > 2 || side < 0 || side > 1 || c->G.n[dir] == 1) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  ++c->launches;
  return xf_launch_halo(c->G, c->Nv, dir, side, true, const_cast<double *>(U), const_cast<double *>(T), buf,
                        static_cast<cudaStream_t>(stream));
}

int xf_unpack_halo(xf_ctx *c, double *U, double *T, int dir, int side, const double *buf, void *stream) {
  if (!c || !U || !T || !buf || dir < 0 || dir > 2 || side < 0 || side > 1 || c->G.n[dir] == 1) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  ++c->launches;
  return xf_launch_halo(c->G, c->Nv, dir, side, false, U, T, const_cast<double *>(buf), static_cast<cudaStream_t>(stream));
}

int xf_rk3_stage(xf_ctx *c, int stage, const double *Un, double *Uin, double *Uout, double *T, double dt, void *work,
                 void *stream) {
  if (!c || !Un || !Uin || !Uout || !T || !work || stage < 0 || stage > 2 || !(dt > 0.0) || isinf(dt)) return XF_EINVAL;
  Range r("xf_rk3_stage");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  const size_t n = (size_t)c->G.cells;
  double *acc = static_cast<double *>(work) + (size_t)(c->N + 4) * n + 2 * (size_t)c->Nv * n;   // as in xf_rk3_step
  static const double al[3] = {0.0, 0.75, 1.0 / 3.0}, be[3] = {1.0, 0.25, 2.0 / 3.0};   // Eq. 16
  XfEpilogue E;
  memset(&E, 0, sizeof(E));
  E.mode = 2;
  E.dt = dt;
  E.Un = Un;
  E.alpha = al[stage];
  E.beta = be[stage];
  E.out = Uout;
  return residual(c, Uin, T, work, acc, E, static_cast<cudaStream_t>(stream), nullptr, true, true);
}

int xf_viscous_rhs(xf_ctx *c, const double *U, const double *T, double *rhs, void *work, void *stream) {
  if (!c || !U || !T || !rhs || !work || !c->tr_dev) return XF_EINVAL;
  Range r("xf_viscous_rhs");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  double *vtab = static_cast<double *>(work) + (size_t)(c->N + 4) * (size_t)c->G.cells;
  int rc;
  {
    Timed t(c, XF_K_TRANSPORT, s);
    rc = xf_launch_transport(c->G, c->Th, c->tr_dev, U, T, vtab, s);
    ++c->launches;
  }
  if (rc != XF_OK) return rc;
  Timed t(c, XF_K_VISCOUS, s);
  return xf_launch_viscous(c->G, c->N, vtab, T, rhs, nullptr, s, &c->launches);
}

int xf_set_rhs_dt(xf_ctx *c, double dt) {
  if (!c || !(dt >= 0.0) || isinf(dt)) return XF_EINVAL;
  c->rhs_dt = dt;
  return XF_OK;
}

int xf_rk3_step(xf_ctx *c, double *U, double *T, double dt, void *work, void *stream) {
  if (!c || !U || !T || !work || !(dt > 0.0) || isinf(dt)) return XF_EINVAL;   // dt = 0, negative, inf, NaN
  Range r("xf_rk3_step");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  return rk3(c, U, T, dt, 0.0, nullptr, work, static_cast<cudaStream_t>(stream));
}

int xf_rk3_step_cfl(xf_ctx *c, double *U, double *T, double cfl, const double *S_dev, void *work, void *stream) {
  if (!c || !U || !T || !work || !S_dev || !(cfl > 0.0)) return XF_EINVAL;
  Range r("xf_rk3_step_cfl");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  return rk3(c, U, T, 0.0, cfl, S_dev, work, static_cast<cudaStream_t>(stream));
}

int xf_step_cfl(xf_ctx *c, double *U, double *T, double cfl, double *S_dev, void *work, void *stream) {
  if (!c || !U || !T || !work || !S_dev || !(cfl > 0.0)) return XF_EINVAL;
  Range r("xf_step_cfl");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  return rk3(c, U, T, 0.0, cfl, S_dev, work, static_cast<cudaStream_t>(stream), S_dev);
}

int xf_max_wavespeed(xf_ctx *c, const double *U, double *T, double *S_dev, void *stream) {
  if (!c || !U || !T || !S_dev) return XF_EINVAL;
  Range r("xf_max_wavespeed");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  ++c->launches;
  Timed t(c, XF_K_WAVESPEED, static_cast<cudaStream_t>(stream));
  return xf_launch_wavespeed(c->G, c->Th, U, T, S_dev, c->status_dev, static_cast<cudaStream_t>(stream));
}

int xf_status(xf_ctx *c, void *stream) {
  if (!c) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int flag = 0;
  if (cudaMemcpyAsync(&flag, c->status_dev, sizeof(int), cudaMemcpyDeviceToHost, s) != cudaSuccess) return XF_ECUDA;
  if (cudaMemsetAsync(c->status_dev, 0, sizeof(int), s) != cudaSuccess) return XF_ECUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return XF_ECUDA;
  if (flag & XF_FLAG_NONPHYSICAL) return XF_ENONPHYSICAL;
  if (flag & XF_FLAG_NOCONV) return XF_ENOCONV;
  return XF_OK;
}

int xf_newton_mean_iterations(xf_ctx *c, void *stream, double *mean_out) {
  if (!c || !mean_out) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  unsigned long long sum = 0;
  if (cudaMemcpyAsync(&sum, c->itersum_dev, sizeof(sum), cudaMemcpyDeviceToHost, s) != cudaSuccess) return XF_ECUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return XF_ECUDA;
  *mean_out = (double)sum / (double)c->G.cells;
  return XF_OK;
}

long xf_launch_count(const xf_ctx *c) { return c ? c->launches : 0; }

int xf_timing_enable(xf_ctx *c, int max_records) {
  if (!c || max_records < 0) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  timing_free(c);
  if (max_records == 0) return XF_OK;
  c->ev0 = static_cast<cudaEvent_t *>(calloc(max_records, sizeof(cudaEvent_t)));
  c->ev1 = static_cast<cudaEvent_t *>(calloc(max_records, sizeof(cudaEvent_t)));
  c->ev_kind = static_cast<int *>(calloc(max_records, sizeof(int)));
  if (!c->ev0 || !c->ev1 || !c->ev_kind) {
    timing_free(c);
    return XF_ENOMEM;
  }
  for (int q = 0; q < max_records; ++q) {
    if (cudaEventCreate(&c->ev0[q]) != cudaSuccess || cudaEventCreate(&c->ev1[q]) != cudaSuccess) {
      c->timing_cap = q;
      timing_free(c);
      return XF_ECUDA;
    }
    c->timing_cap = q + 1;
  }
  return XF_OK;
}

int xf_timing_read(xf_ctx *c, void *stream, double *ms_out, long *count_out) {
  if (!c || !ms_out || !count_out) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  if (cudaStreamSynchronize(static_cast<cudaStream_t>(stream)) != cudaSuccess) return XF_ECUDA;
  for (int k = 0; k < XF_K_COUNT; ++k) {
    ms_out[k] = 0.0;
    count_out[k] = 0;
  }
  for (int q = 0; q < c->timing_n; ++q) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->ev0[q], c->ev1[q]) != cudaSuccess) return XF_ECUDA;
    ms_out[c->ev_kind[q]] += (double)ms;
    ++count_out[c->ev_kind[q]];
  }
  c->timing_n = 0;
  return XF_OK;
}

int xf_convective_rhs_host(xf_ctx *c, const double *U_host, double *T_host, double *rhs_host) {
  if (!c || !U_host || !T_host || !rhs_host) return XF_EINVAL;
  Range r("xf_convective_rhs_host");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  int rc = ensure_host_mirrors(c);
  if (rc != XF_OK) return rc;
  const size_t fb = field_bytes(c);
  cudaStream_t s = nullptr;
  if (cudaMemcpyAsync(c->hU, U_host, fb * c->Nv, cudaMemcpyHostToDevice, s) != cudaSuccess) return XF_ECUDA;
  if (cudaMemcpyAsync(c->hT, T_host, fb, cudaMemcpyHostToDevice, s) != cudaSuccess) return XF_ECUDA;
  if (cudaMemsetAsync(c->hR, 0, fb * c->Nv, s) != cudaSuccess) return XF_ECUDA;
  XfEpilogue E;
  memset(&E, 0, sizeof(E));
  E.out = c->hR;
  rc = residual(c, c->hU, c->hT, c->hW, c->hR, E, s);
  if (rc != XF_OK) return rc;
  if (cudaMemcpyAsync(rhs_host, c->hR, fb * c->Nv, cudaMemcpyDeviceToHost, s) != cudaSuccess) return XF_ECUDA;
  if (cudaMemcpyAsync(T_host, c->hT, fb, cudaMemcpyDeviceToHost, s) != cudaSuccess) return XF_ECUDA;
  return cudaStreamSynchronize(s) == cudaSuccess ? XF_OK : XF_ECUDA;
}

int xf_rk3_steps_host(xf_ctx *c, double *U_host, double *T_host, double cfl, int nsteps, double *t_advanced) {
  if (!c || !U_host || !T_host || !(cfl > 0.0) || nsteps < 0) return XF_EINVAL;
  Range r("xf_rk3_steps_host");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  int rc = ensure_host_mirrors(c);
  if (rc != XF_OK) return rc;
  const size_t fb = field_bytes(c);
  cudaStream_t s = nullptr;
  if (cudaMemcpyAsync(c->hU, U_host, fb * c->Nv, cudaMemcpyHostToDevice, s) != cudaSuccess) return XF_ECUDA;
  if (cudaMemcpyAsync(c->hT, T_host, fb, cudaMemcpyHostToDevice, s) != cudaSuccess) return XF_ECUDA;
  double t = 0.0;
  for (int k = 0; k < nsteps; ++k) {
    rc = rk3(c, c->hU, c->hT, 0.0, cfl, c->S_dev, c->hW, s, c->S_dev);
    if (rc != XF_OK) return rc;
    if (t_advanced) {
      double S = 0.0;
      if (cudaMemcpyAsync(&S, c->S_dev, sizeof(double), cudaMemcpyDeviceToHost, s) != cudaSuccess) return XF_ECUDA;
      if (cudaStreamSynchronize(s) != cudaSuccess) return XF_ECUDA;
      t += cfl / S;
    }
  }
  if (cudaMemcpyAsync(U_host, c->hU, fb * c->Nv, cudaMemcpyDeviceToHost, s) != cudaSuccess) return XF_ECUDA;
  if (cudaMemcpyAsync(T_host, c->hT, fb, cudaMemcpyDeviceToHost, s) != cudaSuccess) return XF_ECUDA;
  if (cudaStreamSynchronize(s) != cudaSuccess) return XF_ECUDA;
  if (t_advanced) *t_advanced = t;
  return XF_OK;
}

int xf_probe_fp64_peak(int device, int iters, double *tflops, double *ms_out) {
  if (!tflops || iters < 1) return XF_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return XF_ECUDA;
  DeviceGuard guard(device);
  if (!guard.ok) return XF_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return XF_ECUDA;
  const int threads = 256, blocks = prop.multiProcessorCount * 8;
  double *sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double) * (size_t)blocks * threads) != cudaSuccess) return XF_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  int rc = xf_probe_fp64_launch(blocks, threads, iters / 8 + 1, sink, nullptr);  // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 5 && rc == XF_OK; ++rep) {
    cudaEventRecord(e0, nullptr);
    rc = xf_probe_fp64_launch(blocks, threads, iters, sink, nullptr);
    cudaEventRecord(e1, nullptr);
    if (cudaEventSynchronize(e1) != cudaSuccess) rc = XF_ECUDA;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (rc != XF_OK) return rc;
  // 16 independent chains x 8 FMAs per round x 2 flops
  const double flops = 2.0 * 16.0 * 8.0 * (double)iters * (double)blocks * (double)threads;
  *tflops = flops / ((double)best * 1e-3) * 1e-12;
  if (ms_out) *ms_out = best;
  return XF_OK;
}

int xf_probe_fp64_sustained(int device, double seconds, double *tflops, double *ms_out) {
  if (!tflops || !(seconds > 0.0) || seconds > 30.0) return XF_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return XF_ECUDA;
  DeviceGuard guard(device);
  if (!guard.ok) return XF_ECUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return XF_ECUDA;
  const int threads = 256, blocks = prop.multiProcessorCount * 8, iters = 40000;   // one launch: about 90 ms
  double *sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double) * (size_t)blocks * threads) != cudaSuccess) return XF_ENOMEM;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  int rc = xf_probe_fp64_launch(blocks, threads, iters, sink, nullptr);   // warm-up, and the length of one launch
  cudaEventRecord(e0, nullptr);
  if (rc == XF_OK) rc = xf_probe_fp64_launch(blocks, threads, iters, sink, nullptr);
  cudaEventRecord(e1, nullptr);
  if (cudaEventSynchronize(e1) != cudaSuccess) rc = XF_ECUDA;
  float one = 0.f;
  cudaEventElapsedTime(&one, e0, e1);
  const int n = one > 0.f ? (int)(seconds * 1e3 / one) + 1 : 1;
  cudaEventRecord(e0, nullptr);
  for (int q = 0; q < n && rc == XF_OK; ++q) rc = xf_probe_fp64_launch(blocks, threads, iters, sink, nullptr);
  cudaEventRecord(e1, nullptr);
  if (cudaEventSynchronize(e1) != cudaSuccess) rc = XF_ECUDA;
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  if (rc != XF_OK) return rc;
  *tflops = 2.0 * 16.0 * 8.0 * (double)iters * (double)blocks * (double)threads * (double)n / ((double)ms * 1e-3) * 1e-12;
  if (ms_out) *ms_out = ms;
  return XF_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// The no-allocation entry point (include/xf.h: xf_convective_rhs_noalloc).  g_noalloc_scratch (file scope, below the
// includes) is the HOST-side stand-in of the device array: host code never passes it to a kernel; it asks the runtime
// for the array's address on the current device, once per device, and passes that.
// ---------------------------------------------------------------------------------------------------------------
size_t xf_noalloc_scratch_bytes(void) { return XF_NOALLOC_SCRATCH_BYTES; }

int xf_noalloc_prepare(xf_ctx *c) {
  if (!c) return XF_EINVAL;
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  double *ptr = nullptr;
  return noalloc_scratch(c->device, &ptr);
}

int xf_convective_rhs_noalloc(xf_ctx *c, double *U, double *T, double *rhs, void *stream) {
  if (!c || !U || !T || !rhs) return XF_EINVAL;
  if (xf_rhs_workspace_bytes(c) > (size_t)XF_NOALLOC_SCRATCH_BYTES) return XF_ETOOBIG;
  Range r("xf_convective_rhs_noalloc");
  DeviceGuard guard(c->device);
  if (!guard.ok) return XF_ECUDA;
  double *scratch = nullptr;
  const int rc = noalloc_scratch(c->device, &scratch);   // cached after the first call for this device
  if (rc != XF_OK) return rc;
  XfEpilogue E;
  memset(&E, 0, sizeof(E));
  E.mode = 0;
  E.out = rhs;
  return residual(c, U, T, scratch, rhs, E, static_cast<cudaStream_t>(stream));
}

const char *xf_strerror(int code) {
  switch (code) {
    case XF_OK: return "ok";
    case XF_EINVAL: return "invalid argument";
    case XF_ECUDA: return "CUDA error (no device, bad device ordinal or launch failure)";
    case XF_ENOMEM: return "out of device memory";
    case XF_ENONPHYSICAL: return "non-physical state on the device (NaN or rho, p, T <= 0)";
    case XF_ENOCONV: return "Newton iteration for T(e) did not converge";
    case XF_ETOOBIG: return "problem exceeds the static scratch of the no-allocation entry point (XF_NOALLOC_SCRATCH_BYTES)";
    default: return "unknown error";
  }
}

}  // extern "C"
