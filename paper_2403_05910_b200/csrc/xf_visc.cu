// xf_visc.cu -- viscous / diffusive right-hand side div F_v for sm_100a (Eq. 1-6,
// PAPER.md:155-178 Eq. 22 and 26, Eq. 29, "central 4th-order accuracy scheme" PAPER.md:107; readings
// R19-R23 of DESIGN.md).  Two kernels:
//
//   transport_kernel   one thread per padded cell: u, v, w, Y_s, h_s(T), and the mixture transport coefficients from the
//                      fitted ln-polynomials (Eq. 29) -- Wilke's rule for mu and kappa (Eq. 22), rho D_sm (Eq. 26) -- into
//                      the cell table vtab [3 N + 5 fields][padded cells].  This is where the exponentials, square roots
//                      and the O(N^2) pair sums live.
//   visc_dir_kernel    one launch per active direction d: a block owns a tile of LD cells along d (x LT lanes along i);
//                      each thread computes ONE face flux F_v (fourth-order face operators of reading R22: normal
//                      derivative, face value, face value of the cell-centred transverse derivatives) into shared memory,
//                      then the cells of the tile take the fourth-order divergence (27 (F_{+1/2} - F_{-1/2}) - (F_{+3/2} -
//                      F_{-3/2}))/(24 dx) of the LD + 3 faces and add it to the residual.  A face flux never reaches HBM.
//
// HBM-bound (stencil reads of the cell table through L1/L2), unlike the convective sweeps.  No tensor cores: nothing
// here is a contraction.  No code is shared with oracle/.
#include "xf_common.cuh"

namespace {

// vtab field order
constexpr int VT_U = 0, VT_MU = 3, VT_KAPPA = 4, VT_Y = 5;
__host__ __device__ constexpr int vt_h(int N) { return 5 + N; }
__host__ __device__ constexpr int vt_rd(int N) { return 5 + 2 * N; }

__device__ __forceinline__ double fit_eval(const double *a, double lnT) {   // Eq. 29
  return exp(fma(lnT, fma(lnT, fma(lnT, a[3], a[2]), a[1]), a[0]));
}

// Per-thread arrays live in shared memory ([species][thread]: conflict-free, indexable by a runtime species number) and
// the transport table is copied there once per block.  What is unrolled and what is not was measured on config 4
// (N = 10): everything unrolled (45 + 20 exponentials inline) took 255 registers, spilled and ran 27.8 ms; everything
// rolled with the table in global memory 15.4 ms at 81 % of the L1 throughput (four memory operations per five fp64
// ones in the pair loops); table in shared memory, the t side of Wilke's pair loop in registers with the s loop rolled,
// and the symmetric 1/D_st pair loop unrolled with its denominators in registers: 10.9 ms at 92 registers.
// Round 2, from the ncu source page (17 % of the warp samples sat on the species loads, a rolled loop of N - 1 DRAM round
// trips; 10 % on the block's copy of the 13 KB table): every global operand of the cell is requested first and the
// table copy overlaps it, 1 / W_s once per block, 256 threads per block (half as many table copies): 11.1 -> 9.35 ms.
// Tried and dropped: persistent blocks with a grid-stride loop (the compiler then keeps 164 registers or spills: 12.6 ms).
constexpr int TR_THREADS = 256;
template <int N_T>
__global__ void __launch_bounds__(TR_THREADS)
transport_kernel(const XfGrid G, const __grid_constant__ XfThermo th, const XfTransportDev *__restrict__ tr_glob,
                 const double *__restrict__ U, const double *__restrict__ T, double *__restrict__ vtab) {
  const int N = N_T > 0 ? N_T : th.N;
  // shared memory: a copy of the transport table (its coefficients are read at warp-uniform addresses inside the pair
  // loops: broadcast LDS instead of one L1 transaction per coefficient -- the kernel sat at 81 % of the L1 throughput
  // with the table in global memory), then X, a, sq, isq: 4 arrays [N][TR_THREADS]; den reuses sq
  extern __shared__ double sh[];
  constexpr int TBL = (int)(sizeof(XfTransportDev) / sizeof(double));
  double *X = sh + TBL + XF_MAXN + threadIdx.x, *a = X + N * TR_THREADS, *sq = a + N * TR_THREADS, *isq = sq + N * TR_THREADS;
  double *den = sq;
#define AT(arr, s) arr[(s) * TR_THREADS]
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long C = G.cells;
  const bool live = idx < C;
  // Every global operand of the cell is requested before the block's copy of the table: as a rolled loop the species
  // loads were N - 1 DRAM round trips in a row (17 % of the warp samples), and the table copy another one (10 %).
  double rho = 1.0, Tk = 300.0;
  if (live) {
    rho = U[idx];
    Tk = T[idx];
    if constexpr (N_T > 0) {
#pragma unroll
      for (int s = 0; s < N_T - 1; ++s) AT(X, s) = U[(5 + s) * C + idx];
    }
  }
  for (int q = threadIdx.x; q < TBL; q += TR_THREADS) sh[q] = reinterpret_cast<const double *>(tr_glob)[q];
  if (threadIdx.x < N) sh[TBL + threadIdx.x] = 1.0 / reinterpret_cast<const XfTransportDev *>(tr_glob)->W[threadIdx.x];
  __syncthreads();
  const XfTransportDev *tr = reinterpret_cast<const XfTransportDev *>(sh);
  const double *iW = sh + TBL;                                     // 1 / W_s: N divisions per block, not per cell
  if (!live) return;
  const double rinv = 1.0 / rho;
#pragma unroll
  for (int q = 0; q < 3; ++q) vtab[(VT_U + q) * C + idx] = U[(1 + q) * C + idx] * rinv;
  double sumY = 0.0, sumYW = 0.0, Rbar = 0.0;
  for (int s = 0; s < N; ++s) {
    const double Y = s < N - 1 ? (N_T > 0 ? AT(X, s) : U[(5 + s) * C + idx]) * rinv : 1.0 - sumY;   // closure, no clipping (reading R12)
    sumY += Y;
    vtab[(VT_Y + s) * C + idx] = Y;
    const double x = Y * iW[s];
    AT(X, s) = x;
    sumYW += x;
    Rbar = fma(Y, th.Rs[s], Rbar);
  }
  const double lnT = log(Tk);
  const double p = rho * Rbar * Tk;   // Eq. 7
  const double isum = 1.0 / sumYW;
  double Wbar = 0.0;
  for (int s = 0; s < N; ++s) {
    const double x = AT(X, s) * isum;
    AT(X, s) = x;
    Wbar = fma(x, tr->W[s], Wbar);
  }
  // ---- species enthalpies h_s(T) (NASA polynomials with the constant-cp continuation, reading R3)
  const double Tc = fmin(fmax(Tk, th.Tlo), th.Thi);
  for (int s = 0; s < N; ++s) {
    const double *ca = th.a[s], *cb = th.b[s];
    const double hp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, cb[3], cb[2]), cb[1]), cb[0]), ca[0]);
    const double cp = fma(Tc, fma(Tc, fma(Tc, fma(Tc, ca[4], ca[3]), ca[2]), ca[1]), ca[0]);
    vtab[(vt_h(N) + s) * C + idx] = th.Rs[s] * fma(cp, Tk - Tc, fma(Tc, hp, ca[5]));
  }
  // ---- Wilke's rule (Eq. 22), once for mu and once for kappa: sqrt(a_s / a_t) = sqrt(a_s) / sqrt(a_t)
#pragma unroll 1
  for (int which = 0; which < 2; ++which) {
    for (int s = 0; s < N; ++s) {
      const double v = fit_eval(which == 0 ? tr->mu[s] : tr->kappa[s], lnT);
      const double ir = rsqrt(v);
      AT(a, s) = v;
      AT(sq, s) = v * ir;
      AT(isq, s) = ir;
    }
    double mix = 0.0;
    if constexpr (N_T > 0) {   // the t-side operands in registers, the t loop unrolled, the s loop rolled
      double Xr[N_T], ir[N_T];
#pragma unroll
      for (int t = 0; t < N_T; ++t) {
        Xr[t] = AT(X, t);
        ir[t] = AT(isq, t);
      }
#pragma unroll 1
      for (int s = 0; s < N_T; ++s) {
        double dn = 0.0;
        const double sqs = AT(sq, s);
#pragma unroll
        for (int t = 0; t < N_T; ++t) {
          const double bb = fma(sqs * ir[t], tr->q4[s][t], 1.0);
          dn = fma(Xr[t] * tr->w8[s][t], bb * bb, dn);
        }
        mix = fma(AT(X, s) * AT(a, s), xf_rcp(dn), mix);
      }
    } else {
#pragma unroll 1
      for (int s = 0; s < N; ++s) {
        double dn = 0.0;
        const double sqs = AT(sq, s);
        for (int t = 0; t < N; ++t) {
          const double bb = fma(sqs * AT(isq, t), tr->q4[s][t], 1.0);
          dn = fma(AT(X, t) * tr->w8[s][t], bb * bb, dn);
        }
        mix = fma(AT(X, s) * AT(a, s), xf_rcp(dn), mix);
      }
    }
    vtab[(which == 0 ? VT_MU : VT_KAPPA) * C + idx] = mix;
  }
  // ---- rho D_sm (Eq. 26 with X_t + 1e-12, reading R20; D_st(T, p) = D_st(T, p_ref) p_ref / p, reading R19)
  const double pscale = p / tr->p_ref;
  // numerator of Eq. 26: sum_{t != s} (X_t + eps) W_t = (the sum over all t) - its own term
  double wsum = 0.0;
  for (int t = 0; t < N; ++t) wsum = fma(AT(X, t) + 1e-12, tr->W[t], wsum);
  if constexpr (N_T > 0) {   // the N (N - 1)/2 pair terms unrolled, the denominators in registers
    double xe[N_T], dn[N_T];
#pragma unroll
    for (int t = 0; t < N_T; ++t) {
      xe[t] = AT(X, t) + 1e-12;
      dn[t] = 0.0;
    }
#pragma unroll
    for (int s = 0; s < N_T; ++s)
#pragma unroll
      for (int t = s + 1; t < N_T; ++t) {
        const double *c = tr->D[s][t];
        const double invD = pscale * exp(-fma(lnT, fma(lnT, fma(lnT, c[3], c[2]), c[1]), c[0]));   // 1 / D_st, symmetric
        dn[s] = fma(xe[t], invD, dn[s]);
        dn[t] = fma(xe[s], invD, dn[t]);
      }
#pragma unroll
    for (int s = 0; s < N_T; ++s)
      vtab[(vt_rd(N) + s) * C + idx] = N > 1 ? rho * fma(-xe[s], tr->W[s], wsum) * xf_rcp(Wbar * dn[s]) : 0.0;
  } else {
    for (int s = 0; s < N; ++s) AT(den, s) = 0.0;
#pragma unroll 1
    for (int s = 0; s < N; ++s) {
      const double xs = AT(X, s) + 1e-12;
      double ds = AT(den, s);
      for (int t = s + 1; t < N; ++t) {
        const double *c = tr->D[s][t];
        const double invD = pscale * exp(-fma(lnT, fma(lnT, fma(lnT, c[3], c[2]), c[1]), c[0]));
        ds = fma(AT(X, t) + 1e-12, invD, ds);
        AT(den, t) = fma(xs, invD, AT(den, t));
      }
      vtab[(vt_rd(N) + s) * C + idx] = N > 1 ? rho * fma(-xs, tr->W[s], wsum) * xf_rcp(Wbar * ds) : 0.0;
    }
  }
#undef AT
}

__device__ __forceinline__ double interp4(double m1, double a, double b, double p2) {
  return (9.0 * (a + b) - (m1 + p2)) * (1.0 / 16.0);
}

struct ViscArgs {
  const double *vtab, *T;
  double *out;
  const double *Un;        // base term kappa_un * U^n of the FIRST launch of a residual evaluation (or nullptr)
  double alpha, beta, dt, cfl;
  const double *S_dev;     // dt = cfl / *S_dev if set (the device-side time step of xf_step_cfl)
  int first;               // 1: out = base + div, 0: out += div
  int seg;                 // cells along d per block
};

#ifndef XF_VISC_LT
#define XF_VISC_LT 16   // lanes along i of a y / z tile (a warp = two rows of 128 bytes)
#define XF_VISC_MINB 4
#endif
#ifndef XF_VISC_PREFETCH
#define XF_VISC_PREFETCH 1
#endif
// DIR = 0: block = LDF threads along i, one face each, LDF - 3 cells; DIR = 1, 2: block = 32 lanes along i x LDF face rows
template <int N_T, int DIR, int LDF>
__global__ void __launch_bounds__(DIR == 0 ? LDF : XF_VISC_LT * LDF, XF_VISC_MINB)
visc_dir_kernel(const XfGrid G, const int Nrt, const ViscArgs A) {
  constexpr int NS = N_T > 0 ? N_T : XF_MAXN;
  const int N = N_T > 0 ? N_T : Nrt, Nv = N + 4;
  constexpr int LT = DIR == 0 ? 1 : XF_VISC_LT, LD = LDF - 3;
  extern __shared__ double fs[];                                  // [Nv - 1][LDF][LT]
  const long long C = G.cells;
  const int k = DIR == 0 ? threadIdx.x : threadIdx.y;             // face index within the tile
  const int lt = DIR == 0 ? 0 : threadIdx.x;
  // tile origin: first cell along d (interior numbering), the transverse position
  int c0, i, j2;                                                  // j2: index along the remaining transverse direction
  if (DIR == 0) {
    c0 = blockIdx.x * LD;
    i = 0;
    j2 = 0;
  } else {
    c0 = blockIdx.y * LD;
    i = blockIdx.x * LT + lt;
    j2 = blockIdx.z;
  }
  const bool lane_ok = DIR == 0 || i < G.n[0];
  long long base;                                                 // padded index of the pencil's cell 0 along d
  if (DIR == 0) base = (long long)(blockIdx.y + G.g[1]) * G.st[1] + (long long)(blockIdx.z + G.g[2]) * G.st[2];
  else if (DIR == 1) base = (long long)(G.g[0] + (lane_ok ? i : 0)) + (long long)(j2 + G.g[2]) * G.st[2];
  else base = (long long)(G.g[0] + (lane_ok ? i : 0)) + (long long)(j2 + G.g[1]) * G.st[1];
  const long long sd = G.st[DIR];
  const int n = G.n[DIR], g = G.g[DIR];
#if XF_VISC_PREFETCH
  // ---- the tile's lines of the cell table are asked into L2 before the first face needs them: a face issues ~250 loads
  //      and a thread holds a dozen of them in flight, so without this every species pays a DRAM round trip of its own
  //      (config 4, three launches: 17.9 -> 15.7 ms; also asking for the transverse neighbour rows of u, v, w and for
  //      the residual rows cost more than it gave: 18.5 ms)
  {
    const int tid = DIR == 0 ? threadIdx.x : threadIdx.y * LT + threadIdx.x;
    constexpr int NTH = DIR == 0 ? LDF : LT * LDF;
    const int nf = 3 * N + 6;                                     // the cell table and T
    const int r0 = c0 - 3 > -g ? c0 - 3 : -g, r1 = c0 + LD + 2 < n + g - 1 ? c0 + LD + 2 : n + g - 1;
    if (DIR == 0) {                                               // cells r0 .. r1 of one row: consecutive doubles
      const long long q0 = base + g + r0;
      const int span = r1 - r0, nl = span / 16 + 2;               // 128-byte lines (one more: the row starts anywhere in a line)
      for (int it = tid; it < nf * nl; it += NTH) {
        const int f = it / nl, l = it - f * nl;
        const long long q = q0 + (l * 16 < span ? l * 16 : span);
        const double *ptr = f < nf - 1 ? A.vtab + f * C + q : A.T + q;
        asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
      }
    } else {                                                      // rows r0 .. r1, LT lanes: first and last lane of each row
      const int i0 = blockIdx.x * LT, i1 = i0 + LT - 1 < G.n[0] - 1 ? i0 + LT - 1 : G.n[0] - 1;
      const long long b0 = base - (lane_ok ? i : 0);              // padded index of the pencil of lane i = 0
      const int nr = r1 - r0 + 1;
      for (int it = tid; it < nf * nr * 2; it += NTH) {
        const int f = it / (nr * 2), rem = it - f * nr * 2, r = rem >> 1;
        const long long q = b0 + ((rem & 1) ? i1 : i0) + (long long)(g + r0 + r) * sd;
        const double *ptr = f < nf - 1 ? A.vtab + f * C + q : A.T + q;
        asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
      }
    }
  }
#endif
  const int a = c0 - 2 + k;                                       // interior number of the cell below this thread's face
  if (lane_ok && a <= n && a >= -2) {                             // faces above cells -2 .. n (reading R22)
    const long long ia = base + (long long)(g + a) * sd;
    const long long q0 = ia - sd, q1 = ia, q2 = ia + sd, q3 = ia + 2 * sd;
    const double *V = A.vtab;
    const double in = G.inv_d[DIR] * (1.0 / 24.0);
    // every load of the cell table goes through the read-only path (__ldg): the table is a generic pointer inside a
    // struct, and without this the compiler must keep each load behind the previous shared-memory store of a flux
    // component -- one or two loads in flight per thread on a kernel that is bound by memory latency
#define VL(f, q) __ldg(V + (f) * C + (q))
#define FACE(f) interp4(VL(f, q0), VL(f, q1), VL(f, q2), VL(f, q3))
#define DN(f) ((27.0 * (VL(f, q2) - VL(f, q1)) - (VL(f, q3) - VL(f, q0))) * in)
    double Gr[3][3];                                              // Gr[p][e] = d u_p / d x_e at the face
#pragma unroll
    for (int p = 0; p < 3; ++p) {
#pragma unroll
      for (int e = 0; e < 3; ++e) {
        if (e == DIR) Gr[p][e] = DN(VT_U + p);
        else if (G.n[e] == 1) Gr[p][e] = 0.0;
        else {
          const long long se = G.st[e];
          const double ie = G.inv_d[e] * (1.0 / 12.0);
          const double *u = V + (VT_U + p) * C;
          double t[4];
#pragma unroll
          for (int m = 0; m < 4; ++m) {
            const long long z = ia + (long long)(m - 1) * sd;
            t[m] = ((__ldg(u + z - 2 * se) - __ldg(u + z + 2 * se)) - 8.0 * (__ldg(u + z - se) - __ldg(u + z + se))) * ie;
          }
          Gr[p][e] = interp4(t[0], t[1], t[2], t[3]);
        }
      }
    }
    const double mu = FACE(VT_MU), kappa = FACE(VT_KAPPA);
    const double div = Gr[0][0] + Gr[1][1] + Gr[2][2];
    double work = 0.0;
#pragma unroll
    for (int p = 0; p < 3; ++p) {                                 // tau_{p d}, Eq. 3
      const double tau = mu * (Gr[p][DIR] + Gr[DIR][p]) - (p == DIR ? (2.0 / 3.0) * mu * div : 0.0);
      fs[(p * LDF + k) * LT + lt] = tau;
      work = fma(tau, FACE(VT_U + p), work);
    }
    double tJ[NS], corr = 0.0;
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if (s < N) {
        tJ[s] = FACE(vt_rd(N) + s) * DN(VT_Y + s);
        corr += tJ[s];
      }
    double qd = 0.0;
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if (s < N) {                                                // Eq. 6 (reading R21), Eq. 5
        const double J = -(tJ[s] - FACE(VT_Y + s) * corr);
        qd = fma(FACE(vt_h(N) + s), J, qd);
        if (s < N - 1) fs[((4 + s) * LDF + k) * LT + lt] = -J;
      }
    const double dT = (27.0 * (__ldg(A.T + q2) - __ldg(A.T + q1)) - (__ldg(A.T + q3) - __ldg(A.T + q0))) * in;
    fs[(3 * LDF + k) * LT + lt] = work + kappa * dT - qd;         // tau.u - q_c - q_d (Eq. 2, 4)
#undef FACE
#undef DN
#undef VL
  }
  __syncthreads();
  const int cell = c0 + k;                                        // this thread's cell: faces k .. k + 3 of the tile
  if (k < LD && lane_ok && cell < n) {
    const long long ic = base + (long long)(g + cell) * sd;
    const double in = G.inv_d[DIR] * (1.0 / 24.0);
    double kap = 0.0;
    if (A.first && A.Un) {                                        // the stage's alpha / (beta dt) U^n term (XfEpilogue mode 3)
      const double dt = A.S_dev ? A.cfl / *A.S_dev : A.dt;
      kap = A.alpha / (A.beta * dt);
    }
    if (A.first) A.out[ic] = A.Un ? kap * A.Un[ic] : 0.0;         // the density row has no viscous flux
    // all the operands of the update first, then the stores: written as one loop the compiler must keep every load of
    // `out` behind the previous store to it (it cannot tell the rows apart), a chain of DRAM round trips
    // (config 4, three launches: 21.6 -> 17.9 ms)
    double old[NS + 4];
#pragma unroll
    for (int v = 1; v < NS + 4; ++v)
      if (v < Nv) {
        const long long o = v * C + ic;
        old[v] = A.first ? (A.Un ? kap * A.Un[o] : 0.0) : A.out[o];
      }
#pragma unroll
    for (int v = 1; v < NS + 4; ++v)
      if (v < Nv) {
        const double *f = fs + ((v - 1) * LDF + k) * LT + lt;
        const double dv = (27.0 * (f[2 * LT] - f[LT]) - (f[3 * LT] - f[0])) * in;
        A.out[v * C + ic] = old[v] + dv;
      }
  }
}

#define XF_DISPATCH_N(N, CALL)        \
  switch (N) {                        \
    case 1: { CALL(1); break; }       \
    case 2: { CALL(2); break; }       \
    case 3: { CALL(3); break; }       \
    case 4: { CALL(4); break; }       \
    case 10: { CALL(10); break; }     \
    default: { CALL(0); break; }      \
  }

constexpr int LDF_X = 256, LDF_YZ = 16;

template <int NT, int DIR>
int launch_dir(const XfGrid &G, int N, const ViscArgs &A, cudaStream_t s) {
  constexpr int LDF = DIR == 0 ? LDF_X : LDF_YZ, LD = LDF - 3;
  const int OD = DIR == 1 ? 2 : 1;
  const dim3 block = DIR == 0 ? dim3(LDF) : dim3(XF_VISC_LT, LDF);
  const dim3 grid = DIR == 0 ? dim3((G.n[0] + LD - 1) / LD, G.n[1], G.n[2])
                             : dim3((G.n[0] + XF_VISC_LT - 1) / XF_VISC_LT, (G.n[DIR] + LD - 1) / LD, G.n[OD]);
  const size_t smem = sizeof(double) * (size_t)(N + 3) * LDF * (DIR == 0 ? 1 : XF_VISC_LT);
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(visc_dir_kernel<NT, DIR, LDF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)(sizeof(double) * (XF_MAXN + 3) * LDF * (DIR == 0 ? 1 : XF_VISC_LT)));
    attr_done = true;
  }
  visc_dir_kernel<NT, DIR, LDF><<<grid, block, smem, s>>>(G, N, A);
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

}  // namespace

int xf_launch_transport(const XfGrid &G, const XfThermo &Th, const XfTransportDev *tr_dev, const double *U, const double *T,
                        double *vtab, cudaStream_t s) {
  const int threads = TR_THREADS;
  const unsigned blocks = (unsigned)((G.cells + threads - 1) / threads);
  const size_t smem = sizeof(XfTransportDev) + sizeof(double) * (XF_MAXN + 4 * (size_t)Th.N * TR_THREADS);   // N = 16: 13 + 64 KB
#define CALL(NT)                                                                                                   \
  cudaFuncSetAttribute(transport_kernel<NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(XfTransportDev) + sizeof(double) * (XF_MAXN + 4 * XF_MAXN * TR_THREADS))); \
  transport_kernel<NT><<<blocks, threads, smem, s>>>(G, Th, tr_dev, U, T, vtab)
  XF_DISPATCH_N(Th.N, CALL)
#undef CALL
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}

// out = base + sum over active directions of the fourth-order divergence of F_v; base = kappa_un U^n or 0 (see ViscArgs)
int xf_launch_viscous(const XfGrid &G, int N, const double *vtab, const double *T, double *out, const XfEpilogue *stage,
                      cudaStream_t s, long *launches) {
  ViscArgs A;
  A.vtab = vtab;
  A.T = T;
  A.out = out;
  A.Un = nullptr;
  A.alpha = A.beta = A.dt = A.cfl = 0.0;
  A.S_dev = nullptr;
  if (stage) {   // the first sweep of this stage would have carried alpha / (beta dt) U^n: the viscous term carries it instead
    A.Un = stage->Un;
    A.alpha = stage->alpha;
    A.beta = stage->beta;
    A.dt = stage->dt;
    A.cfl = stage->cfl;
    A.S_dev = stage->S_dev;
  }
  A.first = 1;
  A.seg = 0;
  for (int d = 0; d < 3; ++d) {
    if (G.n[d] == 1) continue;
    int rc = XF_OK;
#define CALL(NT) rc = d == 0 ? launch_dir<NT, 0>(G, N, A, s) : (d == 1 ? launch_dir<NT, 1>(G, N, A, s) : launch_dir<NT, 2>(G, N, A, s))
    XF_DISPATCH_N(N, CALL)
#undef CALL
    if (rc != XF_OK) return rc;
    if (launches) ++*launches;
    A.first = 0;
  }
  return XF_OK;
}
