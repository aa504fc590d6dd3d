// xf_sweeps.cuh -- the marching sweep kernels built around xf::face_flux (see xf_flux.cuh).
//
// x sweep: lanes run ALONG the stencil.  All interior rows of one k-plane are contiguous in memory (row pitch =
//   padded nx), so a plane is swept as ONE long flat pencil; the few faces whose stencil straddles a row end are
//   computed on valid (ghost) data and never used (5 of every nx+6).  A block marches a segment of that pencil in
//   chunks of TX faces: stage TX+5 cells in shared memory, one face per thread, fluxes to shared memory, one cell
//   update per thread; the last face of a chunk is carried to the next, so no face is computed twice.
// y / z sweeps: lanes run ACROSS 32 neighbouring pencils (consecutive i -> coalesced), warps along the stencil.
//   A block marches a column in chunks of W faces over a ring of W+5 staged rows.
#pragma once
#include "xf_flux.cuh"

namespace xf {

constexpr int TX = 128;        // x sweep: faces per chunk = threads per block
constexpr int XCHUNKS = 8;     // x sweep: chunks per block segment (segment = XCHUNKS*TX - 1 cells)
constexpr int YZ_W = 8;        // y/z sweeps: warps per block = faces per chunk
constexpr int YZ_R = YZ_W + 5; // ring rows

template <int N_T>
__host__ __device__ constexpr int nspec_static() { return N_T > 0 ? N_T : XF_MAXN; }

__host__ inline size_t sweep_x_smem(int N) {
  return sizeof(double) * ((size_t)nfields(N) * (TX + 5) + (size_t)(N + 4) * (TX + 1));
}
__host__ inline size_t sweep_yz_smem(int N) {
  return sizeof(double) * ((size_t)nfields(N) * YZ_R * 32 + (size_t)(N + 4) * (YZ_W + 1) * 32);
}

template <int N_T>
__global__ void __launch_bounds__(TX)
sweep_x_kernel(const XfGrid G, const int Nrt, const double *__restrict__ U, const double *__restrict__ P,
               const double *__restrict__ Cs, const double *__restrict__ Gam, const double *__restrict__ chi,
               const XfEpilogue E, int *__restrict__ status, const int segs_per_plane) {
  const int N = N_T > 0 ? N_T : Nrt;
  const int Nv = N + 4, NF = nfields(N);
  extern __shared__ double smem[];
  constexpr int CS = TX + 5;          // cell slots per field
  constexpr int FSL = TX + 1;         // flux slots per variable
  double *sm = smem;
  double *fb = smem + (size_t)NF * CS;

  const int t = threadIdx.x;
  const int plane = blockIdx.x / segs_per_plane;            // interior k
  const int seg = blockIdx.x - plane * segs_per_plane;
  const long long L = (long long)G.n[1] * G.np[0];          // flat cells of the plane's interior rows
  const long long base = (long long)(plane + G.g[2]) * G.st[2] + (long long)G.g[1] * G.st[1];
  constexpr int SEG = XCHUNKS * TX - 1;
  const long long c0 = (long long)seg * SEG;                // first cell of this block's segment
  const long long c1 = c0 + SEG < L ? c0 + SEG : L;         // one past the last cell
  const double dt = E.mode == 2 ? (E.S_dev ? E.cfl / *E.S_dev : E.dt) : 0.0;
  const double ninv = -G.inv_d[0];

  for (int q = 0; q < XCHUNKS; ++q) {
    const long long f0 = c0 + (long long)q * TX;            // first face of the chunk (face f = left face of cell f)
    if (f0 > c1) break;
    // ---- stage cells f0-3 .. f0+TX+1 (slot x <-> cell f0-3+x)
    for (int x = t; x < CS; x += TX) {
      long long gi = base + f0 - 3 + x;
      gi = gi < 0 ? 0 : (gi >= G.cells ? G.cells - 1 : gi);  // garbage faces at the very ends stay in bounds
      for (int v = 0; v < Nv; ++v) sm[v * CS + x] = U[v * G.cells + gi];
      sm[Nv * CS + x] = P[gi];
      sm[(Nv + 1) * CS + x] = Cs[gi];
      double ud, ri, sr;
      derive_cell(sm[x], sm[1 * CS + x], ud, ri, sr);
      sm[(Nv + 2) * CS + x] = ud;
      sm[(Nv + 3) * CS + x] = ri;
      sm[(Nv + 4) * CS + x] = sr;
    }
    __syncthreads();
    // ---- one face per thread: face f0+t between cells f0+t-1 (slot t+2) and f0+t (slot t+3)
    const long long f = f0 + t;
    if (f <= c1) {
      const int o[6] = {t, t + 1, t + 2, t + 3, t + 4, t + 5};
      long long ga = base + f - 1, gb = base + f;
      ga = ga < 0 ? 0 : ga;
      gb = gb >= G.cells ? G.cells - 1 : gb;
      face_flux<N_T, 0>(N, sm, CS, o, Gam, chi, ga, gb, G.cells, fb + (t + 1), FSL, status);
    }
    __syncthreads();
    // ---- one cell per thread: cell f0+t-1 from the faces in flux slots t and t+1
    const long long cc = f0 + t - 1;
    if (cc >= c0 && cc < c1) {
      const int i = (int)(cc % G.np[0]);
      if (i >= G.g[0] && i < G.g[0] + G.n[0]) {
        const long long gi = base + cc;
        for (int v = 0; v < Nv; ++v) {
          const double div = (fb[v * FSL + t + 1] - fb[v * FSL + t]) * ninv;
          write_out(E, dt, v * G.cells + gi, div, sm[v * CS + t + 2]);
        }
      }
    }
    __syncthreads();
    if (t < Nv) fb[t * FSL] = fb[t * FSL + TX];             // carry the last face to the next chunk
  }
}

// DIR = 1 (y) or 2 (z).  Block (32, YZ_W): lane <-> i, warp <-> face within the chunk.
template <int N_T, int DIR>
__global__ void __launch_bounds__(32 * YZ_W)
sweep_yz_kernel(const XfGrid G, const int Nrt, const double *__restrict__ U, const double *__restrict__ P,
                const double *__restrict__ Cs, const double *__restrict__ Gam, const double *__restrict__ chi,
                const XfEpilogue E, int *__restrict__ status, const int seg_len) {
  const int N = N_T > 0 ? N_T : Nrt;
  const int Nv = N + 4, NF = nfields(N);
  extern __shared__ double smem[];
  constexpr int CS = YZ_R * 32;
  constexpr int FSL = (YZ_W + 1) * 32;
  double *sm = smem;
  double *fb = smem + (size_t)NF * CS;

  const int lane = threadIdx.x, w = threadIdx.y;
  constexpr int OD = DIR == 1 ? 2 : 1;                      // the other transverse direction
  const int i = G.g[0] + blockIdx.x * 32 + lane;
  const bool lane_ok = i < G.g[0] + G.n[0];
  const int ic = lane_ok ? i : G.g[0] + G.n[0] - 1;         // clamped: idle lanes stage valid data
  const long long colbase = (long long)(blockIdx.y + G.g[OD]) * G.st[OD] + ic;
  const long long sst = G.st[DIR];
  const int n = G.n[DIR];
  const int q0 = blockIdx.z * seg_len;                      // first interior cell of this block's segment
  const int q1 = q0 + seg_len < n ? q0 + seg_len : n;       // one past the last
  const double dt = E.mode == 2 ? (E.S_dev ? E.cfl / *E.S_dev : E.dt) : 0.0;
  const double ninv = -G.inv_d[DIR];

  // stage padded row r into ring slot r % YZ_R (each warp stages whole rows: 32 consecutive i per field)
  auto stage_row = [&](int r) {
    const int x = (r % YZ_R) * 32 + lane;
    const long long gi = colbase + (long long)r * sst;
    for (int v = 0; v < Nv; ++v) sm[v * CS + x] = U[v * G.cells + gi];
    sm[Nv * CS + x] = P[gi];
    sm[(Nv + 1) * CS + x] = Cs[gi];
    double ud, ri, sr;
    derive_cell(sm[x], sm[(1 + DIR) * CS + x], ud, ri, sr);
    sm[(Nv + 2) * CS + x] = ud;
    sm[(Nv + 3) * CS + x] = ri;
    sm[(Nv + 4) * CS + x] = sr;
  };

  const int nfaces = q1 - q0 + 1;                           // faces q0 .. q1 (face f lies between padded rows f+2, f+3)
  const int nchunks = (nfaces + YZ_W - 1) / YZ_W;
  for (int c = 0; c < nchunks; ++c) {
    const int f0 = q0 + c * YZ_W;
    // ---- rows needed by this chunk: f0 .. f0+W+4; all but the last W are already in the ring (except chunk 0)
    if (c == 0) {
      for (int r = f0 + w; r < f0 + 5; r += YZ_W) stage_row(r);
    }
    {
      const int r = f0 + 5 + w;
      if (r <= q1 + 5) stage_row(r);
    }
    __syncthreads();
    const int f = f0 + w;
    if (f <= q1 && lane_ok) {
      int o[6];
#pragma unroll
      for (int m = 0; m < 6; ++m) o[m] = ((f + m) % YZ_R) * 32 + lane;
      const long long ga = colbase + (long long)(f + 2) * sst, gb = ga + sst;
      face_flux<N_T, DIR>(N, sm, CS, o, Gam, chi, ga, gb, G.cells, fb + (w + 1) * 32 + lane, FSL, status);
    }
    __syncthreads();
    const int qq = f - 1;                                   // cell between faces qq (slot w) and qq+1 (slot w+1)
    if (qq >= q0 && qq < q1 && lane_ok) {
      const long long gi = colbase + (long long)(qq + 3) * sst;
      const int x = ((qq + 3) % YZ_R) * 32 + lane;
      for (int v = 0; v < Nv; ++v) {
        const double div = (fb[v * FSL + (w + 1) * 32 + lane] - fb[v * FSL + w * 32 + lane]) * ninv;
        write_out(E, dt, v * G.cells + gi, div, sm[v * CS + x]);
      }
    }
    __syncthreads();
    for (int v = w; v < Nv; v += YZ_W) fb[v * FSL + lane] = fb[v * FSL + YZ_W * 32 + lane];  // carry the last face
  }
}

}  // namespace xf

#define XF_DISPATCH_SWEEP_N(N, CALL) \
  switch (N) {                       \
    case 1: { CALL(1); break; }      \
    case 2: { CALL(2); break; }      \
    case 3: { CALL(3); break; }      \
    case 4: { CALL(4); break; }      \
    case 10: { CALL(10); break; }    \
    default: { CALL(0); break; }     \
  }
