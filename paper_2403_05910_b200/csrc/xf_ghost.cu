// xf_ghost.cu -- ghost-cell fill (reading R10), one launch per active direction, x then y then z.
// Each launch covers the padded extent of the directions already filled, so edges and corners end up defined.
#include "xf_common.cuh"

namespace {

// thread <-> (transverse cell, layer l, side); loops over the Nv variables (stride = cells keeps every access of a
// warp on consecutive i for the y and z fills; the x fill touches 3- or 4-cell runs and is tiny).
__global__ void __launch_bounds__(256)
ghost_kernel(const XfGrid G, int Nv, int d, int bc_lo, int bc_hi, const double *__restrict__ bc_state,
             double *__restrict__ U) {
  // transverse extents: padded for directions < d (already filled), interior for directions > d
  int lo[3], ext[3];
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    if (q < d) { lo[q] = 0; ext[q] = G.np[q]; }
    else { lo[q] = G.g[q]; ext[q] = G.n[q]; }
  }
  const int a1 = d == 0 ? 1 : 0;          // faster transverse axis
  const int a2 = d == 2 ? 1 : 2;          // slower transverse axis
  const long long ntrans = (long long)ext[a1] * ext[a2];
  const int ng = G.g[d];                  // ghost layers per side: 3, or 4 for WENO7
  const long long total = ntrans * ng * 2;
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= total) return;
  long long tr;
  int l, side;
  if (d == 0) {  // x fill: the ng layers of one row end are neighbours in memory -> make them neighbours in the warp
    l = (int)(t % ng);
    side = (int)((t / ng) & 1);
    tr = t / (2 * ng);
  } else {       // y / z fill: consecutive threads on consecutive i
    tr = t % ntrans;
    const int ls = (int)(t / ntrans);
    l = ls % ng;
    side = ls / ng;
  }
  const int p1 = lo[a1] + (int)(tr % ext[a1]);
  const int p2 = lo[a2] + (int)(tr / ext[a1]);
  const int n = G.n[d], g = G.g[d];
  const int bc = side == 0 ? bc_lo : bc_hi;
  if (bc == XF_BC_EXCHANGE) return;   // filled by the halo exchange with the neighbouring block (xf_halo.cu)
  const int ighost = side == 0 ? g - 1 - l : g + n + l;
  int isrc = ighost;
  if (bc == XF_BC_PERIODIC) isrc = side == 0 ? ighost + n : ighost - n;
  else if (bc == XF_BC_TRANSMISSIVE) isrc = side == 0 ? g : g + n - 1;
  else if (bc == XF_BC_REFLECTIVE) isrc = side == 0 ? g + l : g + n - 1 - l;
  const long long base = (long long)p1 * G.st[a1] + (long long)p2 * G.st[a2];
  const long long ig = base + (long long)ighost * G.st[d];
  const long long is = base + (long long)isrc * G.st[d];
  // U is read and written: the compiler must keep every load behind the previous store.  Batches of loads first, then
  // their stores (a ghost cell is never a source of the same launch: sources are interior along d), so a thread has
  // several loads in flight instead of one.
  constexpr int VB = 7;
  for (int v0 = 0; v0 < Nv; v0 += VB) {
    double val[VB];
#pragma unroll
    for (int q = 0; q < VB; ++q) {
      const int v = v0 + q;
      if (v < Nv) {
        if (bc == XF_BC_DIRICHLET) val[q] = bc_state[(2 * d + side) * XF_MAXNV + v];
        else {
          val[q] = U[v * G.cells + is];
          if (bc == XF_BC_REFLECTIVE && v == 1 + d) val[q] = -val[q];  // wall-normal momentum negated
        }
      }
    }
#pragma unroll
    for (int q = 0; q < VB; ++q) {
      const int v = v0 + q;
      if (v < Nv) U[v * G.cells + ig] = val[q];
    }
  }
}

}  // namespace

int xf_launch_ghosts(const XfGrid &G, int Nv, const XfBc &bc, const double *bc_state_dev, double *U, cudaStream_t s,
                     long *launches, int only_dir) {
  for (int d = 0; d < 3; ++d) {
    if (G.n[d] == 1 || (only_dir >= 0 && d != only_dir)) continue;
    if (bc.kind[2 * d] == XF_BC_EXCHANGE && bc.kind[2 * d + 1] == XF_BC_EXCHANGE) continue;
    long long ntrans = 1;
    for (int q = 0; q < 3; ++q)
      if (q != d) ntrans *= (q < d ? G.np[q] : G.n[q]);
    const long long total = ntrans * G.g[d] * 2;
    const int threads = 256;
    const unsigned blocks = (unsigned)((total + threads - 1) / threads);
    ghost_kernel<<<blocks, threads, 0, s>>>(G, Nv, d, bc.kind[2 * d], bc.kind[2 * d + 1], bc_state_dev, U);
    if (launches) ++*launches;
    if (cudaGetLastError() != cudaSuccess) return XF_ECUDA;
  }
  return XF_OK;
}
