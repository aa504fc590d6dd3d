// xf_halo.cu -- halo exchange between the blocks of a Cartesian domain decomposition (
// one block per GPU / MPI rank, the 3-deep "border" layers of a block become the "boundary" layers of
// its face neighbour; x, then y, then z, each over the padded extent of the directions already done, so edge and corner
// ghosts arrive without diagonal messages).  This file is the device side: pack the g interior layers next to a face
// into a contiguous buffer [Nv + 1][g][transverse cells] (U and T), unpack a received buffer into the g ghost layers beyond a face.
// The transfer itself (NCCL send / recv through torch.distributed, or a device copy between two blocks of one process)
// is plumbing and lives in paper_2403_05910_b200/halo.py.  A face whose boundary kind is XF_BC_EXCHANGE is skipped by
// the ghost-fill kernel.
#include "xf_common.cuh"

namespace {

// thread <-> (transverse cell t, layer l); loops over the Nv variables.  PACK: buf <- U, else U <- buf.
template <bool PACK>
__global__ void __launch_bounds__(256)
halo_kernel(const XfGrid G, int Nv, int d, int side, double *__restrict__ U, double *__restrict__ T,
            double *__restrict__ buf) {
  int lo[3], ext[3];
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    if (q < d) { lo[q] = 0; ext[q] = G.np[q]; }
    else { lo[q] = G.g[q]; ext[q] = G.n[q]; }
  }
  const int a1 = d == 0 ? 1 : 0, a2 = d == 2 ? 1 : 2;
  const long long ntrans = (long long)ext[a1] * ext[a2];
  const int g = G.g[d], n = G.n[d];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntrans * g) return;
  const long long tr = t % ntrans;
  const int l = (int)(t / ntrans);
  const int p1 = lo[a1] + (int)(tr % ext[a1]), p2 = lo[a2] + (int)(tr / ext[a1]);
  // PACK: the interior layers next to the face, in ascending order of the d-coordinate; UNPACK: the ghost layers beyond it
  const int c = PACK ? (side == 0 ? g + l : n + l) : (side == 0 ? l : g + n + l);
  const long long cell = (long long)p1 * G.st[a1] + (long long)p2 * G.st[a2] + (long long)c * G.st[d];
  for (int v = 0; v < Nv; ++v) {
    const long long b = ((long long)v * g + l) * ntrans + tr;
    if (PACK) buf[b] = U[v * G.cells + cell];
    else U[v * G.cells + cell] = buf[b];
  }
  // the temperature travels along as field Nv: a ghost cell then starts its Newton iteration from the same guess as the
  // cell it mirrors, which makes a decomposed run reproduce the single-block run bit for bit
  const long long b = ((long long)Nv * g + l) * ntrans + tr;
  if (PACK) buf[b] = T[cell];
  else T[cell] = buf[b];
}

long long halo_cells(const XfGrid &G, int d) {
  long long ntrans = 1;
  for (int q = 0; q < 3; ++q)
    if (q != d) ntrans *= (q < d ? G.np[q] : G.n[q]);
  return ntrans * G.g[d];
}

}  // namespace

long long xf_halo_count(const XfGrid &G, int Nv, int d) { return G.n[d] > 1 ? halo_cells(G, d) * (Nv + 1) : 0; }

int xf_launch_halo(const XfGrid &G, int Nv, int d, int side, bool pack, double *U, double *T, double *buf, cudaStream_t s) {
  if (G.n[d] == 1) return XF_EINVAL;
  const long long total = halo_cells(G, d);
  const int threads = 256;
  const unsigned blocks = (unsigned)((total + threads - 1) / threads);
  if (pack) halo_kernel<true><<<blocks, threads, 0, s>>>(G, Nv, d, side, U, T, buf);
  else halo_kernel<false><<<blocks, threads, 0, s>>>(G, Nv, d, side, U, T, buf);
  return cudaGetLastError() == cudaSuccess ? XF_OK : XF_ECUDA;
}
