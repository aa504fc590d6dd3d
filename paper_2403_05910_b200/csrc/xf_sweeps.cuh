// xf_sweeps.cuh -- the directional sweep kernels built around xf::face_flux (see xf_flux.cuh): staging of the stencil
// data, flux divergence (Eq. 13) and the fused Runge-Kutta stage combination (Eq. 16).
//
// Production kernels (second half of this file), all warp-specialised with TMA staging:
//   sweep_x_ws_kernel        x: one k-plane = one flat pencil, 128-face chunks in two stages
//   sweep_yz_ws_kernel<DIR>  y, z: 32 lanes along i x 4 face rows, ring of 13 / 9 rows
// Fallbacks for arrays TMA cannot describe (odd padded extents): the same y/z kernel with cp.async staging, and for x
// the warp-autonomous sweep_kernel below (first half of this file):
//
// sweep_kernel: every WARP is autonomous: it owns a private ring of staged stencil rows in shared memory, fills it
// with cp.async (LDGSTS), exchanges face fluxes with warp shuffles, and never meets a block-wide barrier.
// A warp's 32 lanes are laid out LI (contiguous, along i) x LJ (along the sweep direction); one lane = one face.
//   x sweep: LI = 1, LJ = 32.  All interior rows of one k-plane are contiguous in memory (row pitch = padded nx),
//     so a plane is swept as ONE long flat pencil; the few faces whose stencil straddles a row end are computed
//     on valid (ghost) data and never used (5 of every nx+6).
// With S stencil cells per face (6; 8 for WENO7; ghost width S/2) a chunk of LJ face rows needs LJ + S - 1 stencil rows;
// the ring holds RR rows (LJ + S - 1 .. 2 LJ + S - 1: the rows beyond the first count let part of the next chunk land while
// the current one is computed).  Face row f of a segment is the lower face of cell f; its stencil is rows f .. f+S-1; the
// lane that owns face f updates cell f-1 (stencil row f + S/2 - 1) from its own flux and that of face f-1 (the lane LI below it, or the carry left in shared memory by the previous chunk).
#pragma once
#include "xf_flux.cuh"

namespace xf {

constexpr int X_LI = 1, X_LJ = 32, X_NCH = 16;   // x sweep: segment = X_NCH chunks = 32*X_NCH faces, 32*X_NCH - 1 cells
constexpr int X_MINB = 12;                        // ring of exactly one chunk (X_LJ + S - 1 rows), 12 warps per SM
constexpr int YZ_W = 4;                           // y/z sweeps: warps per block = face rows per chunk

__host__ __device__ constexpr int ring_rows(int LJ, int S) { return 2 * LJ + S - 1; }   // S stencil cells per face
__host__ __device__ inline size_t warp_smem_doubles(int N, int LI, int RR) {   // ring, carry x 2, flux scratch [Nv][32]
  return (size_t)nstaged(N) * RR * LI + 2 * (size_t)(N + 4) * LI + (size_t)(N + 4) * 32;
}

__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory");
}

// dt of a Runge-Kutta stage: the host's, or CFL / S read on the device (xf_rk3_step_cfl, xf_step_cfl).  A step that is
// not finite and positive (S = 0, inf or NaN on the device; the host entry points reject such a dt) raises the
// non-physical flag instead of silently turning U into NaN through alpha / (beta dt).
__device__ __forceinline__ double stage_dt(const XfEpilogue &E, int *status) {
  if (E.mode < 2) return 0.0;
  const double dt = E.S_dev ? E.cfl / *E.S_dev : E.dt;
  if (!(dt > 0.0 && dt < 1.0e300)) atomicOr(status, XF_FLAG_NONPHYSICAL);
  return dt;
}

// Differences each flux component against the face below (Eq. 13) and writes the cell value: a plain residual,
// an accumulated residual, or the Runge-Kutta stage combination out = alpha*Un + beta*(Us + dt*(acc + div)) (Eq. 16).
// The acc / Un operands of the NEXT component are fetched while the current one is being reconstructed.
template <int LI>
struct CellWriter {
  const XfEpilogue &E;
  const double *sm_us;    // staged U^s of the cell this lane updates: sm_us[v * FS]
  double *carry_rd, *carry_wr;
  long long gi, cells;
  double dt, ninv, nacc, nun, kappa;
  int FS, li;
  bool write_ok, first_row, last_row, need_acc, need_un;

  __device__ __forceinline__ void preload(int v) {
    if (write_ok) {
      if (need_acc) nacc = E.acc[v * cells + gi];
      if (need_un) nun = E.Un[v * cells + gi];
    }
  }
  __device__ __forceinline__ void operator()(int v, double F, int vnext) {
    double prev = __shfl_up_sync(0xffffffffu, F, LI);
    if (first_row) prev = carry_rd[v * LI + li];
    if (last_row) carry_wr[v * LI + li] = F;
    if (write_ok) {
      const double div = (F - prev) * ninv;
      const long long idx = v * cells + gi;
      if (E.mode == 0) {
        E.out[idx] = div;
      } else if (E.mode == 3) {
        E.out[idx] = fma(kappa, nun, div);
      } else if (E.mode == 1) {
        E.out[idx] = nacc + div;
      } else {
        const double L = need_acc ? nacc + div : div;
        const double us = sm_us[v * FS];
        E.out[idx] = need_un ? fma(E.alpha, nun, E.beta * fma(dt, L, us)) : E.beta * fma(dt, L, us);
      }
    }
    if (vnext >= 0) preload(vnext);   // after the use: no register copy, the load flies during the next field
  }
  // pull the acc / Un operands of cell g (this lane's cell of a later chunk) into L2 ahead of time
  __device__ __forceinline__ void prefetch_l2(long long g, int Nv) const {
    if (need_acc)
      for (int v = 0; v < Nv; ++v) asm volatile("prefetch.global.L2 [%0];" ::"l"(E.acc + v * cells + g));
    if (need_un)
      for (int v = 0; v < Nv; ++v) asm volatile("prefetch.global.L2 [%0];" ::"l"(E.Un + v * cells + g));
  }
};

struct FluxScratch {   // face_flux emitter that only parks the components: scr[v * 32]
  double *scr;
  __device__ __forceinline__ void operator()(int v, double F, int) { scr[v * 32] = F; }
};

// One warp = one segment of one pencil group.  DIR = 0: blockIdx.x enumerates (k-plane, segment of the flat pencil).
// DIR = 1, 2: blockIdx = (group of LI pencils along i, index along the other transverse direction, segment).
template <int N_T, int DIR, int LI, int LJ, int RR, int MINB, int RECON>
__global__ void __launch_bounds__(32, MINB)
sweep_kernel(const XfGrid G, const int Nrt, const double *__restrict__ U, const double *__restrict__ prim,
             const XfEpilogue E, int *__restrict__ status, const int seg_param) {
  static_assert(LI * LJ == 32, "one lane per face");
  const int N = N_T > 0 ? N_T : Nrt;
  const int Nv = N + 4, NST = nstaged(N);
  constexpr int S = stencil_cells(RECON), HW = S / 2, MA = S / 2 - 1;   // stencil cells, ghost width, cell below the face
  static_assert(RR >= LJ + S - 1 && RR <= 2 * LJ + S - 1, "ring: one chunk plus 0..LJ rows of prefetch");
  constexpr int PF = RR - (LJ + S - 1);                     // rows of the next chunk that land during the arithmetic
  constexpr int FS = RR * LI;
  extern __shared__ double smem[];
  double *sm = smem;
  double *carry = smem + (size_t)NST * FS;

  const int lane = threadIdx.x;
  const int li = lane % LI, lj = lane / LI;

  // ---- this warp's segment: faces f_begin .. f_end (inclusive), cells f_begin .. f_end - 1
  long long base;      // global index of stencil row 0 at li = 0 (may be negative for the x sweep: clamped on use)
  long long sst;       // stride between stencil rows
  int f_begin, f_end;
  int i0 = 0, imax = 0;  // y/z: first i of this pencil group, last valid i
  if (DIR == 0) {
    const int segs_per_plane = seg_param;
    const int plane = blockIdx.x / segs_per_plane;
    const int seg = blockIdx.x - plane * segs_per_plane;
    const int L = G.n[1] * G.np[0];                          // flat cells of the plane's interior rows
    constexpr int SEGC = X_NCH * 32 - 1;
    f_begin = seg * SEGC;
    f_end = f_begin + SEGC < L ? f_begin + SEGC : L;
    base = (long long)(plane + G.g[2]) * G.st[2] + (long long)G.g[1] * G.st[1] - HW;  // row r <-> flat cell r - HW
    sst = 1;
  } else {
    constexpr int OD = DIR == 1 ? 2 : 1;                     // the other transverse direction
    const int seg_len = seg_param;
    i0 = G.g[0] + blockIdx.x * LI;
    imax = G.g[0] + G.n[0] - 1;
    base = (long long)(blockIdx.y + G.g[OD]) * G.st[OD];     // + i, + r * sst
    sst = G.st[DIR];
    f_begin = blockIdx.z * seg_len;
    f_end = f_begin + seg_len < G.n[DIR] ? f_begin + seg_len : G.n[DIR];
  }
  auto row_addr = [&](int r, int l) -> long long {           // global cell index of stencil row r, lane column l
    if (DIR == 0) {
      long long gi = base + r;
      return gi < 0 ? 0 : (gi >= G.cells ? G.cells - 1 : gi);  // garbage faces at the very ends stay in bounds
    }
    const int ii = i0 + l < imax ? i0 + l : imax;            // idle lanes stage valid data
    const int rr = r < G.np[DIR] ? r : G.np[DIR] - 1;        // rows past the last chunk's needs stay in bounds
    return base + ii + (long long)rr * sst;
  };
  auto stage = [&](int slot, long long gi) {
    double *dst = sm + slot;
#pragma unroll
    for (int f = 0; f < (N_T > 0 ? nstaged(N_T) : 1); ++f) {
      if (N_T > 0) cp_async8(dst + f * FS, (f < Nv ? U + (size_t)f * G.cells : prim + (size_t)(f - Nv) * G.cells) + gi);
    }
    if (N_T == 0) {
      for (int f = 0; f < NST; ++f)
        cp_async8(dst + f * FS, (f < Nv ? U + (size_t)f * G.cells : prim + (size_t)(f - Nv) * G.cells) + gi);
    }
  };

  // ---- prologue: rows f_begin .. f_begin + LJ + S - 2 into ring slots 0 .. LJ + S - 2
  for (int idx = lane; idx < (LJ + S - 1) * LI; idx += 32) {
    const int r = idx / LI, l = idx - r * LI;
    stage(r * LI + l, row_addr(f_begin + r, l));
  }
  cp_async_commit();

  const double dt = stage_dt(E, status);
  CellWriter<LI> W{E};
  W.cells = G.cells;
  W.dt = dt;
  W.ninv = -G.inv_d[DIR];
  W.FS = FS;
  W.li = li;
  W.first_row = lj == 0;
  W.last_row = lj == LJ - 1;
  W.need_acc = E.mode == 1 || (E.mode == 2 && E.has_acc);
  W.need_un = (E.mode == 2 && E.alpha != 0.0) || E.mode == 3;
  W.kappa = E.mode == 3 ? E.alpha / (E.beta * dt) : 0.0;
  W.nacc = 0.0;
  W.nun = 0.0;
  const bool lane_ok = DIR == 0 || i0 + li <= imax;

  int rb = 0;       // ring slot (row) of stencil row fc
  int par = 0;
  bool bad = false;
  for (int fc = f_begin; fc <= f_end; fc += LJ) {
    // ---- prefetch the first PF new rows of the next chunk (rows fc + LJ + S - 1 + lj) into the free part of the ring
    if (PF > 0 && lj < PF && fc + LJ <= f_end) {
      int slot = rb + LJ + S - 1 + lj;
      slot -= slot >= RR ? RR : 0;
      stage(slot * LI + li, row_addr(fc + LJ + S - 1 + lj, li));
    }
    cp_async_commit();
    cp_async_wait<1>();   // everything but the group just committed has landed
    __syncwarp();

    const int f = fc + lj;
    int o[S];
#pragma unroll
    for (int m = 0; m < S; ++m) {
      int s = rb + lj + m;
      s -= s >= RR ? RR : 0;
      o[m] = s * LI + li;
    }
    // the cell this lane updates: f - 1 (between faces f - 1 and f), staged at stencil row f + MA (m = MA)
    bool ok = lane_ok && f > f_begin && f <= f_end;
    long long gi;
    if (DIR == 0) {
      const int cc = f - 1;
      const int i = cc % G.np[0];
      ok = ok && i >= G.g[0] && i < G.g[0] + G.n[0];
      gi = base + HW + cc;
    } else {
      gi = base + (i0 + li) + (long long)(f + MA) * sst;
    }
    W.write_ok = ok;
    W.gi = gi;
    if (W.need_acc || W.need_un) {                          // operands of this lane's cell in the NEXT chunk -> L2
      const long long gnext = gi + (long long)LJ * sst;
      if (fc == f_begin && ok) W.prefetch_l2(gi, Nv);
      if (lane_ok && f + LJ <= f_end && gnext < G.cells) W.prefetch_l2(gnext, Nv);
    }
#pragma unroll
    for (int m = 0; m < S; ++m) asm volatile("" : "+r"(o[m]));   // keep the ring offsets in registers (see the y/z kernel)
    W.sm_us = sm + o[MA];
    W.carry_rd = carry + par * Nv * LI;
    W.carry_wr = carry + (par ^ 1) * Nv * LI;
    W.preload(0);
    bool c2ok;
    if (E.pp) {   // the limiter needs the whole flux vector: park it in the warp's scratch, blend (Eq. 20), then difference
      double *scr = carry + 2 * Nv * LI + lane;
      FluxScratch fs{scr};
      c2ok = face_flux<DIR, RECON>(N, sm, sm + Nv * FS, FS, o, sm + (Nv + 3) * FS, FS, o[MA], o[MA + 1], E.visc, E.lam_glob + 3 * DIR, fs);
      positivity_blend<DIR>(N, sm, sm + Nv * FS, FS, o[MA], o[MA + 1], pp_kappa(E, G, DIR), scr, 32);
      constexpr int nd = Axes<DIR>::nd, t1 = Axes<DIR>::t1, t2 = Axes<DIR>::t2;
      W(0, scr[0], 1 + nd);                                 // same component order as face_flux emits
      W(1 + nd, scr[(1 + nd) * 32], 1 + t1);
      W(1 + t1, scr[(1 + t1) * 32], 1 + t2);
      W(1 + t2, scr[(1 + t2) * 32], N > 1 ? 5 : 4);
      for (int i = 0; i < N - 1; ++i) W(5 + i, scr[(5 + i) * 32], i + 2 < N ? 6 + i : 4);
      W(4, scr[4 * 32], -1);
    } else {
      c2ok = face_flux<DIR, RECON>(N, sm, sm + Nv * FS, FS, o, sm + (Nv + 3) * FS, FS, o[MA], o[MA + 1], E.visc, E.lam_glob + 3 * DIR, W);
    }
    bad = bad || (!c2ok && lane_ok && f <= f_end);
    __syncwarp();         // all lanes are done with the rows the next iteration's prefetch overwrites
    if (PF < LJ) {        // the remaining LJ - PF rows of the next chunk go where this chunk's first rows were
      if (lj >= PF && fc + LJ <= f_end) {
        int slot = rb + LJ + S - 1 + lj;
        slot -= slot >= RR ? RR : 0;
        slot -= slot >= RR ? RR : 0;
        stage(slot * LI + li, row_addr(fc + LJ + S - 1 + lj, li));
      }
      cp_async_commit();
    }
    rb += LJ;
    rb -= rb >= RR ? RR : 0;
    par ^= 1;
  }
  cp_async_wait<0>();
  if (bad) atomicOr(status, XF_FLAG_NONPHYSICAL);
}


// ---------------------------------------------------------------------------------------------------------------
// y / z sweeps: block-cooperative, every global access a full 256-byte row.
// Block = 32 lanes (consecutive i) x W face rows along the sweep direction.  The stencil rows live in a shared ring
// of 2 W + 5 rows: while the W face rows of a chunk are computed, the W new rows of the next chunk land through
// cp.async (one row per warp: 32 consecutive doubles per field).  Face fluxes go to a small shared buffer (row w + 1;
// row 0 is the last face of the previous chunk) and are differenced from there.
// ---------------------------------------------------------------------------------------------------------------
// TMA layout (doubles).  A box must start 16-byte aligned in global memory and 128-byte aligned in shared memory
// (measured: anything else raises "illegal instruction" / "misaligned address"), and with ghost width 3 the interior
// starts at the odd index 3, so a row is fetched as 34 doubles from i0 - (g & 1): lane l reads element l + (g & 1).  One ring row = the U box
// [Nv][34] and the p, c, 1/rho box [3][34], each padded to 128 bytes; Gamma and chi_s (needed only at the two cells
// next to a face) live in a second, shallower ring of [N + 1][34] boxes.
constexpr int TMA_RW = 34;
__host__ __device__ constexpr int tma_box_doubles(int nf) { return (nf * TMA_RW * 8 + 127) / 128 * 16; }
__host__ __device__ constexpr int tma_deep_slot(int N) { return tma_box_doubles(N + 4) + tma_box_doubles(3); }
__host__ __device__ constexpr int tma_shallow_slot(int N) { return tma_box_doubles(N + 1); }
__host__ __device__ inline size_t yz_smem_doubles(int N, int W, int S) {   // ring(s), flux buffer, two mbarriers
  const size_t plain = (size_t)nstaged(N) * ring_rows(W, S) * 32;
  const size_t tma = (size_t)ring_rows(W, S) * tma_deep_slot(N) + (size_t)(2 * W + 1) * tma_shallow_slot(N);
  return (plain > tma ? plain : tma) + (size_t)(N + 4) * (W + 1) * 32 + 4;
}

// ---------------------------------------------------------------------------------------------------------------
// Warp-specialised.  Measured on config 4 (profiles/): with every warp doing staging, arithmetic and the cell
// update in turn, a quarter of the warp time sits in the update
// (global operands, stores) and in issuing copies, and while one of the SM's two blocks is there the fp64 pipe is
// fed by a single warp per scheduler.  Here a block is two warp groups:
//   * W COMPUTE warps (warp w = face row fc + w) run xf::face_flux back to back and nothing else;
//   * W SERVICE warps keep the ring one chunk ahead (cp.async) and, concurrently with the next chunk's arithmetic,
//     difference the fluxes of the chunk just finished and write the cells (Eq. 13, Eq. 16).
// setmaxnreg moves registers from the service group (88) to the compute group (168): two blocks per SM.
// Named barriers (ids alternate with the chunk parity): RING_FULL  service -> compute  rows of chunk c landed (cp.async path)
//                                                        FLUX_READY compute -> service  fluxes of chunk c in fb
// mbarriers (one per chunk parity):                      full       TMA -> compute      rows of chunk c landed
//                                                        fb_empty   service -> compute  fb of chunk c - 1 consumed
// The compute warps only ever ARRIVE on a named barrier; what they wait on are mbarriers, whose phase has as a rule
// completed long before they look, so a compute warp never stalls on another compute warp.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void named_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void named_arrive(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
// mbarrier / TMA (cp.async.bulk.tensor) primitives of the ring's producer side
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "XF_MBAR_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra XF_MBAR_DONE;\n"
      "bra XF_MBAR_WAIT;\n"
      "XF_MBAR_DONE:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// one box {32 cells along i} x {nf fields} of row (c1, c2) -> dst, completion counted in bytes on `bar`
__device__ __forceinline__ void tma_load_row(unsigned dst, const void *tmap, int c0, int c1, int c2, unsigned bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(dst),
      "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(0), "r"(bar)
      : "memory");
}

constexpr int BAR_RING_FULL = 1, BAR_FLUX_READY = 3;   // + chunk parity
constexpr int BAR_SERVICE = 7;   // among the service warps: all have read U^s before any of them overwrites ring rows
#ifndef XF_WS_RC
#define XF_WS_RC 168   // 2 blocks x 128 threads x (168 + 88) registers = the SM's 64 K
#define XF_WS_RS 88
#endif
constexpr int WS_REGS_COMPUTE = XF_WS_RC, WS_REGS_SERVICE = XF_WS_RS;

struct FluxStoreWS {
  double *dst;       // fb + row * 32 + lane
  int stride;        // doubles between components
  unsigned wait_bar; // mbarrier to pass before the first component is written: the service warps have read the
  unsigned parity;   //   previous chunk's fluxes (0: nothing to wait for).  Not a bar.sync: the compute warps never
                     //   wait for ONE ANOTHER, only for the consumer of the buffer they are about to overwrite
  __device__ __forceinline__ void operator()(int v, double F, int) {
    if (v == 0 && wait_bar) mbar_wait(wait_bar, parity);
    dst[v * stride] = F;
  }
};

template <int N_T, int DIR, int W, bool TMA, int RECON>
__global__ void __launch_bounds__(64 * W, 2)
sweep_yz_ws_kernel(const XfGrid G, const int Nrt, const double *__restrict__ U, const double *__restrict__ prim,
                   const XfEpilogue E, int *__restrict__ status, const int seg_len,
                   const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmP,
                   const __grid_constant__ CUtensorMap tmS) {
  constexpr int S = stencil_cells(RECON), MA = S / 2 - 1;    // stencil cells per face; m of the cell below the face
  static_assert(W > MA, "the service warps' ring-row hand-over needs W > S/2 - 1");
  const int N = N_T > 0 ? N_T : Nrt;
  const int Nv = N + 4, NST = nstaged(N);
  constexpr int NVS = N_T > 0 ? N_T + 4 : XF_MAXNV;        // static bound of Nv for register arrays
  constexpr int RR = ring_rows(W, S);
  // ring layout: TMA -> sm[slot][box][field][34] (see above), cp.async -> sm[field][slot][32]
  constexpr int RS = 2 * W + 1;                             // rows of the shallow ring (TMA only)
  const int FS = TMA ? TMA_RW : RR * 32;                    // doubles between fields
  const int SLOT = TMA ? tma_deep_slot(N) : 32;             // doubles between ring rows
  const int SSLOT = TMA ? tma_shallow_slot(N) : 32;
  constexpr int FBS = (W + 1) * 32;                         // flux-buffer doubles per component
  constexpr int NT = 64 * W;                                // threads that take part in every named barrier
  extern __shared__ __align__(128) double smem[];
  double *sm = smem;                                                            // U fields
  double *smp = TMA ? smem + tma_box_doubles(Nv) : smem + (size_t)Nv * FS;      // p, c, 1/rho
  double *sms = TMA ? smem + (size_t)RR * SLOT : smem + (size_t)(Nv + 3) * FS;  // Gamma, chi_s
  double *fb = TMA ? sms + (size_t)RS * SSLOT : smem + (size_t)NST * RR * 32;
  const unsigned full_bar = (unsigned)__cvta_generic_to_shared(fb + (size_t)Nv * FBS);   // two mbarriers (TMA only)
  const unsigned fbe_bar = full_bar + 16;                   // two more: flux buffer consumed
  if (threadIdx.x == 0 && threadIdx.y == 0) {
    mbar_init(full_bar, W);                                 // one arrival (with its byte count) per service warp
    mbar_init(full_bar + 8, W);
    mbar_init(fbe_bar, W);                                  // one arrival per service warp
    mbar_init(fbe_bar + 8, W);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const int lane = threadIdx.x;
  const bool service = threadIdx.y >= W;
  const int w = service ? threadIdx.y - W : threadIdx.y;    // face row within the chunk / ring row staged
  constexpr int OD = DIR == 1 ? 2 : 1;                      // the other transverse direction
  const int lo = TMA ? (G.g[0] & 1) : 0;                    // TMA rows start at the even index below the strip's first cell
  const int i = G.g[0] + blockIdx.x * 32 + lane;
  const int imax = G.g[0] + G.n[0] - 1;
  const bool lane_ok = i <= imax;
  const long long colbase = (long long)(blockIdx.y + G.g[OD]) * G.st[OD] + (lane_ok ? i : imax);  // idle lanes: valid data
  const long long sst = G.st[DIR];
  const int f_begin = blockIdx.z * seg_len;                 // faces f_begin .. f_end, cells f_begin .. f_end - 1
  const int f_end = f_begin + seg_len < G.n[DIR] ? f_begin + seg_len : G.n[DIR];

  if (!service) {
    // =========================================================== compute warps
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(WS_REGS_COMPUTE));
    int rb = 0, rs = 0, par = 0;
    unsigned phase = 0;
    bool bad = false, first = true;
    for (int fc = f_begin; fc <= f_end; fc += W) {
      if (TMA) mbar_wait(full_bar + 8 * par, phase);        // rows fc .. fc + W + S - 2 are in the ring
      else named_sync(BAR_RING_FULL + par, NT);
      const int f = fc + w;
      int o[S];
#pragma unroll
      for (int m = 0; m < S; ++m) {
        int sl = rb + w + m;
        sl -= sl >= RR ? RR : 0;
        o[m] = sl * SLOT + lane + lo;
      }
      int s2 = o[MA], s3 = o[MA + 1];
      if (TMA) {                                            // shallow ring: slot of stencil row r is (r - f_begin - MA) mod RS
        int q2 = rs + w;
        q2 -= q2 >= RS ? RS : 0;
        int q3 = q2 + 1;
        q3 -= q3 >= RS ? RS : 0;
        s2 = q2 * SSLOT + lane + lo;
        s3 = q3 * SSLOT + lane + lo;
      }
      // the ring offsets are made opaque: otherwise the compiler, short of registers, re-derives every one of them
      // (wrap selects and multiplies, ~40 integer instructions per species field) instead of keeping six registers
#pragma unroll
      for (int m = 0; m < S; ++m) asm volatile("" : "+r"(o[m]));
      asm volatile("" : "+r"(s2), "+r"(s3));
      if (f <= f_end) {                                     // warp-uniform
        // fb_empty[c & 1] completes each time the service warps have read the fluxes of a chunk c - 1: for the
        // ((c - 1) >> 1)-th time (c odd) or the ((c - 2) >> 1)-th (c even), i.e. phase parity `phase` or `phase ^ 1`
        // with `phase` = (c >> 1) & 1 as for the ring
        FluxStoreWS st{fb + (w + 1) * 32 + lane, FBS, first ? 0u : fbe_bar + 8 * par, par ? phase : phase ^ 1u};
        const bool c2ok = face_flux<DIR, RECON>(N, sm, smp, FS, o, sms, FS, s2, s3, E.visc, E.lam_glob + 3 * DIR, st);
        bad = bad || (!c2ok && lane_ok);
        if (E.pp)                                           // Eq. 20 on this lane's own flux, before the hand-over
          positivity_blend<DIR>(N, sm, smp, FS, o[MA], o[MA + 1], pp_kappa(E, G, DIR), fb + (w + 1) * 32 + lane, FBS);
      }
      named_arrive(BAR_FLUX_READY + par, NT);
      rb += W;
      rb -= rb >= RR ? RR : 0;
      rs += W;
      rs -= rs >= RS ? RS : 0;
      phase ^= par;                                         // each mbarrier is used every other chunk
      par ^= 1;
      first = false;
    }
    if (bad) atomicOr(status, XF_FLAG_NONPHYSICAL);
    return;
  }

  // ============================================================= service warps
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(WS_REGS_SERVICE));
  const int rmax = G.np[DIR] - 1;
  const unsigned deep_bytes = (unsigned)(Nv + 3) * TMA_RW * sizeof(double);
  const unsigned shallow_bytes = (unsigned)(N + 1) * TMA_RW * sizeof(double);
  const int c0 = G.g[0] + blockIdx.x * 32 - lo, co = blockIdx.y + G.g[OD];     // TMA box origin (c0 is even)
  auto stage_row = [&](int slot, int r, unsigned bar) {     // stencil row r (= padded row r) -> ring slot
    const int rc = r < rmax ? r : rmax;
    if (TMA) {                                              // boxes U [Nv][34] and p, c, 1/rho [3][34]
      if (lane == 0) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(sm + (size_t)slot * SLOT);
        tma_load_row(dst, &tmU, c0, DIR == 1 ? rc : co, DIR == 1 ? co : rc, bar);
        tma_load_row(dst + (unsigned)(tma_box_doubles(Nv) * sizeof(double)), &tmP, c0, DIR == 1 ? rc : co,
                     DIR == 1 ? co : rc, bar);
      }
    } else {
      const long long gi = colbase + (long long)rc * sst;
      double *dst = sm + slot * 32 + lane;
#pragma unroll 4
      for (int f = 0; f < NST; ++f)
        cp_async8(dst + f * FS, (f < Nv ? U + (size_t)f * G.cells : prim + (size_t)(f - Nv) * G.cells) + gi);
    }
  };
  auto stage_shallow = [&](int slot, int r, unsigned bar) { // TMA only: box Gamma, chi_s [N + 1][34] of stencil row r
    const int rc = r < rmax ? r : rmax;
    if (lane == 0)
      tma_load_row((unsigned)__cvta_generic_to_shared(sms + (size_t)slot * SSLOT), &tmS, c0, DIR == 1 ? rc : co,
                   DIR == 1 ? co : rc, bar);
  };
  const double dt = stage_dt(E, status);
  const double kappa = E.mode == 3 ? E.alpha / (E.beta * dt) : 0.0;   // mode 3: out = div + kappa U^n (see XfEpilogue)
  const double ninv = -G.inv_d[DIR];
  const bool need_acc = E.mode == 1 || (E.mode == 2 && E.has_acc);
  const bool need_un = (E.mode == 2 && E.alpha != 0.0) || E.mode == 3;

  // cell row of face f (cell f - 1, staged at stencil row f + MA): Eq. 13 and the stage combination
  double d[NVS];
  auto read_fluxes = [&](int ous) {                         // part 1: everything the update needs from shared memory
#pragma unroll
    for (int v = 0; v < NVS; ++v) {
      if (v < Nv) {
        d[v] = (fb[v * FBS + (w + 1) * 32 + lane] - fb[v * FBS + w * 32 + lane]) * ninv;
        if (E.mode == 2) d[v] = fma(dt, d[v], sm[v * FS + ous]);   // U^s + dt div: U^s is still in the ring
      }
    }
    if (w == 0) {                                           // carry the chunk's last face to row 0 (only warp 0 reads row 0)
      for (int v = 0; v < Nv; ++v) fb[v * FBS + lane] = fb[v * FBS + W * 32 + lane];
    }
  };
  // The update reads ONE global operand per component: the partial residual (modes 1, 2 after an earlier sweep) or U^n
  // (mode 3, or mode 2 when this is the only sweep) -- never both (xf_api.cu: residual()).  It is requested BEFORE the
  // service warp waits for the chunk's fluxes, so the loads fly while the compute warps are still at work and the
  // part after the barrier is short.
  const double *__restrict__ opnd_src = need_acc ? E.acc : E.Un;
  const bool need_opnd = need_acc || need_un;
  double opnd[NVS];
  auto load_operands = [&](int f) {
    if (!need_opnd || !(f > f_begin && f <= f_end) || !lane_ok) return;
    const long long gi = colbase + (long long)(f + MA) * sst;
#pragma unroll
    for (int v = 0; v < NVS; ++v)
      if (v < Nv) opnd[v] = opnd_src[v * G.cells + gi];
  };
  auto write_cells = [&](int f) {                           // part 2: Eq. 13 / Eq. 16 and the stores
    if (!(f > f_begin && f <= f_end) || !lane_ok) return;
    const long long gi = colbase + (long long)(f + MA) * sst;
#pragma unroll
    for (int v = 0; v < NVS; ++v) {
      if (v < Nv) {
        const long long idx = v * G.cells + gi;
        if (E.mode == 0) {
          E.out[idx] = d[v];
        } else if (E.mode == 3) {
          E.out[idx] = fma(kappa, opnd[v], d[v]);
        } else if (E.mode == 1) {
          E.out[idx] = opnd[v] + d[v];
        } else {
          const double L = need_acc ? fma(dt, opnd[v], d[v]) : d[v];   // U^s + dt (acc + div)
          E.out[idx] = need_un ? fma(E.alpha, opnd[v], E.beta * L) : E.beta * L;
        }
      }
    }
  };

  // ---- prologue: rows f_begin .. f_begin + W + S - 2 into ring slots 0 .. W + S - 2
  if (TMA) {                                                // shallow rows f_begin + MA .. f_begin + MA + W into slots 0 .. W
    if (lane == 0)
      mbar_expect_tx(full_bar, deep_bytes * (unsigned)((W + S - 1 - w + W - 1) / W) + shallow_bytes * (w == 0 ? 2u : 1u));
    for (int r = w; r < W + 1; r += W) stage_shallow(r, f_begin + MA + r, full_bar);
  }
  for (int r = w; r < W + S - 1; r += W) stage_row(r, f_begin + r, full_bar);
  cp_async_commit();

  int rb = 0, rs = 0, par = 0;
  bool first = true;
  int fprev = 0, ous = 0;
  for (int fc = f_begin; fc <= f_end; fc += W) {
    if (!TMA) {
      cp_async_wait<0>();
      named_arrive(BAR_RING_FULL + par, NT);                // this chunk's rows have landed
    }
    if (!first) {
      load_operands(fprev);
      named_sync(BAR_FLUX_READY + (par ^ 1), NT);           // the previous chunk's fluxes are in fb, its ring rows are dead
      read_fluxes(ous);
      __syncwarp();
      if (lane == 0) mbar_arrive(fbe_bar + 8 * par);
    }
    if (fc + W <= f_end) {                                  // the W new rows of the next chunk: rows fc + W + S - 1 + q
      // warp w fetches row q = (w + MA) mod W: it lands in the ring slot of the previous chunk's row q, and the only
      // service warp that has just read U^s from that slot (stencil row f + MA of its cell row) is warp q - MA = w
      // itself; rows 0 .. MA - 1 hold no cell of the previous chunk.  So no barrier among the service warps is needed.
      const int q = w + MA < W ? w + MA : w + MA - W;
      int slot = rb + W + S - 1 + q;
      slot -= slot >= RR ? RR : 0;
      const unsigned bar = full_bar + 8 * (par ^ 1);
      if (TMA && lane == 0) mbar_expect_tx(bar, deep_bytes + shallow_bytes);
      stage_row(slot, fc + W + S - 1 + q, bar);
      if (TMA) {                                            // shallow row fc + W + MA + 1 + w
        int q = rs + W + 1 + w;
        q -= q >= RS ? RS : 0;
        stage_shallow(q, fc + W + MA + 1 + w, bar);
      }
    }
    cp_async_commit();
    if (!first) write_cells(fprev);
    fprev = fc + w;
    {                                                       // where U^s of that cell row (stencil row f + MA) sits
      int sl = rb + w + MA;
      sl -= sl >= RR ? RR : 0;
      ous = sl * SLOT + lane + lo;
    }
    rb += W;
    rb -= rb >= RR ? RR : 0;
    rs += W;
    rs -= rs >= RS ? RS : 0;
    par ^= 1;
    first = false;
  }
  load_operands(fprev);
  named_sync(BAR_FLUX_READY + (par ^ 1), NT);               // the last chunk
  read_fluxes(ous);
  write_cells(fprev);
}


// ---------------------------------------------------------------------------------------------------------------
// x sweep, warp-specialised with TMA.  The interior rows of one k-plane are contiguous in memory, so a plane is one
// flat pencil (see the top of this file) and a chunk is XW_W x 32 = 128 consecutive faces.  No ring: the chunk's
// 133 stencil cells (+ alignment) are fetched as three dense boxes [fields][136] of a rank-2 tensor {cell, field}
// into one of two stages; the 5-cell overlap between chunks is re-read from L2.  The stencil offsets of a lane are
// then consecutive (immediate offsets in the loads).  Roles and barriers as in the y/z kernel.
// ---------------------------------------------------------------------------------------------------------------
constexpr int XW_W = 4;                    // compute warps = service warps per block
constexpr int XW_CH = XW_W * 32;           // faces per chunk
constexpr int XW_BOX = XW_CH + 8;          // cells per box: 128 + S - 1 (133 or 135) needed, from an even index, 16-byte multiple
constexpr int XW_NCH = 16;                 // chunks per block
constexpr int XW_FBW = XW_CH + 2;          // flux-buffer doubles per component: [0] = last face of the previous chunk
__host__ __device__ constexpr int xw_box_doubles(int nf) { return (nf * XW_BOX * 8 + 127) / 128 * 16; }
__host__ __device__ constexpr int xw_stage_doubles(int N) {
  return xw_box_doubles(N + 4) + xw_box_doubles(3) + xw_box_doubles(N + 1);
}
__host__ __device__ inline size_t xw_smem_doubles(int N) {
  return 2 * (size_t)xw_stage_doubles(N) + (size_t)(N + 4) * XW_FBW + 4;
}
__device__ __forceinline__ void tma_load_span(unsigned dst, const void *tmap, int c0, unsigned bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
      "l"(tmap), "r"(c0), "r"(0), "r"(bar)
      : "memory");
}

template <int N_T, int RECON>
__global__ void __launch_bounds__(64 * XW_W, 2)
sweep_x_ws_kernel(const XfGrid G, const int Nrt, const double *__restrict__ U, const XfEpilogue E,
                  int *__restrict__ status, const int segs_per_plane, const __grid_constant__ CUtensorMap tmU,
                  const __grid_constant__ CUtensorMap tmP, const __grid_constant__ CUtensorMap tmS) {
  constexpr int W = XW_W, NT = 64 * W, FS = XW_BOX;
  constexpr int S = stencil_cells(RECON), HW = S / 2, MA = S / 2 - 1;
  static_assert(XW_CH + S - 1 + 1 <= XW_BOX, "a chunk's stencil cells (+ one for the even start) fit the box");
  const int N = N_T > 0 ? N_T : Nrt;
  const int Nv = N + 4;
  constexpr int NVS = N_T > 0 ? N_T + 4 : XF_MAXNV;
  const int STAGE = xw_stage_doubles(N), OFFP = xw_box_doubles(Nv), OFFS = OFFP + xw_box_doubles(3);
  extern __shared__ __align__(128) double smem[];
  double *fb = smem + 2 * (size_t)STAGE;                    // face fluxes [Nv][XW_FBW]
  const unsigned full_bar = (unsigned)__cvta_generic_to_shared(fb + (size_t)Nv * XW_FBW);
  const unsigned fbe_bar = full_bar + 16;                   // flux buffer consumed (see the y/z kernel)
  if (threadIdx.x == 0 && threadIdx.y == 0) {
    mbar_init(full_bar, 1);
    mbar_init(full_bar + 8, 1);
    mbar_init(fbe_bar, W);
    mbar_init(fbe_bar + 8, W);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const int lane = threadIdx.x;
  const bool service = threadIdx.y >= W;
  const int w = service ? threadIdx.y - W : threadIdx.y;
  const int plane = blockIdx.x / segs_per_plane, seg = blockIdx.x - plane * segs_per_plane;
  const int L = G.n[1] * G.np[0];                           // flat cells of the plane's interior rows
  constexpr int SEGC = XW_NCH * XW_CH - 1;
  const int f_begin = seg * SEGC;                           // faces f_begin .. f_end, cells f_begin .. f_end - 1
  const int f_end = f_begin + SEGC < L ? f_begin + SEGC : L;
  const long long P0 = (long long)(plane + G.g[2]) * G.st[2] + (long long)G.g[1] * G.st[1];  // flat cell 0
  // chunk c needs flat cells fc - HW .. fc + 127 + HW; its boxes start at the even global index below P0 + fc - HW
  const long long g0 = P0 + f_begin - HW;
  const int delta = (int)(g0 & 1);                          // same for every chunk: they are 128 cells apart
  const int u = 32 * w + lane;                              // face within the chunk (compute) / cell slot (service)

  if (!service) {
    // =========================================================== compute warps
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(WS_REGS_COMPUTE));
    int par = 0;
    unsigned phase = 0;
    bool bad = false, first = true;
    for (int fc = f_begin; fc <= f_end; fc += XW_CH) {
      mbar_wait(full_bar + 8 * par, phase);
      const double *st = smem + (size_t)par * STAGE;
      const int f = fc + u;
      int o[S];
#pragma unroll
      for (int m = 0; m < S; ++m) o[m] = u + delta + m;
      // every lane of the block passes the same barriers; lanes past f_end compute on staged (valid or zero) data
      FluxStoreWS fsw{fb + u + 1, XW_FBW, first ? 0u : fbe_bar + 8 * par, par ? phase : phase ^ 1u};
      const bool c2ok = face_flux<0, RECON>(N, st, st + OFFP, FS, o, st + OFFS, FS, o[MA], o[MA + 1], E.visc, E.lam_glob, fsw);
      if (E.pp) positivity_blend<0>(N, st, st + OFFP, FS, o[MA], o[MA + 1], pp_kappa(E, G, 0), fb + u + 1, XW_FBW);
      {
        const int ia = (f - 1 + G.np[0]) % G.np[0], ib = f % G.np[0];
        const bool used = f <= f_end && ((ia >= G.g[0] && ia < G.g[0] + G.n[0]) || (ib >= G.g[0] && ib < G.g[0] + G.n[0]));
        bad = bad || (!c2ok && used);
      }
      named_arrive(BAR_FLUX_READY + par, NT);
      phase ^= par;
      par ^= 1;
      first = false;
    }
    if (bad) atomicOr(status, XF_FLAG_NONPHYSICAL);
    return;
  }
  // ============================================================= service warps
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(WS_REGS_SERVICE));
  const unsigned stage_bytes = (unsigned)(2 * N + 8) * XW_BOX * sizeof(double);
  auto stage_chunk = [&](int fc, int st) {                  // the three boxes of chunk fc -> stage st (one lane issues)
    if (w != 0 || lane != 0) return;
    const unsigned bar = full_bar + 8 * st;
    const unsigned dst = (unsigned)__cvta_generic_to_shared(smem + (size_t)st * STAGE);
    const int c0 = (int)(P0 + fc - HW - delta);             // even; may be negative or run past the array: zero-filled
    mbar_expect_tx(bar, stage_bytes);
    tma_load_span(dst, &tmU, c0, bar);
    tma_load_span(dst + (unsigned)(OFFP * sizeof(double)), &tmP, c0, bar);
    tma_load_span(dst + (unsigned)(OFFS * sizeof(double)), &tmS, c0, bar);
  };
  const double dt = stage_dt(E, status);
  const double kappa = E.mode == 3 ? E.alpha / (E.beta * dt) : 0.0;   // mode 3: out = div + kappa U^n (see XfEpilogue)
  const double ninv = -G.inv_d[0];
  const bool need_acc = E.mode == 1 || (E.mode == 2 && E.has_acc);
  const bool need_un = (E.mode == 2 && E.alpha != 0.0) || E.mode == 3;

  // lane (w, lane) of the service group owns slot u of a chunk: cell fc + u - 1, between the chunk's faces u - 1 and u
  double d[NVS];
  auto read_fluxes = [&](int st) {                          // st: stage of the chunk whose cells are updated
    const double *us = smem + (size_t)st * STAGE + u + delta + MA;  // cell fc + u - 1 = stencil cell m = MA of face fc + u
#pragma unroll
    for (int v = 0; v < NVS; ++v) {
      if (v < Nv) {
        d[v] = (fb[v * XW_FBW + u + 1] - fb[v * XW_FBW + u]) * ninv;
        if (E.mode == 2) d[v] = fma(dt, d[v], us[v * FS]);   // U^s + dt div: U^s is still in the stage
      }
    }
    __syncwarp();
    if (w == 0 && lane < Nv) fb[lane * XW_FBW] = fb[lane * XW_FBW + XW_CH];   // carry: only slot 0 (this warp) reads [0]
  };
  auto cell_index = [&](int fc, long long &gi) -> bool {    // global index of this lane's cell; false if it is not updated
    const int cf = fc + u - 1;
    gi = P0 + cf;
    if (cf < f_begin || cf >= f_end) return false;
    const int i = cf % G.np[0];
    return i >= G.g[0] && i < G.g[0] + G.n[0];
  };
  // one global operand per component, requested before the wait for the chunk's fluxes (see the y/z kernel)
  const double *__restrict__ opnd_src = need_acc ? E.acc : E.Un;
  const bool need_opnd = need_acc || need_un;
  double opnd[NVS];
  auto load_operands = [&](int fc) {
    long long gi;
    if (!need_opnd || !cell_index(fc, gi)) return;
#pragma unroll
    for (int v = 0; v < NVS; ++v)
      if (v < Nv) opnd[v] = opnd_src[v * G.cells + gi];
  };
  auto write_cells = [&](int fc) {
    long long gi;
    if (!cell_index(fc, gi)) return;
#pragma unroll
    for (int v = 0; v < NVS; ++v) {
      if (v < Nv) {
        const long long idx = v * G.cells + gi;
        if (E.mode == 0) {
          E.out[idx] = d[v];
        } else if (E.mode == 3) {
          E.out[idx] = fma(kappa, opnd[v], d[v]);
        } else if (E.mode == 1) {
          E.out[idx] = opnd[v] + d[v];
        } else {
          const double Lr = need_acc ? fma(dt, opnd[v], d[v]) : d[v];   // U^s + dt (acc + div)
          E.out[idx] = need_un ? fma(E.alpha, opnd[v], E.beta * Lr) : E.beta * Lr;
        }
      }
    }
  };

  stage_chunk(f_begin, 0);
  int par = 0, fprev = 0;
  bool first = true;
  for (int fc = f_begin; fc <= f_end; fc += XW_CH) {
    if (!first) {
      load_operands(fprev);
      named_sync(BAR_FLUX_READY + (par ^ 1), NT);           // the previous chunk's fluxes are in fb, its stage is free
      read_fluxes(par ^ 1);
      __syncwarp();
      if (lane == 0) mbar_arrive(fbe_bar + 8 * par);
      if (E.mode == 2) named_sync(BAR_SERVICE, 32 * W);     // U^s was read from the stage the next copy overwrites
    }
    if (fc + XW_CH <= f_end) stage_chunk(fc + XW_CH, par ^ 1);
    if (!first) write_cells(fprev);
    fprev = fc;
    par ^= 1;
    first = false;
  }
  load_operands(fprev);
  named_sync(BAR_FLUX_READY + (par ^ 1), NT);               // the last chunk
  read_fluxes(par ^ 1);
  write_cells(fprev);
}

}  // namespace xf

// Host side of the TMA path: a rank-4 tensor map {i, j, k, field} over `nf` consecutive fields of the padded box, with
// one box = 34 cells along i (from an even index) of every field.  Returns false where TMA cannot describe the array (odd padded extents
// make the strides no multiple of 16 bytes, or an unaligned base): the launcher then takes the cp.async kernel.
typedef CUresult (*XfTensorMapEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                        const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                        CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                        CUtensorMapFloatOOBfill);
inline XfTensorMapEncodeFn xf_tensor_map_encoder() {
  static XfTensorMapEncodeFn encode = [] {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      fn = nullptr;
    return reinterpret_cast<XfTensorMapEncodeFn>(fn);
  }();
  return encode;
}
inline bool xf_row_tensor_map(CUtensorMap *tm, const XfGrid &G, const double *base, int nf) {
  XfTensorMapEncodeFn encode = xf_tensor_map_encoder();
  if (!encode || (G.np[0] & 1) || (G.cells & 1) || (reinterpret_cast<uintptr_t>(base) & 15)) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)G.np[0], (cuuint64_t)G.np[1], (cuuint64_t)G.np[2], (cuuint64_t)nf};
  const cuuint64_t strides[3] = {(cuuint64_t)G.st[1] * 8, (cuuint64_t)G.st[2] * 8, (cuuint64_t)G.cells * 8};
  const cuuint32_t box[4] = {xf::TMA_RW, 1, 1, (cuuint32_t)nf};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double *>(base), dims, strides, box, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// x sweep: a rank-2 map {flat cell, field}; one box = XW_BOX consecutive cells (from an even index) of every field.
inline bool xf_span_tensor_map(CUtensorMap *tm, const XfGrid &G, const double *base, int nf) {
  XfTensorMapEncodeFn encode = xf_tensor_map_encoder();
  if (!encode || (G.cells & 1) || (reinterpret_cast<uintptr_t>(base) & 15)) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)G.cells, (cuuint64_t)nf};
  const cuuint64_t strides[1] = {(cuuint64_t)G.cells * 8};
  const cuuint32_t box[2] = {xf::XW_BOX, (cuuint32_t)nf};
  const cuuint32_t estr[2] = {1, 1};
  return encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double *>(base), dims, strides, box, estr,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// cached tensor map of `nf` fields at `base` (kind 0: row map, 1: span map); nullptr where TMA cannot describe the array
inline const CUtensorMap *xf_tmap(XfTmapCache *c, const XfGrid &G, const double *base, int nf, int kind) {
  for (int q = 0; q < c->n; ++q)
    if (c->e[q].base == base && c->e[q].nf == nf && c->e[q].kind == kind) return c->e[q].ok ? &c->e[q].tm : nullptr;
  const int cap = (int)(sizeof(c->e) / sizeof(c->e[0]));
  XfTmapCache::Entry &en = c->e[c->n < cap ? c->n++ : (c->next = (c->next + 1) % cap)];
  en.base = base;
  en.nf = nf;
  en.kind = kind;
  en.ok = kind == 0 ? xf_row_tensor_map(&en.tm, G, base, nf) : xf_span_tensor_map(&en.tm, G, base, nf);
  return en.ok ? &en.tm : nullptr;
}

#define XF_DISPATCH_SWEEP_N(N, CALL) \
  switch (N) {                       \
    case 1: { CALL(1); break; }      \
    case 2: { CALL(2); break; }      \
    case 3: { CALL(3); break; }      \
    case 4: { CALL(4); break; }      \
    case 10: { CALL(10); break; }    \
    default: { CALL(0); break; }     \
  }
