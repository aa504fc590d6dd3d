"""Domain decomposition and halo exchange around the C-ABI.

The paper's scheme: a Cartesian decomposition px x py x pz, one block per GPU / rank; before every residual evaluation
each block sends the ng "border" layers next to a shared face to its face neighbour, where they become the "boundary"
(ghost) layers; one scalar reduction (the global time step) per step.  Everything that touches field data runs in the
library's kernels (``xf_fill_ghosts_dir``, ``xf_pack_halo``, ``xf_unpack_halo``, ``xf_rk3_stage``, ``xf_max_wavespeed``);
this module is plumbing only: who is whose neighbour, which buffer goes where, and the transfer itself --

* ``DistTransport``: one block per process, ``torch.distributed`` point-to-point (``batch_isend_irecv``: NCCL send / recv
  over NVLink on GPUs; any backend works, the CPU test drives it over gloo) and ``all_reduce(MAX)`` for the wave speed;
* ``LocalTransport``: several blocks in ONE process on one device, device-to-device copies -- how the decomposition is
  verified on a single GPU: a run on 2 x 2 x 2 blocks must reproduce the single-block run BIT FOR BIT, because every
  cell sees the same stencil values and the same arithmetic.

Directions are exchanged in the order x, y, z, each over the padded extent of the directions already done (as the
physical ghost fill, reading R10), so edge and corner ghosts arrive without diagonal messages.  Not supported
across blocks: XF_VISC_GLF (its global maxima would need one more reduction per residual evaluation).
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

BC_PERIODIC, BC_EXCHANGE = 0, 4
Coord = Tuple[int, int, int]


def _split(n: int, p: int) -> List[Tuple[int, int]]:
    """p contiguous pieces of n cells, sizes differing by at most one -> [(offset, size)]"""
    base, rem = divmod(n, p)
    out, off = [], 0
    for q in range(p):
        size = base + (1 if q < rem else 0)
        out.append((off, size))
        off += size
    return out


@dataclass
class BlockSpec:
    coord: Coord
    offset: Tuple[int, int, int]      # first interior cell of the block in the global interior numbering (x, y, z)
    n: Tuple[int, int, int]           # interior cells (x, y, z)
    bc: Tuple[int, ...]               # local boundary kinds: the global one on a physical face, BC_EXCHANGE on a shared one
    neighbour: Dict[Tuple[int, int], Optional[Coord]]   # (direction, side) -> coordinates of the face neighbour


class Decomposition:
    """Cartesian decomposition of a global box.  A periodic direction split over p > 1 blocks turns
    into exchange faces all the way round; with p = 1 it stays a local periodic fill."""

    def __init__(self, n: Sequence[int], procs: Sequence[int], bc: Sequence[int], ng: int = 3):
        self.n, self.procs, self.bc, self.ng = tuple(int(v) for v in n), tuple(int(v) for v in procs), tuple(bc), int(ng)
        for d in range(3):
            if self.procs[d] < 1 or (self.n[d] == 1 and self.procs[d] != 1):
                raise ValueError("an inactive direction cannot be split")
            if self.procs[d] > 1 and self.n[d] // self.procs[d] < self.ng:
                raise ValueError("every block needs at least ng interior cells per split direction")
        self.pieces = [_split(self.n[d], self.procs[d]) for d in range(3)]

    @property
    def coords(self) -> List[Coord]:
        px, py, pz = self.procs
        return [(i, j, k) for k in range(pz) for j in range(py) for i in range(px)]

    def rank_of(self, c: Coord) -> int:
        return (c[2] * self.procs[1] + c[1]) * self.procs[0] + c[0]

    def coord_of(self, rank: int) -> Coord:
        px, py, _ = self.procs
        return (rank % px, (rank // px) % py, rank // (px * py))

    def block(self, c: Coord) -> BlockSpec:
        bc = list(self.bc)
        nb: Dict[Tuple[int, int], Optional[Coord]] = {}
        for d in range(3):
            p = self.procs[d]
            periodic = self.bc[2 * d] == BC_PERIODIC
            for side in (0, 1):
                q = c[d] + (1 if side else -1)
                other: Optional[Coord] = None
                if p > 1 and (0 <= q < p or periodic):
                    o = list(c)
                    o[d] = q % p
                    other = tuple(o)
                    bc[2 * d + side] = BC_EXCHANGE
                nb[(d, side)] = other
        off = tuple(self.pieces[d][c[d]][0] for d in range(3))
        n = tuple(self.pieces[d][c[d]][1] for d in range(3))
        return BlockSpec(coord=c, offset=off, n=n, bc=tuple(bc), neighbour=nb)


class Block:
    """One block of the decomposition on one device: its context, fields, stage arrays and face buffers."""

    def __init__(self, spec: BlockSpec, ctx, U, T):
        import torch

        self.spec, self.ctx, self.U, self.T = spec, ctx, U, T
        self.U1, self.U2 = torch.empty_like(U), torch.empty_like(U)
        self.work = ctx.workspace()
        self.S = torch.zeros(1, dtype=torch.float64, device=U.device)
        self.send: Dict[Tuple[int, int], "torch.Tensor"] = {}
        self.recv: Dict[Tuple[int, int], "torch.Tensor"] = {}
        for (d, side), other in spec.neighbour.items():
            if other is not None:
                m = ctx.xf_halo_doubles(d)
                self.send[(d, side)] = torch.empty(m, dtype=torch.float64, device=U.device)
                self.recv[(d, side)] = torch.empty(m, dtype=torch.float64, device=U.device)


class LocalTransport:
    """All blocks live in this process: a face buffer travels by a device copy."""

    def __init__(self, blocks: Dict[Coord, Block]):
        self.blocks = blocks

    def exchange(self, d: int) -> None:
        for b in self.blocks.values():
            for side in (0, 1):
                other = b.spec.neighbour[(d, side)]
                if other is not None:      # my side-`side` border becomes the neighbour's ghost layers on its opposite side
                    self.blocks[other].recv[(d, 1 - side)].copy_(b.send[(d, side)])

    def max(self, values: List[float]) -> float:
        return max(values)


class DistTransport:
    """One block per process; ``torch.distributed`` is initialised by the caller (backend "nccl" on GPUs).  Point-to-point
    messages between a pair of ranks are matched in posting order (NCCL has no tags): sends go out low side first, and
    the receives are posted in the order the NEIGHBOUR sends -- its low-side border is my high-side ghost."""

    def __init__(self, decomp: Decomposition, block, dist=None):
        if dist is None:
            import torch.distributed as dist
        self.dist, self.decomp, self.block = dist, decomp, block
        self.blocks = {block.spec.coord: block}

    def exchange(self, d: int) -> None:
        b, ops = self.block, []
        for side in (0, 1):
            other = b.spec.neighbour[(d, side)]
            if other is not None:
                ops.append(self.dist.P2POp(self.dist.isend, b.send[(d, side)], self.decomp.rank_of(other)))
        for side in (1, 0):
            other = b.spec.neighbour[(d, side)]
            if other is not None:
                ops.append(self.dist.P2POp(self.dist.irecv, b.recv[(d, side)], self.decomp.rank_of(other)))
        if ops:
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()

    def max(self, values: List[float]) -> float:
        import torch

        t = torch.tensor([max(values)], dtype=torch.float64, device=self.block.S.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())


class Solver:
    """SSP-RK3 time stepping of a decomposed box: per stage, for each direction in turn, physical ghost fill, pack, transfer,
    unpack; then the stage's residual and combination in every block (``xf_rk3_stage``)."""

    def __init__(self, transport):
        self.tr = transport
        self.blocks: Dict[Coord, Block] = transport.blocks

    def fill_and_exchange(self, which: str) -> None:
        for d in range(3):
            for b in self.blocks.values():
                U = getattr(b, which)
                if b.spec.n[d] > 1:
                    b.ctx.xf_fill_ghosts_dir(U, d)
                for (dd, side), buf in b.send.items():
                    if dd == d:
                        b.ctx.xf_pack_halo(U, b.T, d, side, buf)
            self.tr.exchange(d)
            for b in self.blocks.values():
                U = getattr(b, which)
                for (dd, side), buf in b.recv.items():
                    if dd == d:
                        b.ctx.xf_unpack_halo(U, b.T, d, side, buf)

    def max_wavespeed(self) -> float:
        vals = []
        for b in self.blocks.values():
            b.ctx.xf_max_wavespeed(b.U, b.T, b.S)
            vals.append(float(b.S.item()))
        return self.tr.max(vals)

    def step(self, dt: float) -> None:
        for stage, (src, dst) in enumerate((("U", "U1"), ("U1", "U2"), ("U2", "U"))):
            self.fill_and_exchange(src)
            for b in self.blocks.values():
                b.ctx.xf_rk3_stage(stage, b.U, getattr(b, src), getattr(b, dst), b.T, dt, b.work)

    def step_cfl(self, cfl: float) -> float:
        dt = cfl / self.max_wavespeed()
        self.step(dt)
        return dt


def make_blocks(wl, procs: Sequence[int], coords: Optional[Sequence[Coord]] = None, device: int = 0, **ctx_kw):
    """Cut a global workload (workloads.Workload: padded numpy U, T_guess) into the blocks ``coords`` (default: all) of a
    ``procs`` decomposition, each with its own context on ``device``.  -> (Decomposition, {coord: Block})"""
    import torch

    from . import xf

    ng = getattr(wl, "ng", 3)
    dec = Decomposition((wl.nx, wl.ny, wl.nz), procs, wl.bc, ng)
    g = [ng if m > 1 else 0 for m in (wl.nx, wl.ny, wl.nz)]
    t = wl.table
    blocks: Dict[Coord, Block] = {}
    for c in (dec.coords if coords is None else coords):
        spec = dec.block(c)
        sl = [slice(spec.offset[d], spec.offset[d] + spec.n[d] + 2 * g[d]) for d in range(3)]   # padded window, global ghosts included
        U = np.ascontiguousarray(wl.U[:, sl[2], sl[1], sl[0]])
        T = np.ascontiguousarray(wl.T_guess[sl[2], sl[1], sl[0]])
        ctx = xf.Context(spec.n[0], spec.n[1], spec.n[2], wl.dx, wl.dy, wl.dz, t.W, t.nasa7, t.Ru, t.Tlo, t.Thi, spec.bc,
                         wl.bc_state, device=device, ng=ng, **ctx_kw)
        blocks[c] = Block(spec, ctx, torch.from_numpy(U).to(f"cuda:{device}"), torch.from_numpy(T).to(f"cuda:{device}"))
    return dec, blocks


def gather_interior(wl, dec: Decomposition, blocks: Dict[Coord, Block], which: str = "U") -> np.ndarray:
    """the global interior field [Nv, nz, ny, nx] assembled from the blocks' interiors"""
    ng = dec.ng
    g = [ng if m > 1 else 0 for m in dec.n]
    out = np.zeros((blocks[next(iter(blocks))].U.shape[0], dec.n[2], dec.n[1], dec.n[0]))
    for b in blocks.values():
        A = getattr(b, which).cpu().numpy()
        o, n = b.spec.offset, b.spec.n
        out[:, o[2]:o[2] + n[2], o[1]:o[1] + n[1], o[0]:o[0] + n[0]] = \
            A[:, g[2]:g[2] + n[2], g[1]:g[1] + n[1], g[0]:g[0] + n[0]]
    return out
