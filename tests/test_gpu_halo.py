"""-m gpu: the domain decomposition and halo exchange verified on ONE GPU:
several blocks of a Cartesian decomposition live in one process (halo.LocalTransport: face buffers travel by device
copies; the same xf_fill_ghosts_dir / xf_pack_halo / xf_unpack_halo / xf_rk3_stage calls a multi-GPU run makes), and the
decomposed run must reproduce the single-block run -- bit for bit where no periodic direction is split (every cell then
sees the same stencil values, the same Newton guess and the same arithmetic), to 1e-12 where one is (the single block's
periodic ghost cells keep their own Newton guess, the split run's receive the neighbour's: both converge to 1e-13).
The transfer over torch.distributed is covered on CPU over gloo (tests/test_multirank_cpu.py).
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _single(w, steps, cfl, **kw):
    from gpu_helpers import GpuRun

    g = GpuRun(w, **kw)
    dts = []
    for _ in range(steps):
        S = g.max_wavespeed()
        dts.append(cfl / S)
        g.step(dts[-1])
    assert g.ctx.xf_status() == 0
    U = w.interior(g.host_U()).copy()
    g.close()
    return U, dts


def _decomposed(w, procs, steps, cfl, **kw):
    from paper_2403_05910_b200 import halo

    dec, blocks = halo.make_blocks(w, procs, **kw)
    sol = halo.Solver(halo.LocalTransport(blocks))
    dts = [sol.step_cfl(cfl) for _ in range(steps)]
    for b in blocks.values():
        assert b.ctx.xf_status() == 0
    U = halo.gather_interior(w, dec, blocks)
    for b in blocks.values():
        b.ctx.close()
    return U, dts


@pytest.mark.parametrize("shape,n,bc,procs", [
    ((64, 1, 1), 2, (1, 1, 0, 0, 0, 0), (4, 1, 1)),
    ((48, 40, 1), 3, (3, 1, 2, 2, 0, 0), (2, 3, 1)),
    ((36, 30, 24), 4, (1, 2, 2, 1, 3, 1), (2, 2, 2)),
    ((33, 27, 20), 2, (2, 2, 1, 1, 1, 1), (3, 1, 2)),          # uneven pieces, odd extents (fallback kernels)
])
def test_decomposed_run_is_bitwise_the_single_block_run(shape, n, bc, procs):
    w = wl.random_smooth_box(*shape, nspecies=n, seed=600 + n, bc=bc)
    U1, dt1 = _single(w, 4, 0.4)
    U2, dt2 = _decomposed(w, procs, 4, 0.4)
    assert dt1 == dt2                                          # the reduced max wave speed is the global one, exactly
    assert np.array_equal(U1, U2)


def test_split_periodic_directions_and_shocked_data():
    w = wl.config3_shock_bubble_3d(32)                         # x: Dirichlet / transmissive, y, z periodic
    U1, dt1 = _single(w, 6, 0.5)
    U2, dt2 = _decomposed(w, (2, 2, 2), 6, 0.5)
    assert np.allclose(dt1, dt2, rtol=1e-13, atol=0)
    nv = U1.shape[0]
    den = np.abs(U1).reshape(nv, -1).max(axis=1)
    den[1:4] = np.abs(U1[0]).max() * np.sqrt(2.0)
    assert (np.abs(U1 - U2).reshape(nv, -1).max(axis=1) / den).max() < 1e-12


def test_decomposed_run_with_weno7_limiter_and_viscous_terms():
    """four ghost layers travel, the limiter and the viscous stencil read exchanged ghosts incl. edges and corners"""
    w = wl.with_ghost_width(wl.rough_box(24, 20, 18, nspecies=3, seed=8, bc=(1, 1, 2, 2, 1, 1)), 4)
    tr = wl.synthetic_transport(w.table, seed=5, mu0=1e-3)
    kw = dict(reconstruction=2, positivity=True, transport=tr)
    U1, dt1 = _single(w, 3, 0.15, **kw)
    U2, dt2 = _decomposed(w, (2, 2, 2), 3, 0.15, **kw)
    assert dt1 == dt2
    assert np.array_equal(U1, U2)
