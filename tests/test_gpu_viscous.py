"""-m gpu parity of the viscous / diffusive right-hand side (Eq. 1-6, 155-178,
505-513; readings R19-R23) on the CUDA path (csrc/xf_visc.cu) against the oracle (xo_viscous_rhs,
xo_rk3_step_ns): 1e-12 per residual evaluation, 1e-9 over steps, per variable (the momentum rows share their scale).
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RHS_TOL = 1e-12
STEPS_TOL = 1e-9


def rhs_tol(w):
    """div F_v is a SECOND difference: rounding the O(u, T, Y) cell values (eps |f|) is divided by dx^2 on both sides, while
    the residual itself is |f''| ~ k^2 |f|: the common round-off floor relative to the residual grows like (cells per
    wavelength)^2.  The seeded boxes hold modes up to wavenumber 2 per unit length; 1e-12 is held up to 32 cells per unit
    length and scaled by (n / 32)^2 beyond."""
    n = max(w.nx, w.ny, w.nz)
    return RHS_TOL * max(1.0, (n / 32.0) ** 2)


def _gpu(w, **kw):
    from gpu_helpers import GpuRun

    return GpuRun(w, **kw)


def field_err(a, b):
    nv = a.shape[0]
    a2, b2 = a.reshape(nv, -1), b.reshape(nv, -1)
    den = np.abs(b2).max(axis=1)
    den[1:4] = den[1:4].max()
    den[0] = max(den[0], den[4] * 1e-300)                      # the density row of div F_v is identically zero
    return np.abs(a2 - b2).max(axis=1) / np.maximum(den, 1e-300)


def state_err(w, a, b, cmax):
    nv = a.shape[0]
    ai, bi = w.interior(a).reshape(nv, -1), w.interior(b).reshape(nv, -1)
    den = np.abs(bi).max(axis=1)
    den[1:4] = np.abs(bi[0]).max() * cmax
    return np.abs(ai - bi).max(axis=1) / np.maximum(den, 1e-300)


# 1-D / 2-D / 3-D, every species-count instantiation, extents around the tile sizes (x: 253 cells per block, y/z: 13 cell
# rows x 32 lanes), even and odd, every boundary kind
CASES = [((64, 1, 1), 1, (0,) * 6), ((600, 1, 1), 2, (1, 1, 0, 0, 0, 0)), ((1, 41, 1), 3, (0,) * 6), ((1, 1, 27), 2, (0, 0, 0, 0, 2, 1)),
         ((70, 36, 1), 4, (3, 1, 2, 2, 0, 0)), ((33, 14, 1), 3, (0,) * 6), ((36, 30, 22), 4, (0,) * 6),
         ((21, 13, 27), 5, (1, 2, 2, 1, 0, 0)), ((40, 12, 10), 10, (3, 1, 2, 2, 2, 2)), ((3, 3, 3), 2, (0,) * 6),
         ((254, 5, 4), 2, (0,) * 6), ((19, 9, 8), 16, (0,) * 6)]


@pytest.mark.parametrize("shape,n,bc", CASES)
def test_viscous_rhs_parity(oracle_mod, shape, n, bc):
    w = wl.random_smooth_box(*shape, nspecies=n, seed=9000 + n + shape[0], bc=bc)
    tr = wl.synthetic_transport(w.table, seed=n)
    orc = oracle_mod.Oracle.from_workload(w)
    Uo, To = w.U.copy(), w.T_guess.copy()
    orc.rhs(Uo, To)                                            # ghosts filled, T converged on every padded cell
    rv = orc.viscous_rhs(oracle_mod.make_transport(tr), Uo, To)
    g = _gpu(w, transport=tr)
    import torch

    g.rhs()                                                    # the same on the device
    out = torch.zeros_like(g.U)
    g.ctx.xf_viscous_rhs(g.U, g.T, out, g.work)
    assert g.ctx.xf_status() == 0
    err = field_err(w.interior(out.cpu().numpy()), w.interior(rv))
    assert err[1:].max() < rhs_tol(w), err
    assert float(np.abs(w.interior(out.cpu().numpy())[0]).max()) == 0.0
    g.close()


def test_viscous_rhs_on_shocked_states_and_with_four_ghost_layers(oracle_mod):
    for ng, recon in ((3, 0), (4, 2)):
        w = wl.config3_shock_bubble_3d(24)
        if ng == 4:
            w = wl.with_ghost_width(w, 4)
        tr = wl.synthetic_transport(w.table, seed=3)
        orc = oracle_mod.Oracle.from_workload(w, recon=recon)
        Uo, To = w.U.copy(), w.T_guess.copy()
        orc.rhs(Uo, To)
        rv = orc.viscous_rhs(oracle_mod.make_transport(tr), Uo, To)
        g = _gpu(w, transport=tr, reconstruction=recon)
        import torch

        g.rhs()
        out = torch.zeros_like(g.U)
        g.ctx.xf_viscous_rhs(g.U, g.T, out, g.work)
        err = field_err(w.interior(out.cpu().numpy()), w.interior(rv))
        assert err[1:].max() < rhs_tol(w), err
        g.close()


@pytest.mark.parametrize("shape,n,steps", [((48, 1, 1), 2, 30), ((30, 26, 1), 3, 20), ((24, 20, 18), 4, 12), ((16, 14, 12), 10, 6)])
def test_navier_stokes_rk3_steps_parity(oracle_mod, shape, n, steps):
    """xf_rk3_step of a context with a transport table integrates convective + viscous residual: parity with
    xo_rk3_step_ns after every step; the device-dt variant (xf_step_cfl) gives the same state as the host-dt one."""
    w = wl.random_smooth_box(*shape, nspecies=n, seed=9100 + n)
    tr = wl.synthetic_transport(w.table, seed=n + 7, mu0=5e-3)
    ot = oracle_mod.make_transport(tr)
    orc = oracle_mod.Oracle.from_workload(w)
    Uo, To = w.U.copy(), w.T_guess.copy()
    g = _gpu(w, transport=tr)
    g2 = _gpu(w, transport=tr)
    worst = 0.0
    for _ in range(steps):
        S = orc.max_wavespeed(Uo, To)
        dt = 0.4 / S
        assert orc.rk3_step_ns(ot, Uo, To, dt) == 0
        g.step(dt)
        g2.ctx.xf_step_cfl(g2.U, g2.T, 0.4, g2.S, g2.work)
        cmax = S * min(w.dx, w.dy if w.ny > 1 else 1e300, w.dz if w.nz > 1 else 1e300)
        worst = max(worst, state_err(w, g.host_U(), Uo, cmax).max(), state_err(w, g2.host_U(), Uo, cmax).max())
    assert g.ctx.xf_status() == 0 and g2.ctx.xf_status() == 0
    assert worst < STEPS_TOL, worst
    g.close()
    g2.close()


def test_viscous_shock_tube_100_steps(oracle_mod):
    w = wl.config1_shock_tube()
    tr = wl.synthetic_transport(w.table, seed=1, mu0=2e-4, T0=30.0)   # T = p W / (rho Ru) is 28 .. 4 here
    ot = oracle_mod.make_transport(tr)
    orc = oracle_mod.Oracle.from_workload(w)
    Uo, To = w.U.copy(), w.T_guess.copy()
    g = _gpu(w, transport=tr)
    worst = 0.0
    for _ in range(100):
        S = orc.max_wavespeed(Uo, To)
        dt = w.cfl / S
        assert orc.rk3_step_ns(ot, Uo, To, dt) == 0
        g.step(dt)
        worst = max(worst, state_err(w, g.host_U(), Uo, S * w.dx).max())
    assert g.ctx.xf_status() == 0
    assert worst < STEPS_TOL, worst
    g.close()


def test_viscous_rhs_needs_a_transport_table():
    from paper_2403_05910_b200 import xf
    import torch

    w = wl.random_smooth_box(12, 10, 1, nspecies=2, seed=1)
    g = _gpu(w)
    out = torch.zeros_like(g.U)
    with pytest.raises(xf.XfError):
        g.ctx.xf_viscous_rhs(g.U, g.T, out, g.work)
    g.close()
