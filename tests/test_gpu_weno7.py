"""-m gpu parity of the WENO7 reconstruction ("WENO7 [36]", validated at
PAPER.md:523; reading R18) on the CUDA path against the oracle (oracle/xf_oracle.c: xo_weno7).

WENO7 reaches one cell further than WENO5 / WENO-CU6 (stencil i-3..i+4): the context carries ng = 4 ghost layers, the
rings of the sweeps are two rows deeper and the boxes of the x sweep two cells wider.  Same bar as the other
reconstructions: 1e-12 per RHS, 1e-9 over steps, bit-exact ghost fill.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RHS_TOL = 1e-12
STEPS_TOL = 1e-9
W7 = 2   # XF_RECON_WENO7


def _gpu(w, **kw):
    from gpu_helpers import GpuRun

    return GpuRun(w, **kw)


def field_err(a, b):
    nv = a.shape[0]
    a2, b2 = a.reshape(nv, -1), b.reshape(nv, -1)
    den = np.abs(b2).max(axis=1)
    den[1:4] = den[1:4].max()
    return np.abs(a2 - b2).max(axis=1) / np.maximum(den, 1e-300)


def state_err(w, a, b, cmax):
    nv = a.shape[0]
    ai, bi = w.interior(a).reshape(nv, -1), w.interior(b).reshape(nv, -1)
    den = np.abs(bi).max(axis=1)
    den[1:4] = np.abs(bi[0]).max() * cmax
    return np.abs(ai - bi).max(axis=1) / np.maximum(den, 1e-300)


@pytest.mark.parametrize("shape", [(17, 1, 1), (9, 12, 1), (8, 5, 7), (1, 7, 9)])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0, 0, 0), (1, 1, 2, 2, 1, 2), (3, 1, 2, 1, 3, 3)])
def test_ghost_fill_four_layers_bit_exact(oracle_mod, shape, bc):
    import torch

    w = wl.with_ghost_width(wl.random_smooth_box(*shape, nspecies=3, seed=5, bc=bc), 4)
    rng = np.random.default_rng(9)
    U = rng.normal(size=w.U.shape)                            # ghosts hold garbage before the fill
    U[(slice(None),) + tuple(slice(4, -4) if m > 1 else slice(None) for m in (w.nz, w.ny, w.nx))] = w.interior(w.U)
    orc = oracle_mod.Oracle.from_workload(w, recon=W7)
    Uo = U.copy()
    orc.fill_ghosts(Uo)
    g = _gpu(w, reconstruction=W7)
    Ud = torch.from_numpy(U.copy()).cuda()
    g.ctx.xf_fill_ghosts(Ud)
    assert np.array_equal(Ud.cpu().numpy(), Uo)
    g.close()


# even extents -> TMA kernels, odd -> the fallbacks; several x chunks; every species-count instantiation
CASES = [((400, 1, 1), 1, (0,) * 6), ((1031, 1, 1), 2, (1, 1, 0, 0, 0, 0)), ((1, 70, 1), 2, (0,) * 6),
         ((1, 1, 45), 4, (0, 0, 0, 0, 2, 1)), ((150, 37, 1), 3, (3, 1, 2, 2, 0, 0)), ((150, 38, 1), 3, (3, 1, 2, 2, 0, 0)),
         ((45, 19, 23), 4, (3, 1, 0, 0, 0, 0)), ((70, 10, 8), 10, (3, 1, 2, 2, 2, 2)), ((34, 36, 38), 1, (0,) * 6),
         ((20, 18, 40), 7, (1, 2, 2, 1, 0, 0)), ((131, 6, 5), 16, (0,) * 6), ((4, 4, 4), 2, (0,) * 6),
         ((5, 4, 6), 5, (1, 1, 2, 2, 0, 0))]


@pytest.mark.parametrize("shape,n,bc", CASES)
def test_rhs_parity_weno7(oracle_mod, shape, n, bc):
    if shape[0] > 1000:
        w = wl.config1_shock_tube(nx=shape[0])               # long pencil: shock-tube data
    else:
        w = wl.random_smooth_box(*shape, nspecies=n, seed=7000 + n + shape[0], bc=bc)
    w = wl.with_ghost_width(w, 4)
    orc = oracle_mod.Oracle.from_workload(w, recon=W7)
    Uo, To = w.U.copy(), w.T_guess.copy()
    ro = orc.rhs(Uo, To)
    assert orc.last_status == 0
    g = _gpu(w, reconstruction=W7)
    err = field_err(w.interior(g.rhs()), w.interior(ro))
    assert err.max() < RHS_TOL, err
    assert np.array_equal(g.host_U(), Uo)                     # ghosts filled identically, interior untouched
    g.close()


@pytest.mark.parametrize("visc", [1, 2])
@pytest.mark.parametrize("shape,n,bc", [((150, 38, 1), 3, (3, 1, 2, 2, 0, 0)), ((45, 19, 23), 4, (3, 1, 0, 0, 0, 0)),
                                         ((70, 10, 8), 10, (3, 1, 2, 2, 2, 2))])
def test_rhs_parity_weno7_roe_glf(oracle_mod, visc, shape, n, bc):
    w = wl.with_ghost_width(wl.random_smooth_box(*shape, nspecies=n, seed=7100 + n + shape[0], bc=bc), 4)
    orc = oracle_mod.Oracle.from_workload(w, recon=W7, viscosity=visc)
    ro = orc.rhs(w.U.copy(), w.T_guess.copy())
    assert orc.last_status == 0
    g = _gpu(w, reconstruction=W7, viscosity=visc)
    err = field_err(w.interior(g.rhs()), w.interior(ro))
    assert err.max() < RHS_TOL, err
    g.close()


def test_rhs_parity_weno7_shocked_states(oracle_mod):
    w = wl.with_ghost_width(wl.config3_shock_bubble_3d(24), 4)
    orc = oracle_mod.Oracle.from_workload(w, recon=W7)
    ro = orc.rhs(w.U.copy(), w.T_guess.copy())
    g = _gpu(w, reconstruction=W7)
    err = field_err(w.interior(g.rhs()), w.interior(ro))
    assert err.max() < RHS_TOL, err
    g.close()


def test_shock_tube_and_bubble_steps_weno7(oracle_mod):
    for w, steps in ((wl.config1_shock_tube(), 100), (wl.config3_shock_bubble_3d(32), 12)):
        w = wl.with_ghost_width(w, 4)
        orc = oracle_mod.Oracle.from_workload(w, recon=W7)
        Uo, To = w.U.copy(), w.T_guess.copy()
        g = _gpu(w, reconstruction=W7)
        worst = 0.0
        for _ in range(steps):
            So = orc.max_wavespeed(Uo, To)
            Sg = g.max_wavespeed()
            assert abs(Sg - So) <= 1e-12 * So
            dt = w.cfl / So
            assert orc.rk3_step(Uo, To, dt) == 0
            g.step(dt)
            cmax = So * min(w.dx, w.dy, w.dz)
            worst = max(worst, state_err(w, g.host_U(), Uo, cmax).max())
        assert g.ctx.xf_status() == 0
        assert worst < STEPS_TOL, worst
        g.close()


def test_ghost_width_must_match_the_reconstruction():
    from paper_2403_05910_b200 import xf

    w = wl.random_smooth_box(12, 10, 1, nspecies=2, seed=1)
    with pytest.raises(xf.XfError):
        xf.Context.from_workload(w, reconstruction=W7)        # ng = 3 arrays with the eight-cell stencil
    with pytest.raises(xf.XfError):
        xf.Context.from_workload(wl.with_ghost_width(w, 4), reconstruction=0)


def test_config4_shape_weno7_sampled(oracle_mod):
    """config 4's set-up at 128 x 64 x 64 (N = 10, the TMA kernels with several strips and segments) on sampled cells."""
    w = wl.with_ghost_width(wl.config4_shock_bubble_3d_10sp(128, 64, 64), 4)
    orc = oracle_mod.Oracle.from_workload(w, recon=W7)
    U = w.U.copy()
    orc.fill_ghosts(U)
    rng = np.random.default_rng(11)
    nzp, nyp, nxp = w.padded_shape
    i = np.concatenate([rng.integers(0, w.nx, 1500), rng.integers(int(0.14 * w.nx), int(0.4 * w.nx), 2500)])
    j, k = rng.integers(0, w.ny, i.size), rng.integers(0, w.nz, i.size)
    idx = ((k + 4).astype(np.int64) * nyp + (j + 4)) * nxp + (i + 4)
    ro = orc.rhs_cells(U, w.T_guess, idx)
    assert orc.last_status == 0
    g = _gpu(w, reconstruction=W7)
    r = g.rhs().reshape(w.nvars, -1)[:, idx].T
    scale = np.abs(ro).max(axis=0)
    scale[1:4] = scale[1:4].max()
    Ymax = (np.abs(w.interior(w.U)[5:]) / w.interior(w.U)[0]).reshape(w.nvars - 5, -1).max(axis=1)
    scale[5:] = np.maximum(scale[5:], Ymax * scale[0])       # the floor of a partial-density row
    err = np.abs(r - ro).max(axis=0) / scale
    assert err.max() < RHS_TOL, err
    g.close()
