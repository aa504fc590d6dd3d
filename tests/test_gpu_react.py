"""-m gpu parity of the reaction step (Eq. 8-12, 180-198 Eq. 27-28; DESIGN.md readings
R24-R30) on the CUDA path (csrc/xf_react.cu) against the oracle (xo_react), on a seeded synthetic element-balanced
mechanism (workloads.synthetic_mechanism): the species after a reaction step per variable to 1e-11 of the variable's
maximum (the rates pass through exponentials of O(20) arguments: 1e-14 relative each, a few sub-steps of a stiff system on
top), T to 1e-12; everything the step must not touch bit for bit; a Strang-split reacting-flow step sequence to 1e-9.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _reacting_box(shape, seed, bc=(0,) * 6, smooth=False):
    w = wl.reacting_box(*shape, seed=seed, bc=bc, smooth=smooth)
    return w, wl.reacting_table()[1]


@pytest.mark.parametrize("shape,n_sub,n_corr,nreac", [((40, 1, 1), 1, 1, 19), ((17, 13, 1), 4, 1, 19), ((12, 10, 9), 2, 2, 30),
                                                     ((9, 8, 7), 8, 1, 8)])
def test_react_parity(oracle_mod, shape, n_sub, n_corr, nreac):
    import torch

    from gpu_helpers import GpuRun

    w, comp = _reacting_box(shape, seed=70 + shape[0])
    mech = wl.synthetic_mechanism(w.table, comp, nreac, seed=nreac, rate=5.0)
    om = oracle_mod.make_mechanism(mech)
    orc = oracle_mod.Oracle.from_workload(w)
    Uo, To = w.U.copy(), w.T_guess.copy()
    dt = 5e-4
    assert orc.react(om, Uo, To, dt, n_sub, n_corr) == 0
    g = GpuRun(w)
    g.ctx.xf_set_mechanism(mech)
    U0 = g.U.clone()
    g.ctx.xf_react(g.U, g.T, dt, n_sub, n_corr)
    assert g.ctx.xf_status() == 0
    Ug, Tg = g.host_U(), g.host_T()
    assert np.max(np.abs(w.interior(Uo)[5:] - w.interior(w.U)[5:])) > 1e-3        # the step really changes the composition
    den = np.abs(w.interior(Uo)[5:]).reshape(8, -1).max(axis=1)
    err = np.abs(w.interior(Ug)[5:] - w.interior(Uo)[5:]).reshape(8, -1).max(axis=1) / den
    assert err.max() < 1e-11, err
    Ti, Toi = w.interior(Tg[None])[0], w.interior(To[None])[0]
    assert np.max(np.abs(Ti - Toi) / Toi) < 1e-12
    # untouched, bit for bit: rho, momentum, E everywhere; every ghost entry of the species and of T
    assert torch.equal(g.U[:5], U0[:5])
    mask = np.ones(w.padded_shape, dtype=bool)
    mask[tuple(slice(3, -3) if m > 1 else slice(None) for m in (w.nz, w.ny, w.nx))] = False
    assert np.array_equal(Ug[5:][:, mask], w.U[5:][:, mask]) and np.array_equal(Tg[mask], w.T_guess[mask])
    g.close()


def test_react_parity_outside_the_fit_range(oracle_mod):
    """half of the cells hotter than T_hi: the constant-c_p continuation of h_s and S_s in the rates and in the Newton
    iteration (readings R3, R24) -- the corner the oracle pin test_rates_outside_the_fit_range_use_the_continuation holds
    (cold cells below T_lo are left to that pin: the seeded exothermic mechanism leaves the range within one step)"""
    from gpu_helpers import GpuRun

    w, comp = _reacting_box((16, 12, 1), seed=91)
    t = w.table
    Ui = w.interior(w.U)
    rho = Ui[0]
    Y = np.concatenate([Ui[5:] / rho, (1.0 - (Ui[5:] / rho).sum(axis=0))[None]])
    hot = np.broadcast_to(np.arange(16)[None, None, :] < 8, rho.shape)
    Tnew = np.where(hot, 1.2 * t.Thi, w.interior(w.T_guess[None])[0])
    e = t.internal_energy(Y.reshape(9, -1), Tnew.reshape(-1)).reshape(rho.shape)
    k = 0.5 * (Ui[1] ** 2 + Ui[2] ** 2 + Ui[3] ** 2) / rho
    Ui[4] = np.where(hot, rho * e + k, Ui[4])
    w.interior(w.T_guess[None])[0][...] = np.where(hot, Tnew * 1.01, Tnew)
    mech = wl.synthetic_mechanism(w.table, comp, 19, seed=19, rate=5.0)
    om = oracle_mod.make_mechanism(mech)
    orc = oracle_mod.Oracle.from_workload(w)
    Uo, To = w.U.copy(), w.T_guess.copy()
    assert orc.react(om, Uo, To, 2e-4, 2, 1) == 0
    g = GpuRun(w)
    g.ctx.xf_set_mechanism(mech)
    g.ctx.xf_react(g.U, g.T, 2e-4, 2, 1)
    assert g.ctx.xf_status() == 0
    Ug, Tg = g.host_U(), g.host_T()
    Toi = w.interior(To[None])[0]
    assert Toi[..., :8].min() > t.Thi and Toi[..., 8:].max() < t.Thi            # the hot half is still above the range
    den = np.abs(w.interior(Uo)[5:]).reshape(8, -1).max(axis=1)
    err = np.abs(w.interior(Ug)[5:] - w.interior(Uo)[5:]).reshape(8, -1).max(axis=1) / den
    assert err.max() < 1e-11, err
    assert np.max(np.abs(w.interior(Tg[None])[0] - Toi) / Toi) < 1e-12
    g.close()


def test_react_parity_with_absent_species(oracle_mod):
    """one species absent from every cell, another from half of them: p_s = d_s / Y_s is 0 where Y_s <= 0 (reading R25)"""
    from gpu_helpers import GpuRun

    w, comp = _reacting_box((14, 11, 1), seed=93)
    Ui = w.interior(w.U)
    Ui[5 + 7] += Ui[5 + 2]                                       # move species 2's mass to species 7: rho unchanged
    Ui[5 + 2] = 0.0
    half = np.broadcast_to(np.arange(14)[None, None, :] < 7, Ui[0].shape)
    Ui[5 + 7] += np.where(half, Ui[5 + 4], 0.0)
    Ui[5 + 4] = np.where(half, 0.0, Ui[5 + 4])
    mech = wl.synthetic_mechanism(w.table, comp, 19, seed=19, rate=5.0)
    om = oracle_mod.make_mechanism(mech)
    orc = oracle_mod.Oracle.from_workload(w)
    Uo, To = w.U.copy(), w.T_guess.copy()
    assert orc.react(om, Uo, To, 3e-4, 2, 2) == 0
    g = GpuRun(w)
    g.ctx.xf_set_mechanism(mech)
    g.ctx.xf_react(g.U, g.T, 3e-4, 2, 2)
    assert g.ctx.xf_status() == 0
    Ug, Tg = g.host_U(), g.host_T()
    assert np.all(np.isfinite(Ug)) and np.all(np.isfinite(Tg))
    den = np.abs(w.interior(Uo)[5:]).reshape(8, -1).max(axis=1)
    err = np.abs(w.interior(Ug)[5:] - w.interior(Uo)[5:]).reshape(8, -1).max(axis=1) / den
    assert err.max() < 1e-11, err
    Toi = w.interior(To[None])[0]
    assert np.max(np.abs(w.interior(Tg[None])[0] - Toi) / Toi) < 1e-12
    g.close()


def test_strang_split_reacting_flow_steps(oracle_mod):
    """react(dt/2), convective SSP-RK3 step, react(dt/2), five times: the composed path against the
    oracle's composition of the same pieces"""
    from gpu_helpers import GpuRun

    w, comp = _reacting_box((20, 16, 12), seed=5, smooth=True)
    mech = wl.synthetic_mechanism(w.table, comp, 19, seed=3, rate=200.0)
    om = oracle_mod.make_mechanism(mech)
    orc = oracle_mod.Oracle.from_workload(w)
    Uo, To = w.U.copy(), w.T_guess.copy()
    g = GpuRun(w)
    g.ctx.xf_set_mechanism(mech)
    worst = 0.0
    for _ in range(5):
        S = orc.max_wavespeed(Uo, To)
        dt = 0.4 / S
        assert orc.react(om, Uo, To, 0.5 * dt, 2, 1) == 0
        assert orc.rk3_step(Uo, To, dt) == 0
        assert orc.react(om, Uo, To, 0.5 * dt, 2, 1) == 0
        g.ctx.xf_react(g.U, g.T, 0.5 * dt, 2, 1)
        g.step(dt)
        g.ctx.xf_react(g.U, g.T, 0.5 * dt, 2, 1)
        a, b = w.interior(g.host_U()), w.interior(Uo)
        den = np.abs(b).reshape(w.nvars, -1).max(axis=1)
        den[1:4] = np.abs(b[0]).max() * S * w.dx
        worst = max(worst, (np.abs(a - b).reshape(w.nvars, -1).max(axis=1) / den).max())
    assert g.ctx.xf_status() == 0
    assert worst < 1e-9, worst
    g.close()


def test_react_needs_a_mechanism_and_checks_it():
    from gpu_helpers import GpuRun
    from paper_2403_05910_b200 import xf

    w, comp = _reacting_box((8, 1, 1), seed=1)
    g = GpuRun(w)
    with pytest.raises(xf.XfError):
        g.ctx.xf_react(g.U, g.T, 1e-3)
    mech = wl.synthetic_mechanism(w.table, comp, 4, seed=1)
    mech.nu_r[0, 0] = 4                                        # more than three molecules on a side
    with pytest.raises(xf.XfError):
        g.ctx.xf_set_mechanism(mech)
    g.close()
