"""Pins of the oracle's ROE and GLF artificial-viscosity options.  LLF is
pinned in test_oracle_pins.py; the variants differ only in Lambda~ of Eq. 14, so what is pinned here is what Lambda~
is (against values written out in the test), that consistency, conservation, design order and the exact Riemann
solution survive, and that the three options are really different schemes at a shock."""
import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl
from helpers import exact_riemann, single_species_workload

LLF, ROE, GLF = 0, 1, 2


def _oracle(oracle_mod, w, visc):
    return oracle_mod.Oracle.from_workload(w, viscosity=visc)


@pytest.mark.parametrize("visc", [ROE, GLF])
def test_uniform_flow_preserved(oracle_mod, visc):
    rng = np.random.default_rng(77)
    table = wl.synthetic_nasa7_table(rng.uniform(2, 100, 3), Ru=0.1, rng=rng, formation=True)
    Y = rng.dirichlet(np.ones(3))
    T0, rho0 = 700.0, 1.3
    c0 = float(np.sqrt(table.frozen_gamma(Y.reshape(3, 1), np.array([T0])) * table.mixture_R(Y.reshape(3, 1)) * T0)[0])
    vel = 0.6 * c0 * np.array([0.5, -0.7, 0.4])
    U0 = wl.conserved_from_primitive(table, np.array([rho0]), vel[:1], vel[1:2], vel[2:], np.array([T0]),
                                     Y.reshape(3, 1))[:, 0]
    nx, ny, nz = 8, 7, 6
    Ui = np.tile(U0.reshape(-1, 1, 1, 1), (1, nz, ny, nx))
    w = wl._finish("uniform", nx, ny, nz, 0.1, 0.2, 0.3, table, (wl.BC_PERIODIC,) * 6, Ui, np.full((nz, ny, nx), T0), rng)
    o = _oracle(oracle_mod, w, visc)
    U, T = w.U.copy(), w.T_guess.copy()
    rhs = o.rhs(U, T)
    P = o.cell_primitives(U0, T0)
    for d in range(3):
        F = o.phys_flux(U0, P, d)
        assert np.max(np.abs(w.interior(rhs)) / (np.abs(F).reshape(-1, 1, 1, 1) / 0.1 + 1e-300)) <= 1e-12
        if visc == ROE:                                        # face level: six identical cells -> the physical flux
            Fh = o.face_flux(d, np.tile(U0, (6, 1)), [T0] * 6)
            assert np.max(np.abs(Fh - F) / (np.abs(F).max())) <= 1e-13


def test_glf_face_flux_equals_llf_when_global_is_stencil_maximum(oracle_mod):
    """Six different cells; lam_glob set by hand to the stencil maxima of |u-c|, |u|, |u+c| -> the LLF flux, bit for bit."""
    w = wl.random_smooth_box(16, 1, 1, nspecies=3, seed=5)
    o0, o2 = _oracle(oracle_mod, w, LLF), _oracle(oracle_mod, w, GLF)
    Ui = w.interior(w.U)[:, 0, 0, 4:10].T.copy()              # [6, Nv]
    Tg = w.interior(w.T_guess)[0, 0, 4:10].copy()
    prims = [o0.cell_primitives(Ui[m], Tg[m]) for m in range(6)]
    for d in range(3):
        u = np.array([p.vel[d] for p in prims])
        c = np.array([p.c for p in prims])
        for k, lam in enumerate((np.abs(u - c).max(), np.abs(u).max(), np.abs(u + c).max())):
            o2.cfg.lam_glob[d][k] = lam
        assert np.array_equal(o2.face_flux(d, Ui, Tg), o0.face_flux(d, Ui, Tg))


def test_glf_global_maxima_are_over_all_padded_cells(oracle_mod):
    """rhs with GLF == rhs of a hand-fed oracle whose lam_glob comes from numpy over the padded field."""
    w = wl.random_smooth_box(10, 9, 1, nspecies=2, seed=9, bc=(1, 1, 2, 2, 0, 0))
    o = _oracle(oracle_mod, w, GLF)
    U, T = w.U.copy(), w.T_guess.copy()
    # a frame moving at three sound speeds in +x and +y: every cell flows supersonically in the NEGATIVE directions, so
    # u + c < 0 and max |u + c| differs from max (u + c) (the maxima are of absolute values)
    cmax = 1.5 * float(np.sqrt(np.max(U[4] / U[0])))
    for q in (1, 2):
        mom = U[q] - 3.0 * cmax * U[0]
        U[4] += 0.5 * (mom ** 2 - U[q] ** 2) / U[0]
        U[q] = mom
    rhs = o.rhs(U, T)                                         # fills ghosts, converges T
    p, c = np.zeros_like(T), np.zeros_like(T)
    oracle_mod.Oracle.from_workload(w).primitives(U, T.copy(), p, c)
    # brute force: the same numbers from a stencil-level call with lam_glob written by this test
    vel = U[1:4] / U[0]
    lam = [[np.abs(vel[d] - c).max(), np.abs(vel[d]).max(), np.abs(vel[d] + c).max()] for d in range(3)]
    o2 = _oracle(oracle_mod, w, GLF)
    for d in range(3):
        for k in range(3):
            o2.cfg.lam_glob[d][k] = lam[d][k]
    nxp = U.shape[3]
    j, i = 5, 6                                               # an interior cell: x faces i-1/2, i+1/2 and y faces
    acc = np.zeros(w.nvars)
    for d, (dj, di, h) in enumerate(((0, 1, w.dx), (1, 0, w.dy))):
        cells = [(j + dj * (m - 3), i + di * (m - 3)) for m in range(7)]
        Ust = np.array([U[:, 0, jj, ii] for jj, ii in cells])
        Tst = np.array([T[0, jj, ii] for jj, ii in cells])
        acc -= (o2.face_flux(d, Ust[1:7].copy(), Tst[1:7].copy()) - o2.face_flux(d, Ust[0:6].copy(), Tst[0:6].copy())) / h
    assert np.abs(acc - rhs[:, 0, j, i]).max() <= 1e-13 * np.abs(rhs[:, 0, j, i]).max()


def test_roe_lambda_is_the_roe_averaged_wave_speed(oracle_mod):
    """Single species, two constant states L | R on a six-cell stencil with IDEAL weights: the scheme is linear, and
    on a stencil L L L R R R the fifth-order reconstruction of a step has a closed form; against it the ROE option
    must use |u~ -+ c~| with the textbook Roe average."""
    g = 1.4
    rhoL, uL, pL, rhoR, uR, pR = 1.0, 0.3, 1.0, 0.4, -0.2, 0.6
    w = single_species_workload(6, np.array([rhoL] * 3 + [rhoR] * 3).reshape(1, 1, 6),
                                np.array([uL] * 3 + [uR] * 3).reshape(1, 1, 6),
                                np.array([pL] * 3 + [pR] * 3).reshape(1, 1, 6))
    o = oracle_mod.Oracle.from_workload(w, viscosity=ROE, ideal_weights=True)
    Ui = w.interior(w.U)[:, 0, 0, :].T.copy()
    Tg = w.interior(w.T_guess)[0, 0, :].copy()
    Fh = o.face_flux(0, Ui, Tg)

    def flux(r, u, p):
        E = p / (g - 1) + 0.5 * r * u * u
        return np.array([r * u, r * u * u + p, 0.0, 0.0, (E + p) * u])

    def cons(r, u, p):
        return np.array([r, r * u, 0.0, 0.0, p / (g - 1) + 0.5 * r * u * u])

    # textbook Roe average and eigenvectors (1-D Euler; the two shear fields carry nothing here)
    sL, sR = np.sqrt(rhoL), np.sqrt(rhoR)
    ut = (sL * uL + sR * uR) / (sL + sR)
    HL = (pL / (g - 1) + 0.5 * rhoL * uL ** 2 + pL) / rhoL
    HR = (pR / (g - 1) + 0.5 * rhoR * uR ** 2 + pR) / rhoR
    Ht = (sL * HL + sR * HR) / (sL + sR)
    ct = np.sqrt((g - 1) * (Ht - 0.5 * ut * ut))
    R = np.array([[1, 1, 1], [ut - ct, ut, ut + ct], [Ht - ut * ct, 0.5 * ut * ut, Ht + ut * ct]]).T  # rows = r_n
    Rm = R.T                                                   # columns r_n over (rho, rho u, E)
    Lm = np.linalg.inv(Rm)
    lam = np.abs(np.array([ut - ct, ut, ut + ct]))
    # ideal-weights WENO5 of point values (a a a b b) at +1/2: (2a - 13a + 47a + 27b - 3b)/60 and the mirrored one
    sel = [0, 1, 4]
    FL, FR, UL, UR = flux(rhoL, uL, pL)[sel], flux(rhoR, uR, pR)[sel], cons(rhoL, uL, pL)[sel], cons(rhoR, uR, pR)[sel]
    fpL, fpR = 0.5 * (Lm @ FL + lam * (Lm @ UL)), 0.5 * (Lm @ FR + lam * (Lm @ UR))
    fmL, fmR = 0.5 * (Lm @ FL - lam * (Lm @ UL)), 0.5 * (Lm @ FR - lam * (Lm @ UR))
    gp = (36 * fpL + 24 * fpR) / 60                            # stencil (L L L R R): 2-13+47 = 36, 27-3 = 24
    gm = (36 * fmR + 24 * fmL) / 60                            # mirrored stencil (R R R L L)
    expect = Rm @ (gp + gm)
    assert np.abs(Fh[sel] - expect).max() <= 1e-13 * np.abs(expect).max()


@pytest.mark.parametrize("visc", [ROE, GLF])
def test_sod_against_exact_riemann(oracle_mod, visc):
    nx, tend = 400, 0.2
    x = (np.arange(nx) + 0.5) / nx
    rho = np.where(x < 0.5, 1.0, 0.125).reshape(1, 1, nx)
    p = np.where(x < 0.5, 1.0, 0.1).reshape(1, 1, nx)
    w = single_species_workload(nx, rho, np.zeros_like(rho), p, bc=(wl.BC_TRANSMISSIVE,) * 6)
    o = _oracle(oracle_mod, w, visc)
    U, T = w.U.copy(), w.T_guess.copy()
    t = 0.0
    while t < tend - 1e-14:
        dt = min(0.5 / o.max_wavespeed(U, T), tend - t)
        assert o.rk3_step(U, T, dt) == 0
        t += dt
    Ui = w.interior(U)[:, 0, 0, :]
    rho_e, u_e, p_e, pstar, ustar = exact_riemann(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4, (x - 0.5) / 0.2)
    assert np.mean(np.abs(Ui[0] - rho_e)) < 3e-3
    u = Ui[1] / Ui[0]
    pr = 0.4 * (Ui[4] - 0.5 * Ui[0] * u * u)
    plateau = (x > 0.72) & (x < 0.80)
    assert np.max(np.abs(pr[plateau] - pstar)) < 2e-3 and np.max(np.abs(u[plateau] - ustar)) < 2e-3


@pytest.mark.parametrize("visc", [ROE, GLF])
def test_design_order_and_conservation(oracle_mod, visc):
    errs = []
    for nx in (32, 64, 128):
        x = (np.arange(nx) + 0.5) / nx
        rho = (1.0 + 0.2 * np.sin(2 * np.pi * x)).reshape(1, 1, nx)
        w = single_species_workload(nx, rho, np.ones_like(rho), np.ones_like(rho))
        o = _oracle(oracle_mod, w, visc)
        U, T = w.U.copy(), w.T_guess.copy()
        m0 = w.interior(U).sum(axis=(1, 2, 3))
        dx = 1.0 / nx
        nsteps = int(np.ceil(1.0 / (0.4 * dx ** (5.0 / 3.0) * 4.0)))
        for _ in range(nsteps):
            o.rk3_step(U, T, 1.0 / nsteps)
        errs.append(np.mean(np.abs(w.interior(U)[0, 0, 0] - rho[0, 0])))
        m1 = w.interior(U).sum(axis=(1, 2, 3))
        assert np.abs(m1 - m0).max() <= 1e-12 * np.abs(m0).max()
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(orders >= 4.8), (errs, orders)


def test_the_three_options_differ_at_a_shock(oracle_mod):
    w = wl.config1_shock_tube(nx=64)
    r = {}
    for visc in (LLF, ROE, GLF):
        o = _oracle(oracle_mod, w, visc)
        r[visc] = w.interior(o.rhs(w.U.copy(), w.T_guess.copy()))
    s = np.abs(r[LLF]).max()
    assert np.abs(r[ROE] - r[LLF]).max() > 1e-6 * s and np.abs(r[GLF] - r[LLF]).max() > 1e-6 * s
