"""Pins of the oracle's positivity-preserving flux blending (Eq. 17-20; the
limiting factor theta is deferred by the paper to its ref 41 -> DESIGN.md reading R17).

What is pinned: Eq. 19 (the Lax-Friedrichs flux) and Eq. 20 (the blend) written out in numpy for one face with a
deliberately wild "high-order" flux; the guarantee that follows from the convex splitting of Eq. 18 (every guarded
quantity of both adjacent half-states ends at or above its floor, the binding one exactly on it); theta = 1 -- a bit-identical
residual -- wherever nothing is violated; non-negative density and mass fractions after whole steps on rough data
where the unlimited scheme undershoots by several per cent; unchanged conservation.
"""
import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

RU = 8.0
W3 = np.array([28.0, 4.0, 40.0])
GAM3 = np.array([1.4, 5.0 / 3.0, 1.3])
A63 = np.array([-350.0, 900.0, 120.0])


def _oracle3(oracle_mod, **kw):
    a = np.zeros((3, 7))
    a[:, 0] = GAM3 / (GAM3 - 1.0)
    a[:, 5] = A63
    return oracle_mod.Oracle(8, 1, 1, 0.125, 1.0, 1.0, W3, a, RU, 0.0, 1e300, **kw)


def _cell(rho, vel, T, Y):
    """conserved vector, pressure and frozen sound speed of a calorically perfect mixture, written out"""
    Rs = RU / W3
    a1 = GAM3 / (GAM3 - 1.0)
    Rbar = float(np.sum(Y * Rs))
    e = float(np.sum(Y * Rs * ((a1 - 1.0) * T + A63)))
    cv = float(np.sum(Y * Rs * (a1 - 1.0)))
    p = rho * Rbar * T
    U = np.array([rho, *(rho * np.asarray(vel)), rho * (e + 0.5 * float(np.dot(vel, vel))), rho * Y[0], rho * Y[1]])
    return U, p, float(np.sqrt((1.0 + Rbar / cv) * p / rho))


def _phys_flux(U, p, d):
    ud = U[1 + d] / U[0]
    F = U * ud
    F[1 + d] += p
    F[4] += p * ud
    return F


def _q(V):
    """the guarded quantities as linear functionals of a conserved (or flux) vector: rho, rho Y_1, rho Y_2, rho Y_3"""
    return np.array([V[0], V[5], V[6], V[0] - V[5] - V[6]])


@pytest.mark.parametrize("d", [0, 1, 2])
def test_one_face_blend_written_out(oracle_mod, d):
    o = _oracle3(oracle_mod)
    rng = np.random.default_rng(41 + d)
    hit = 0
    for trial in range(40):
        Ya, Yb = rng.dirichlet(0.4 * np.ones(3)), rng.dirichlet(0.4 * np.ones(3))
        if trial % 3 == 0:
            Ya[1] = 0.0                                        # a species absent from one cell
            Ya /= Ya.sum()
        Ua, pa, ca = _cell(rng.uniform(0.2, 3), rng.normal(size=3) * 40, rng.uniform(200, 2000), Ya)
        Ub, pb, cb = _cell(rng.uniform(0.2, 3), rng.normal(size=3) * 40, rng.uniform(200, 2000), Yb)
        Pa, Pb = o.cell_primitives(Ua, 500.0), o.cell_primitives(Ub, 500.0)
        Fa, Fb = _phys_flux(Ua, pa, d), _phys_flux(Ub, pb, d)
        Lam = max(abs(Ua[1 + d] / Ua[0]) + ca, abs(Ub[1 + d] / Ub[0]) + cb)
        FLF = 0.5 * (Fa + Fb + Lam * (Ua - Ub))                # Eq. 19
        kappa = rng.uniform(0.3, 1.0) / Lam                    # kappa Lambda~ <= 1: the LF half-states are non-negative
        # a "high-order" flux that overdraws one side or the other
        Fhat = FLF + rng.normal(size=7) * np.abs(FLF).max() * rng.choice([0.0, 0.05, 1.0, 5.0])
        theta, Fstar = o.positivity_blend(d, Ua, Pa, Ub, Pb, kappa, Fhat)
        qpL, qmL = _q(Ua) - kappa * _q(FLF), _q(Ub) + kappa * _q(FLF)
        assert qpL.min() >= -1e-13 and qmL.min() >= -1e-13     # LF is positivity preserving
        qp, qm = _q(Ua) - kappa * _q(Fhat), _q(Ub) + kappa * _q(Fhat)
        th = 1.0
        for k in range(4):                                     # reading R17, written out
            for qh, ql in ((qp[k], qpL[k]), (qm[k], qmL[k])):
                eps = min(1e-13, ql)
                if qh < eps:
                    th = min(th, (ql - eps) / (ql - qh))
        assert abs(theta - th) <= 1e-12 and 0.0 <= theta <= 1.0
        assert np.allclose(Fstar, (1 - th) * FLF + th * Fhat if th < 1 else Fhat, rtol=1e-12, atol=1e-12 * np.abs(FLF).max())
        # the guarantee: both blended half-states at or above their floors, the binding one on it
        sp, sm = _q(Ua) - kappa * _q(Fstar), _q(Ub) + kappa * _q(Fstar)
        floors_p, floors_m = np.minimum(1e-13, qpL), np.minimum(1e-13, qmL)
        tol = 1e-12 * max(np.abs(_q(Ua)).max(), np.abs(_q(Ub)).max())
        assert np.all(sp >= floors_p - tol) and np.all(sm >= floors_m - tol)
        if th < 1.0:
            hit += 1
            assert min((sp - floors_p).min(), (sm - floors_m).min()) <= tol
    assert hit >= 10                                           # the limiter really was exercised


def _rough(nx, ny, nz, n=4, seed=3):
    return wl.rough_box(nx, ny, nz, nspecies=n, seed=seed)


@pytest.mark.parametrize("dims", [(40, 1, 1), (14, 12, 1), (12, 10, 8)])
def test_density_and_mass_fractions_stay_non_negative_on_rough_data(oracle_mod, dims):
    w = _rough(*dims)
    D = sum(m > 1 for m in dims)
    worst = {}
    for pp in (False, True):
        o = oracle_mod.Oracle.from_workload(w, positivity=pp)
        U, T = w.U.copy(), w.T_guess.copy()
        m0 = w.interior(U).sum(axis=(1, 2, 3))
        lo = 1.0
        for _ in range(5):
            S = o.max_wavespeed(U, T)
            # D dt Lambda~/dx_d <= 1/2 in every direction (the condition of reading R17) follows from dt = 0.5/(D S)
            assert o.rk3_step(U, T, 0.5 / (D * S)) == 0
            Ui = w.interior(U)
            Y = Ui[5:] / Ui[0]
            lo = min(lo, Y.min(), (1 - Y.sum(axis=0)).min(), Ui[0].min())
        worst[pp] = lo
        m1 = w.interior(U).sum(axis=(1, 2, 3))
        assert np.max(np.abs(m1 - m0)) <= 1e-13 * np.abs(m0).max()   # a blend of two conservative fluxes telescopes
    assert worst[False] < -1e-2                                # the test bites: the plain scheme undershoots
    assert worst[True] >= 0.0


def test_config1_mass_fraction_undershoot_is_removed(oracle_mod):
    """BASELINE.json configs[0] at CFL 0.5: the oracle without the limiter carries Y = -4e-4 (reading R12); with it Y >= 0
    at every step, and the shock-tube solution stays the same in L1."""
    w = wl.config1_shock_tube()
    res = {}
    for pp in (False, True):
        o = oracle_mod.Oracle.from_workload(w, positivity=pp)
        U, T = w.U.copy(), w.T_guess.copy()
        lo = 1.0
        for _ in range(200):
            S = o.max_wavespeed(U, T)
            assert o.rk3_step(U, T, 0.5 / S) == 0
            Ui = w.interior(U)[:, 0, 0, :]
            lo = min(lo, (Ui[5] / Ui[0]).min(), (1 - Ui[5] / Ui[0]).min())
        res[pp] = (lo, Ui.copy())
    assert res[False][0] < -1e-4 and res[True][0] >= 0.0
    # L1: the limiter acts at the contact, and where one species is absent altogether (floor eps = q^LF, reading R17) it
    # falls back to the LF flux, which damps the seeded 1e-3 density noise of this configuration there
    assert np.mean(np.abs(res[True][1][0] - res[False][1][0])) < 3e-3


@pytest.mark.parametrize("recon,visc", [(0, 0), (1, 1), (2, 2)])
def test_theta_is_one_on_smooth_data_bit_identical_residual(oracle_mod, recon, visc):
    w = wl.random_smooth_box(12, 9, 7, nspecies=3, seed=31, bc=(1, 1, 2, 2, 0, 0))
    if recon == 2:
        w = wl.with_ghost_width(w, 4)
    r = {}
    S = oracle_mod.Oracle.from_workload(w).max_wavespeed(w.U.copy(), w.T_guess.copy())
    for pp in (False, True):
        o = oracle_mod.Oracle.from_workload(w, recon=recon, viscosity=visc, positivity=pp, pp_dt=0.5 / (3 * S))
        U, T = w.U.copy(), w.T_guess.copy()
        r[pp] = o.rhs(U, T)
        assert o.last_status == 0
        if pp:
            nzp, nyp, nxp = w.padded_shape
            g = w.ng
            idx = ((np.arange(g, g + 3)[:, None] * nyp + g + 2) * nxp + np.arange(g, g + 4)[None, :]).ravel()
            rc = o.rhs_cells(U, w.T_guess, idx)                # the sampled-cell checker carries the limiter too
            rf = r[pp].reshape(w.nvars, -1)[:, idx].T
            assert np.max(np.abs(rc - rf)) <= 5e-15 * np.abs(rf).max()
    assert np.array_equal(r[True], r[False])


def test_rhs_cells_with_limiter_active_equals_rhs(oracle_mod):
    w = _rough(12, 10, 8)
    o = oracle_mod.Oracle.from_workload(w, positivity=True)
    U, T = w.U.copy(), w.T_guess.copy()
    S = o.max_wavespeed(U, T.copy())
    o.cfg.pp_dt = 0.5 / (3 * S)
    r = o.rhs(U, T)
    o2 = oracle_mod.Oracle.from_workload(w, positivity=False)
    assert np.max(np.abs(r - o2.rhs(w.U.copy(), w.T_guess.copy()))) > 1e-3 * np.abs(r).max()   # the limiter is active
    nzp, nyp, nxp = w.padded_shape
    kk, jj, ii = np.meshgrid(np.arange(3, 3 + w.nz), np.arange(3, 3 + w.ny), np.arange(3, 3 + w.nx), indexing="ij")
    idx = ((kk * nyp + jj) * nxp + ii).ravel()
    rc = o.rhs_cells(U, w.T_guess, idx)
    rf = r.reshape(w.nvars, -1)[:, idx].T
    assert np.max(np.abs(rc - rf) / np.abs(rf).max(axis=0)) <= 1e-14
