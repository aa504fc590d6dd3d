"""Pins of the oracle's viscous / diffusive right-hand side (Eq. 1-6,
PAPER.md:155-178 Eq. 22 and 26, Eq. 29; readings R19-R23 in oracle/xf_oracle.h and DESIGN.md).

What is pinned, none of it through the oracle's own code: the mixture rules written out in numpy (Wilke's formula,
Eq. 26) and their limits (one species, identical species, binary); the fits against numpy.polyval; the discretisation
against the CONTINUOUS equations -- div F_v derived symbolically (sympy) from Eq. 2-6 -- exactly on polynomial data in
3-D with all cross terms, and to fourth order on smooth data with temperature-dependent coefficients and binary
diffusion; zero flux in uniform flow; sum_s J_s = 0; telescoping conservation; direction consistency; the decay rate of
a shear wave under xo_rk3_step_ns.
"""
import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

sp = pytest.importorskip("sympy")


def _const_fits(n, mu, kappa, D=1.0):
    z = np.zeros((n, 4))
    m, k = z.copy(), z.copy()
    m[:, 0], k[:, 0] = np.log(mu), np.log(kappa)
    Dm = np.zeros((n, n, 4))
    Dm[:, :, 0] = np.log(D)
    return wl.TransportFits(mu=m, kappa=k, D=Dm, p_ref=1.0)


def _box(oracle_mod, table, nx, ny, nz, h, ng=3):
    dims = [nx, ny, nz]
    return oracle_mod.Oracle(nx, ny, nz, h[0], h[1], h[2], table.W, table.nasa7, table.Ru, table.Tlo, table.Thi, ng=ng)


def _coords(o, n, h):
    """cell-centre coordinates of the whole padded box, origin at the first interior cell centre"""
    nzp, nyp, nxp = o.shape
    g = [o.ng if m > 1 else 0 for m in n]
    x = (np.arange(nxp) - g[0]) * h[0]
    y = (np.arange(nyp) - g[1]) * h[1]
    z = (np.arange(nzp) - g[2]) * h[2]
    return np.meshgrid(z, y, x, indexing="ij")


# ------------------------------------------------------------------------------------------------------------
# mixture rules and fits
# ------------------------------------------------------------------------------------------------------------
def test_fits_are_polynomials_in_ln_T_and_D_scales_with_inverse_pressure(oracle_mod):
    table = wl.synthetic_nasa7_table((28.0, 4.0, 40.0), Ru=0.1, rng=np.random.default_rng(0))
    tr = wl.synthetic_transport(table, 3, p_ref=2.5)           # p_ref != 1: D_st(T, p) = D_st(T, p_ref) p_ref / p (reading R19)
    o = oracle_mod.Oracle(8, 1, 1, 0.1, 1, 1, table.W, table.nasa7, table.Ru, table.Tlo, table.Thi)
    ot = oracle_mod.make_transport(tr)
    for T in (250.0, 700.0, 2500.0):
        for s in range(3):
            Y = np.zeros(3)
            Y[s] = 1.0
            mu, ka, rD, h = o.transport_cell(ot, 1.3, Y, T)
            # a pure species: the mixture value is the species value (Phi_ss = 1)
            assert abs(mu - np.exp(np.polyval(tr.mu[s][::-1], np.log(T)))) <= 1e-14 * mu
            assert abs(ka - np.exp(np.polyval(tr.kappa[s][::-1], np.log(T)))) <= 1e-14 * ka
            assert abs(h[s] - table.Rs[s] * table.h_over_R(np.float64(T))[s]) <= 1e-13 * abs(h[s])
    # binary, written out: D_1m = W_2 D_12 / Wbar (Eq. 26 with one other species), D_12 ~ p_ref / p
    Y = np.array([0.3, 0.7, 0.0])
    T, rho = 900.0, 0.8
    X = Y / table.W / np.sum(Y / table.W)
    Wbar = np.sum(X * table.W)
    p = rho * np.sum(Y * table.Rs) * T
    D = lambda s, t: np.exp(np.polyval(tr.D[s, t][::-1], np.log(T))) * tr.p_ref / p   # noqa: E731
    _, _, rD, _ = o.transport_cell(ot, rho, Y, T)
    e = 1e-12
    for s in range(3):
        num = sum((X[t] + e) * table.W[t] for t in range(3) if t != s)
        den = sum((X[t] + e) / D(s, t) for t in range(3) if t != s)
        assert abs(rD[s] - rho * num / (Wbar * den)) <= 1e-13 * rD[s]
    assert abs(rD[0] - rho * table.W[1] * D(0, 1) / Wbar) <= 1e-9 * rD[0]   # the third species is absent
    _, _, rD2, _ = o.transport_cell(ot, 2 * rho, Y, T)                       # twice the pressure: D halves, rho D stays
    assert np.allclose(rD2, rD, rtol=1e-13)


def test_wilke_written_out(oracle_mod):
    rng = np.random.default_rng(4)
    W = np.array([2.0, 28.0, 44.0, 131.0])
    table = wl.synthetic_nasa7_table(W, Ru=0.1, rng=rng)
    tr = wl.synthetic_transport(table, 9)
    o = oracle_mod.Oracle(8, 1, 1, 0.1, 1, 1, table.W, table.nasa7, table.Ru, table.Tlo, table.Thi)
    ot = oracle_mod.make_transport(tr)
    for _ in range(5):
        Y = rng.dirichlet(np.ones(4))
        T = rng.uniform(250, 2500)
        X = Y / W / np.sum(Y / W)
        for name, fits in (("mu", tr.mu), ("kappa", tr.kappa)):
            a = np.array([np.exp(np.polyval(fits[s][::-1], np.log(T))) for s in range(4)])
            val = 0.0
            for s in range(4):                                  # Eq. 22
                den = 0.0
                for t in range(4):
                    phi = (1 + W[s] / W[t]) ** -0.5 / np.sqrt(8.0) * (1 + (a[s] / a[t]) ** 0.5 * (W[t] / W[s]) ** 0.25) ** 2
                    den += X[t] * phi
                val += X[s] * a[s] / den
            mu, ka, _, _ = o.transport_cell(ot, 1.0, Y, T)
            assert abs((mu if name == "mu" else ka) - val) <= 1e-13 * val
    # identical species: any composition gives the common value
    t1 = wl.calorically_perfect_table((28.0, 28.0, 28.0), (1.4, 1.4, 1.4), Ru=1.0)
    o1 = oracle_mod.Oracle(8, 1, 1, 0.1, 1, 1, t1.W, t1.nasa7, t1.Ru, t1.Tlo, t1.Thi)
    mu, ka, _, _ = o1.transport_cell(oracle_mod.make_transport(_const_fits(3, 0.01, 0.02)), 1.0, np.array([0.2, 0.5, 0.3]), 400.0)
    assert abs(mu - 0.01) <= 1e-15 and abs(ka - 0.02) <= 1e-15


# ------------------------------------------------------------------------------------------------------------
# the discretisation against the continuous equations
# ------------------------------------------------------------------------------------------------------------
def _symbolic_div_fv_single_species(u, v, w, T, mu, kappa, X):
    """div F_v of Eq. 2-4 for one species: rows momentum x, y, z and energy, from sympy expressions"""
    vel = [u, v, w]
    G = [[sp.diff(vel[p], X[q]) for q in range(3)] for p in range(3)]
    div = G[0][0] + G[1][1] + G[2][2]
    tau = [[mu * (G[p][q] + G[q][p]) - (sp.Rational(2, 3) * mu * div if p == q else 0) for q in range(3)] for p in range(3)]
    mom = [sum(sp.diff(tau[p][q], X[q]) for q in range(3)) for p in range(3)]
    en = sum(sp.diff(sum(tau[p][q] * vel[p] for p in range(3)) + kappa * sp.diff(T, X[q]), X[q]) for q in range(3))
    return mom + [en]


def test_exact_on_polynomial_data_in_3d_with_all_cross_terms(oracle_mod):
    """velocities quadratic and T cubic in (x, y, z), constant mu and kappa: every face operator of reading R22 is exact on
    such data and F_v is at most cubic, so the fourth-order divergence is exact -- the residual equals the symbolic div F_v
    to round-off.  A wrong coefficient, a dropped cross term, a transposed gradient or a wrong 2/3 fails this."""
    x, y, z = sp.symbols("x y z")
    rng = np.random.default_rng(12)

    def poly(deg):
        e = 0
        for i in range(deg + 1):
            for j in range(deg + 1 - i):
                for k in range(deg + 1 - i - j):
                    e += sp.Float(rng.uniform(-1, 1)) * x ** i * y ** j * z ** k
        return e

    u, v, w, T = poly(2), poly(2), poly(2), 600 + 50 * poly(3)
    mu0, k0 = 0.013, 0.4
    exact = _symbolic_div_fv_single_species(u, v, w, T, mu0, k0, (x, y, z))
    f_exact = [sp.lambdify((x, y, z), e, "numpy") for e in exact]
    f_in = [sp.lambdify((x, y, z), e, "numpy") for e in (u, v, w, T)]
    table = wl.calorically_perfect_table((1.0,), (1.4,), Ru=1.0)
    n, h = (7, 6, 5), (0.11, 0.13, 0.09)
    o = _box(oracle_mod, table, *n, h)
    Z, Y, Xc = _coords(o, n, h)
    rho = 1.7
    U = np.zeros((5,) + o.shape)
    U[0] = rho
    for q in range(3):
        U[1 + q] = rho * f_in[q](Xc, Y, Z)
    Tf = np.ascontiguousarray(f_in[3](Xc, Y, Z))
    r = o.viscous_rhs(oracle_mod.make_transport(_const_fits(1, mu0, k0)), U, Tf)
    sl = (slice(3, -3),) * 3
    assert np.all(r[0] == 0.0)
    for row, f in zip((1, 2, 3, 4), f_exact):
        ref = f(Xc, Y, Z) * np.ones(o.shape)
        assert np.max(np.abs(r[row][sl] - ref[sl])) <= 2e-11 * max(np.abs(ref[sl]).max(), 1.0), row


def test_fourth_order_with_variable_coefficients_and_binary_diffusion_1d(oracle_mod):
    """1-D periodic, two calorically perfect species with different W, gamma and formation enthalpy, mu, kappa, D_12 power
    laws in T: the continuous div F_v (Eq. 2-6 with reading R21, D_sm from Eq. 26 for a binary mixture) by sympy; the error
    of the oracle falls with fourth order."""
    x = sp.symbols("x")
    W1, W2, g1, g2, Ru = 28.0, 4.0, 1.4, 5.0 / 3.0, 1.0
    a61, a62 = -300.0, 500.0
    table = wl.calorically_perfect_table((W1, W2), (g1, g2), Ru=Ru, a6=(a61, a62))
    tr = _const_fits(2, 1.0, 1.0)
    tr.mu[:, 0], tr.mu[:, 1] = np.log([2e-3, 3e-3]) - 0.7 * np.log(300.0), 0.7
    tr.kappa[:, 0], tr.kappa[:, 1] = np.log([4e-3, 9e-3]) - 0.8 * np.log(300.0), 0.8
    tr.D[:, :, 0], tr.D[:, :, 1] = np.log(5e-3) - 1.7 * np.log(300.0), 1.7
    two_pi = 2 * sp.pi
    rho = 1 + sp.Rational(1, 5) * sp.sin(two_pi * x)
    u = sp.Rational(1, 2) * sp.cos(two_pi * x) + sp.Rational(1, 10)
    vv = sp.Rational(3, 10) * sp.sin(two_pi * x + 1)
    T = 400 + 80 * sp.sin(two_pi * x + sp.Rational(1, 2))
    Y1 = sp.Rational(1, 2) + sp.Rational(3, 10) * sp.cos(two_pi * x + sp.Rational(1, 5))
    Y2 = 1 - Y1
    X1 = (Y1 / W1) / (Y1 / W1 + Y2 / W2)
    X2 = 1 - X1
    Wbar = X1 * W1 + X2 * W2
    pw = lambda c0, ex: c0 * (T / 300) ** ex                  # noqa: E731
    m1, m2, k1, k2 = pw(2e-3, 0.7), pw(3e-3, 0.7), pw(4e-3, 0.8), pw(9e-3, 0.8)

    def wilke(a1, a2):
        phi = lambda Ws, Wt, as_, at: (1 + Ws / Wt) ** sp.Rational(-1, 2) / sp.sqrt(8) * (1 + sp.sqrt(as_ / at) * (Wt / Ws) ** sp.Rational(1, 4)) ** 2  # noqa: E731
        return X1 * a1 / (X1 * phi(W1, W1, a1, a1) + X2 * phi(W1, W2, a1, a2)) + X2 * a2 / (X1 * phi(W2, W1, a2, a1) + X2 * phi(W2, W2, a2, a2))

    mu, ka = wilke(m1, m2), wilke(k1, k2)
    p = rho * Ru * (Y1 / W1 + Y2 / W2) * T
    D12 = pw(5e-3, 1.7) * 1.0 / p
    D1m, D2m = W2 * D12 / Wbar, W1 * D12 / Wbar               # Eq. 26, binary
    dY1, dY2 = sp.diff(Y1, x), sp.diff(Y2, x)
    corr = D1m * dY1 + D2m * dY2
    J1, J2 = -rho * (D1m * dY1 - Y1 * corr), -rho * (D2m * dY2 - Y2 * corr)
    h1 = Ru / W1 * (g1 / (g1 - 1) * T + a61)
    h2 = Ru / W2 * (g2 / (g2 - 1) * T + a62)
    txx = sp.Rational(4, 3) * mu * sp.diff(u, x)
    txy = mu * sp.diff(vv, x)
    exact = [sp.diff(txx, x), sp.diff(txy, x), sp.diff(txx * u + txy * vv + ka * sp.diff(T, x) - (h1 * J1 + h2 * J2), x),
             sp.diff(-J1, x)]
    f_exact = [sp.lambdify(x, e, "numpy") for e in exact]
    f_in = [sp.lambdify(x, e, "numpy") for e in (rho, u, vv, T, Y1)]
    errs = []
    for nx in (32, 64, 128):
        hx = 1.0 / nx
        o = _box(oracle_mod, table, nx, 1, 1, (hx, 1.0, 1.0))
        xc = (np.arange(nx + 6) - 3 + 0.5) * hx
        r_, u_, v_, T_, y_ = (f(xc) for f in f_in)
        U = np.zeros((6, 1, 1, nx + 6))
        U[0, 0, 0], U[1, 0, 0], U[2, 0, 0], U[5, 0, 0] = r_, r_ * u_, r_ * v_, r_ * y_
        r = o.viscous_rhs(oracle_mod.make_transport(tr), U, np.ascontiguousarray(T_.reshape(1, 1, -1)))
        e = [np.max(np.abs(r[row, 0, 0, 3:-3] - f(xc[3:-3]))) / np.max(np.abs(f(xc[3:-3]))) for row, f in zip((1, 2, 4, 5), f_exact)]
        errs.append(e)
    errs = np.array(errs)
    order = np.log2(errs[:-1] / errs[1:])
    assert errs[-1].max() < 2e-6, errs
    assert order.min() > 3.8, order


# ------------------------------------------------------------------------------------------------------------
# structure
# ------------------------------------------------------------------------------------------------------------
def _random_state(oracle_mod, shape, n, seed):
    w = wl.random_smooth_box(*shape, nspecies=n, seed=seed)
    o = oracle_mod.Oracle.from_workload(w)
    U, T = w.U.copy(), w.T_guess.copy()
    o.rhs(U, T)                                               # ghosts filled, T converged on every padded cell
    return w, o, U, T, oracle_mod.make_transport(wl.synthetic_transport(w.table, seed + 1))


def test_uniform_flow_has_no_viscous_flux(oracle_mod):
    w, o, U, T, ot = _random_state(oracle_mod, (9, 8, 7), 3, 21)
    rho = U[0].copy()
    Y = np.array([0.2, 0.5])
    U[1], U[2], U[3] = rho * 0.3, rho * -1.1, rho * 0.7
    U[5], U[6] = rho * Y[0], rho * Y[1]
    T[:] = 777.0
    r = o.viscous_rhs(ot, U, T)                               # rho varies, u, T, Y do not: every gradient vanishes
    assert np.max(np.abs(r)) <= 1e-12 * np.abs(U[4]).max()


def test_diffusion_fluxes_sum_to_zero_and_energy_carries_their_enthalpy(oracle_mod):
    w, o, U, T, ot = _random_state(oracle_mod, (10, 9, 8), 4, 33)
    nzp, nyp, nxp = w.padded_shape
    rng = np.random.default_rng(2)
    for d in range(3):
        for _ in range(5):
            k, j, i = (int(rng.integers(3, m - 4)) for m in (nzp, nyp, nxp))
            F, J = o.viscous_face_flux(ot, U, T, (k * nyp + j) * nxp + i, d)
            assert abs(J.sum()) <= 1e-13 * np.abs(J).max()    # reading R21
            assert F[0] == 0.0 and np.allclose(F[5:], -J[:-1], rtol=0, atol=1e-16 * np.abs(J).max())


def test_conservation_on_a_periodic_box(oracle_mod):
    w, o, U, T, ot = _random_state(oracle_mod, (12, 10, 9), 3, 5)
    r = w.interior(o.viscous_rhs(ot, U, T))
    scale = np.abs(r).reshape(w.nvars, -1).max(axis=1) * r[0].size
    assert np.all(np.abs(r.sum(axis=(1, 2, 3))) <= 1e-13 * np.maximum(scale, 1e-300))


def test_a_profile_along_y_or_z_gives_the_x_result(oracle_mod):
    rng = np.random.default_rng(8)
    table = wl.synthetic_nasa7_table((28.0, 4.0), Ru=0.1, rng=rng, formation=True)
    tr = oracle_mod.make_transport(wl.synthetic_transport(table, 2))
    nx = 24
    xs = (np.arange(nx + 6) - 3 + 0.5) / nx
    rho = 1 + 0.2 * np.sin(2 * np.pi * xs)
    vel = [0.4 * np.cos(2 * np.pi * xs), 0.3 * np.sin(4 * np.pi * xs), 0.2 * np.cos(2 * np.pi * xs + 1)]
    Tp = 500 + 90 * np.sin(2 * np.pi * xs + 0.3)
    Y1 = 0.5 + 0.3 * np.cos(2 * np.pi * xs)
    res = []
    for axis in range(3):
        dims, h = [1, 1, 1], [1.0, 1.0, 1.0]
        dims[axis], h[axis] = nx, 1.0 / nx
        o = _box(oracle_mod, table, *dims, h)
        shp = [1, 1, 1]
        shp[2 - axis] = nx + 6
        U = np.zeros((6,) + tuple(shp))
        U[0] = rho.reshape(shp)
        # the profile's normal velocity along `axis`, the two tangential ones on the other axes in cyclic order
        comp = {0: (0, 1, 2), 1: (2, 0, 1), 2: (1, 2, 0)}[axis]
        for q in range(3):
            U[1 + q] = (rho * vel[comp[q]]).reshape(shp)
        U[5] = (rho * Y1).reshape(shp)
        r = o.viscous_rhs(tr, U, np.ascontiguousarray(Tp.reshape(shp)))
        r = r.reshape(6, -1)[:, 3:-3]
        inv = np.argsort(comp)
        res.append(np.stack([r[0], *(r[1 + inv[q]] for q in range(3)), r[4], r[5]]))
    for axis in (1, 2):
        assert np.max(np.abs(res[axis] - res[0])) <= 1e-13 * np.abs(res[0]).max()


def test_shear_wave_decays_at_the_viscous_rate_under_rk3(oracle_mod):
    """v(x) = eps sin(2 pi x) in a gas at rest decays as exp(-nu (2 pi)^2 t): the sign of the viscous term, its coupling
    into xo_rhs_ns / xo_rk3_step_ns and the time integration."""
    table = wl.calorically_perfect_table((1.0,), (1.4,), Ru=1.0)
    nx, mu0 = 32, 5e-3
    o = oracle_mod.Oracle(nx, 1, 1, 1.0 / nx, 1, 1, table.W, table.nasa7, table.Ru, table.Tlo, table.Thi)
    tr = oracle_mod.make_transport(_const_fits(1, mu0, 1e-9))
    x = (np.arange(nx) + 0.5) / nx
    eps = 1e-6
    U = np.zeros((5, 1, 1, nx + 6))
    U[0] = 1.0
    U[2, 0, 0, 3:-3] = eps * np.sin(2 * np.pi * x)
    U[4] = 1.0 / 0.4
    U[4, 0, 0, 3:-3] += 0.5 * U[2, 0, 0, 3:-3] ** 2
    T = np.ones((1, 1, nx + 6))
    t, dt = 0.0, 0.4 / nx / np.sqrt(1.4)
    for _ in range(60):
        assert o.rk3_step_ns(tr, U, T, dt) == 0
        t += dt
    amp = 2 * np.abs(np.sum(U[2, 0, 0, 3:-3] * np.exp(-2j * np.pi * x))) / nx
    assert abs(amp / eps - np.exp(-mu0 * (2 * np.pi) ** 2 * t)) < 2e-5
    # and without the transport table the step is the convective one
    U2, T2 = U.copy(), T.copy()
    U3, T3 = U.copy(), T.copy()
    o.rk3_step(U2, T2, dt)
    import ctypes as C
    oracle_mod.lib().xo_rk3_step_ns(C.byref(o.cfg), None, U3.ctypes.data_as(C.POINTER(C.c_double)),
                                    T3.ctypes.data_as(C.POINTER(C.c_double)), dt)
    assert np.array_equal(U2, U3)
