"""Pins of the oracle's reaction step (Eq. 8-12, Eq. 27-28; readings
R24-R30 in oracle/xf_oracle.h and DESIGN.md).

What is pinned, none of it through the oracle's own code: the QSS parameter alpha against the property that DEFINES it (the
update is exact for constant q and p) and against its closed form in extended precision; the rates of Eq. 9-12 written out
in numpy for a hand-built reversible reaction and a third-body one, detailed balance at the equilibrium composition, mass
balance of a random mechanism; the integrator against scipy's stiff solver on an independent numpy restatement of the
right-hand side (second order in the sub-step); conservation of rho, rho u, E and of the internal energy through T.
"""
import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

scipy_integrate = pytest.importorskip("scipy.integrate")


def _setup(oracle_mod, n_reactions=19, seed=1, rate=50.0):
    table, comp = wl.reacting_table()
    mech = wl.synthetic_mechanism(table, comp, n_reactions, seed=seed, rate=rate)
    o = oracle_mod.Oracle(4, 1, 1, 1.0, 1, 1, table.W, table.nasa7, table.Ru, table.Tlo, table.Thi)
    return table, mech, o, oracle_mod.make_mechanism(mech)


def _cell(table, rho, vel, T, Y):
    e = float(table.internal_energy(Y.reshape(-1, 1), np.array([T]))[0])
    U = np.zeros(table.n + 4)
    U[0], U[1:4], U[4], U[5:] = rho, rho * np.asarray(vel), rho * (e + 0.5 * float(np.dot(vel, vel))), rho * Y[:-1]
    return U, e


# ------------------------------------------------------------------------------------------------------------
# alpha (reading R26)
# ------------------------------------------------------------------------------------------------------------
def test_alpha_closed_form_series_and_limits(oracle_mod):
    L = oracle_mod.lib()
    for r in (1e-12, 1e-6, 3e-3, 0.0099, 0.0101, 0.0999, 0.1001, 0.3, 1.0, 7.0, 40.0, 800.0):
        x = np.longdouble(r)
        em = -np.expm1(-x)
        ref = float((1 - em / x) / em) if r > 1e-4 else float(0.5 + x / 12)
        assert abs(L.xo_qss_alpha(r) - ref) <= 3e-14, r
    assert L.xo_qss_alpha(0.0) == 0.5 and abs(L.xo_qss_alpha(1e4) - 1.0) < 1.1e-4


def test_one_step_is_exact_for_constant_q_and_p(oracle_mod):
    """dY/dt = q - p Y with constant q, p: Y(dt) = Y0 e^{-p dt} + (q/p)(1 - e^{-p dt}).  The predictor with alpha(p dt)
    reproduces it for ANY dt -- the property that defines alpha; the corrector (same q, p) leaves it there."""
    L = oracle_mod.lib()
    rng = np.random.default_rng(3)
    for _ in range(50):
        q, p, Y0 = rng.uniform(0, 5), 10 ** rng.uniform(-3, 3), rng.uniform(0, 1)
        dt = 10 ** rng.uniform(-3, 1)
        a = L.xo_qss_alpha(p * dt)
        Y1 = Y0 + dt * (q - p * Y0) / (1 + a * p * dt)
        exact = Y0 * np.exp(-p * dt) + q / p * -np.expm1(-p * dt)
        assert abs(Y1 - exact) <= 1e-12 * max(exact, Y0)


# ------------------------------------------------------------------------------------------------------------
# rates (readings R24, R25)
# ------------------------------------------------------------------------------------------------------------
def _rates_numpy(table, mech, rho, Y, T):
    """independent restatement of Eq. 9-12 (vectorised numpy; T inside the fit range)"""
    a, W, Ru = table.nasa7, table.W, table.Ru
    conc = rho * Y / W
    SR = a[:, 0] * np.log(T) + a[:, 1] * T + a[:, 2] * T ** 2 / 2 + a[:, 3] * T ** 3 / 3 + a[:, 4] * T ** 4 / 4 + a[:, 6]
    HRT = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
    nu = mech.nu_p - mech.nu_r
    kf = mech.A * T ** mech.B * np.exp(-mech.E / (Ru * T))
    Kc = (mech.p_atm / (Ru * T)) ** nu.sum(axis=1) * np.exp(nu @ (SR - HRT))
    tb = np.where(mech.third == 1, mech.eff @ conc, 1.0)
    Rf = tb * kf * np.prod(conc[None, :] ** mech.nu_r, axis=1)
    Rb = tb * kf / Kc * np.prod(conc[None, :] ** mech.nu_p, axis=1)
    q = W / rho * (mech.nu_p.T @ Rf + mech.nu_r.T @ Rb)
    d = W / rho * (mech.nu_r.T @ Rf + mech.nu_p.T @ Rb)
    return q, d, Rf, Rb


def test_rates_written_out(oracle_mod):
    table, mech, o, om = _setup(oracle_mod)
    rng = np.random.default_rng(5)
    for _ in range(6):
        Y = rng.dirichlet(np.ones(9))
        rho, T = rng.uniform(0.3, 3), rng.uniform(400, 2800)
        q, d = o.reaction_rates(om, rho, Y, T)
        qn, dn, _, _ = _rates_numpy(table, mech, rho, Y, T)
        assert np.allclose(q, qn, rtol=1e-12, atol=1e-13 * np.abs(qn).max())
        assert np.allclose(d, dn, rtol=1e-12, atol=1e-13 * np.abs(dn).max())
        assert abs((q - d).sum()) <= 1e-12 * np.abs(d).max()     # element-balanced reactions conserve mass: sum W nu = 0
        assert q[8] == 0.0 and d[8] == 0.0                          # the inert species


def test_single_reaction_by_hand_and_detailed_balance(oracle_mod):
    """species 0 + species 1 <=> species 5 + species 5 (compositions (2,0) + (0,2) = 2 x (1,1)): rates by hand; at the
    composition with [X5]^2/([X0][X1]) = K_c the net rate vanishes."""
    table, comp = wl.reacting_table()
    n = table.n
    nu_r, nu_p = np.zeros((1, n), dtype=np.int64), np.zeros((1, n), dtype=np.int64)
    nu_r[0, 0] = nu_r[0, 1] = 1
    nu_p[0, 5] = 2
    mech = wl.Mechanism(nu_r=nu_r, nu_p=nu_p, A=np.array([3.0e3]), B=np.array([0.5]), E=np.array([table.Ru * 900.0]),
                        third=np.zeros(1, dtype=np.int64), eff=np.ones((1, n)), p_atm=400.0)
    o = oracle_mod.Oracle(4, 1, 1, 1.0, 1, 1, table.W, table.nasa7, table.Ru, table.Tlo, table.Thi)
    om = oracle_mod.make_mechanism(mech)
    T, rho = 1500.0, 0.7
    a, W, Ru = table.nasa7, table.W, table.Ru
    g = lambda s: (a[s, 0] * np.log(T) + a[s, 1] * T + a[s, 2] * T ** 2 / 2 + a[s, 3] * T ** 3 / 3 + a[s, 4] * T ** 4 / 4 + a[s, 6]) - \
        (a[s, 0] + a[s, 1] * T / 2 + a[s, 2] * T ** 2 / 3 + a[s, 3] * T ** 3 / 4 + a[s, 4] * T ** 4 / 5 + a[s, 5] / T)   # noqa: E731
    Kc = np.exp(2 * g(5) - g(0) - g(1))                          # sum nu = 0: no pressure factor
    kf = 3.0e3 * T ** 0.5 * np.exp(-900.0 / T)
    Y = np.zeros(n)
    Y[0], Y[1], Y[5], Y[8] = 0.1, 0.3, 0.2, 0.4
    c = rho * Y / W
    Rf, Rb = kf * c[0] * c[1], kf / Kc * c[5] ** 2
    q, d = o.reaction_rates(om, rho, Y, T)
    assert abs(q[5] - W[5] / rho * 2 * Rf) <= 1e-13 * q[5] and abs(d[5] - W[5] / rho * 2 * Rb) <= 1e-13 * d[5]
    assert abs(q[0] - W[0] / rho * Rb) <= 1e-13 * q[0] and abs(d[1] - W[1] / rho * Rf) <= 1e-13 * d[1]
    # equilibrium: choose [X5] from K_c
    c5 = np.sqrt(Kc * c[0] * c[1])
    Y[5] = c5 * W[5] / rho
    Y[8] = 1 - Y[0] - Y[1] - Y[5]
    q, d = o.reaction_rates(om, rho, Y, T)
    assert np.max(np.abs(q - d)) <= 1e-12 * np.max(d)
    # third body: the same reaction with M multiplies both rates by sum eff_s [X_s]
    mech.third[0] = 1
    mech.eff[0] = np.linspace(0.5, 2.5, n)
    q3, d3 = o.reaction_rates(oracle_mod.make_mechanism(mech), rho, Y, T)
    tb = float(mech.eff[0] @ (rho * Y / W))
    assert np.allclose(q3, tb * q, rtol=1e-13) and np.allclose(d3, tb * d, rtol=1e-13)


# ------------------------------------------------------------------------------------------------------------
# the integrator (readings R26-R30)
# ------------------------------------------------------------------------------------------------------------
def test_rates_outside_the_fit_range_use_the_continuation(oracle_mod):
    """T above T_hi / below T_lo (readings R3, R24): c_p frozen at the range end, h continued linearly and S with
    c_p ln(T / T_c) -- written out here; the in-range pins never reach those terms (a mutation of the entropy
    continuation survived them)."""
    table, mech, o, om = _setup(oracle_mod)
    a, W, Ru = table.nasa7, table.W, table.Ru
    rng = np.random.default_rng(6)
    for T in (table.Thi * 1.25, table.Tlo * 0.8):
        Tc = min(max(T, table.Tlo), table.Thi)
        Y = rng.dirichlet(np.ones(9))
        rho = 0.7
        cpR = a[:, 0] + a[:, 1] * Tc + a[:, 2] * Tc ** 2 + a[:, 3] * Tc ** 3 + a[:, 4] * Tc ** 4
        hR = (a[:, 0] * Tc + a[:, 1] * Tc ** 2 / 2 + a[:, 2] * Tc ** 3 / 3 + a[:, 3] * Tc ** 4 / 4 + a[:, 4] * Tc ** 5 / 5
              + a[:, 5]) + cpR * (T - Tc)                         # h_s / R_s [K]
        SR = (a[:, 0] * np.log(Tc) + a[:, 1] * Tc + a[:, 2] * Tc ** 2 / 2 + a[:, 3] * Tc ** 3 / 3 + a[:, 4] * Tc ** 4 / 4
              + a[:, 6]) + cpR * np.log(T / Tc)
        conc = rho * Y / W
        nu = mech.nu_p - mech.nu_r
        kf = mech.A * T ** mech.B * np.exp(-mech.E / (Ru * T))
        Kc = (mech.p_atm / (Ru * T)) ** nu.sum(axis=1) * np.exp(nu @ (SR - hR / T))
        tb = np.where(mech.third == 1, mech.eff @ conc, 1.0)
        Rf = tb * kf * np.prod(conc[None, :] ** mech.nu_r, axis=1)
        Rb = tb * kf / Kc * np.prod(conc[None, :] ** mech.nu_p, axis=1)
        qn = W / rho * (mech.nu_p.T @ Rf + mech.nu_r.T @ Rb)
        dn = W / rho * (mech.nu_r.T @ Rf + mech.nu_p.T @ Rb)
        q, d = o.reaction_rates(om, rho, Y, T)
        assert np.allclose(q, qn, rtol=1e-11, atol=1e-13 * np.abs(qn).max())
        assert np.allclose(d, dn, rtol=1e-11, atol=1e-13 * np.abs(dn).max())
        assert np.abs(cpR * np.log(T / Tc)).max() > 0.5            # the continuation term is not small here


def _reference_solution(table, mech, rho, e, Y0, t_end):
    """scipy's implicit solver on the numpy restatement of dY/dt = q - d with T from e(T, Y) by bisection-free Newton"""
    def T_of(Y, Tg):
        T = Tg
        for _ in range(60):
            cv = float((Y * table.Rs * (table.cp_over_R(np.float64(T)) - 1.0)).sum())
            T = T + (e - float(table.internal_energy(Y.reshape(-1, 1), np.array([T]))[0])) / cv
        return T

    state = {"T": 1200.0}

    def rhs(t, y):
        Y = np.append(y, 1.0 - y.sum())
        state["T"] = T_of(Y, state["T"])
        q, d, _, _ = _rates_numpy(table, mech, rho, Y, state["T"])
        return (q - d)[:-1]

    sol = scipy_integrate.solve_ivp(rhs, (0.0, t_end), Y0[:-1], method="Radau", rtol=1e-11, atol=1e-14)
    assert sol.success
    return np.append(sol.y[:, -1], 1.0 - sol.y[:, -1].sum())


def test_second_order_against_a_stiff_reference_and_what_stays_fixed(oracle_mod):
    table, mech, o, om = _setup(oracle_mod, rate=20.0)
    Y0 = np.array([0.1, 0.4, 0.05, 0.01, 0.01, 0.01, 0.01, 0.01, 0.4])
    rho, vel, T0, t_end = 0.9, (3.0, -1.0, 0.5), 1200.0, 4e-3
    U, e = _cell(table, rho, vel, T0, Y0)
    ref = _reference_solution(table, mech, rho, e, Y0, t_end)
    assert np.max(np.abs(ref - Y0)) > 0.02                       # the composition really moves
    errs = []
    for n_sub in (8, 16, 32, 64):
        st, U1, T1 = o.react_cell(om, U, 1000.0, t_end, n_sub, 1)
        assert st == 0
        Y1 = np.append(U1[5:], rho - U1[5:].sum()) / rho
        errs.append(np.max(np.abs(Y1 - ref)))
        assert np.array_equal(U1[:5], U[:5])                     # rho, rho u, E untouched (reading R29)
        assert abs(float(table.internal_energy(Y1.reshape(-1, 1), np.array([T1]))[0]) - e) <= 1e-11 * abs(e)
    order = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert errs[-1] < 2e-5 and order.min() > 1.7, (errs, order)
    # more corrector iterations do not change the order but reduce the error constant or leave it
    st, U2, _ = o.react_cell(om, U, 1000.0, t_end, 16, 3)
    assert np.max(np.abs(np.append(U2[5:], rho - U2[5:].sum()) / rho - ref)) < 2 * errs[1]


def _alpha_ld(r):
    """alpha of reading R26 from its closed form in extended precision (series below 1e-4), not the oracle's function"""
    x = np.longdouble(r)
    if r < 1e-4:
        return float(0.5 + x / 12)
    em = -np.expm1(-x)
    return float((1 - em / x) / em)


@pytest.mark.parametrize("absent", [False, True])
@pytest.mark.parametrize("n_corr", [1, 2])
def test_predictor_corrector_step_written_out(oracle_mod, n_corr, absent):
    """One sub-step of Eq. 27-28 written out in numpy from independent pieces -- the numpy rates of this file, alpha from its
    closed form in extended precision, T from e(T, Y) by a Newton iteration on workloads' forward table evaluation -- and
    compared with xo_react_cell.  A second-order test cannot see a slip in the PREDICTOR's alpha (any alpha leaves the
    predictor first order and the corrector second order): a mutation of its argument survived every other pin."""
    table, mech, o, om = _setup(oracle_mod, rate=60.0)
    Y0 = np.array([0.12, 0.35, 0.06, 0.02, 0.015, 0.01, 0.02, 0.005, 0.4])
    if absent:                                                  # a species that is not there: p_s = 0 where Y_s <= 0 (reading R25)
        Y0[8] += Y0[3]
        Y0[3] = 0.0
    rho, vel, Tstart, h = 1.3, (2.0, 0.5, -1.0), 1500.0, 2.5e-3
    U, e = _cell(table, rho, vel, Tstart, Y0)

    def T_of(Y, Tg):
        T = Tg
        for _ in range(60):
            cv = float((Y * table.Rs * (table.cp_over_R(np.float64(T)) - 1.0)).sum())
            T = T + (e - float(table.internal_energy(Y.reshape(-1, 1), np.array([T]))[0])) / cv
        return T

    T0 = T_of(Y0, 1400.0)
    q0, d0, _, _ = _rates_numpy(table, mech, rho, Y0, T0)
    with np.errstate(divide="ignore", invalid="ignore"):
        p0 = np.where(Y0 > 0.0, d0 / Y0, 0.0)
    assert (p0[:-1] * h).max() > 0.5 and (p0[:-1] * h).min() < 0.05     # alpha far from 1/2 for some species, near it for others
    a0 = np.array([_alpha_ld(r) for r in p0 * h])
    Yp = Y0 + h * (q0 - p0 * Y0) / (1 + a0 * p0 * h)                      # predictor
    Yp[-1] = 1.0 - Yp[:-1].sum()
    Tp = T0
    for _ in range(n_corr):                                               # corrector(s), reading R27
        Tp = T_of(Yp, Tp)
        qp, dp, _, _ = _rates_numpy(table, mech, rho, Yp, Tp)
        with np.errstate(divide="ignore", invalid="ignore"):
            pb = 0.5 * (p0 + np.where(Yp > 0.0, dp / Yp, 0.0))
        ab = np.array([_alpha_ld(r) for r in pb * h])
        qb = ab * qp + (1 - ab) * q0
        Yc = Y0 + h * (qb - pb * Y0) / (1 + ab * pb * h)
        Yc[-1] = 1.0 - Yc[:-1].sum()
        Yp = Yc
    T1 = T_of(Yp, Tp)
    st, U1, T1o = o.react_cell(om, U, 1400.0, h, 1, n_corr)
    assert st == 0
    Y1o = np.append(U1[5:], rho - U1[5:].sum()) / rho
    assert np.max(np.abs(Y1o - Yp)) <= 2e-12 * Yp.max(), np.max(np.abs(Y1o - Yp))
    assert abs(T1o - T1) <= 1e-11 * T1
    assert np.max(np.abs(Yp - Y0)) > 0.01                                  # the step really moves the composition
    # the predictor's alpha matters at this step size: with alpha = 1/2 in the predictor the result is visibly different
    Yp_half = Y0 + h * (q0 - p0 * Y0) / (1 + 0.5 * p0 * h)
    assert np.max(np.abs(Yp_half[:-1] - (Y0 + h * (q0 - p0 * Y0) / (1 + a0 * p0 * h))[:-1])) > 1e-6


def test_a_species_outside_the_mechanism_that_is_absent_stays_absent(oracle_mod):
    """Y_s = 0 and no reaction touches s: q_s = d_s = 0 through predictor AND corrector, where p_s = d_s / Y_s is 0 by the
    guard of reading R25 (0/0 otherwise); the species stays exactly absent and everything else finite."""
    table, mech, o, om = _setup(oracle_mod, n_reactions=3, seed=2)
    used = (mech.nu_r + mech.nu_p).sum(axis=0)
    idle = [s for s in range(8) if used[s] == 0]
    assert idle, "the seeded three-reaction mechanism leaves some species out"
    s0 = idle[-1]
    assert s0 > 0                                                # not the first species: a guard that looked at Y_0 instead must show
    Y0 = np.full(9, 0.1)
    Y0[8] = 0.2
    Y0[8] += Y0[s0]
    Y0[s0] = 0.0
    U, e = _cell(table, 1.1, (1.0, 0.0, 0.0), 1400.0, Y0)
    for n_corr in (1, 3):
        st, U1, T1 = o.react_cell(om, U, 1300.0, 1e-3, 2, n_corr)
        assert st == 0 and np.all(np.isfinite(U1)) and np.isfinite(T1)
        assert U1[5 + s0] == 0.0
        assert np.max(np.abs(U1[5:] - U[5:])) > 1e-6             # the others do react


@pytest.mark.parametrize("nz", [1, 4])
def test_field_call_touches_interior_species_only(oracle_mod, nz):
    table, mech, _, om = _setup(oracle_mod)
    rng = np.random.default_rng(9)
    nx, ny = 6, 5
    o = oracle_mod.Oracle(nx, ny, nz, 0.1, 0.1, 0.1 if nz > 1 else 1, table.W, table.nasa7, table.Ru, table.Tlo, table.Thi)
    gz = 3 if nz > 1 else 0
    shape = (nz + 2 * gz, ny + 6, nx + 6)
    Y = rng.dirichlet(np.ones(9), size=shape).transpose(3, 0, 1, 2)
    T = rng.uniform(900, 1500, shape)
    rho = rng.uniform(0.5, 2, shape)
    U = wl.conserved_from_primitive(table, rho, 0 * rho, 0 * rho, 0 * rho, T, Y)
    U0, T0 = U.copy(), T.copy()
    assert o.react(om, U, T, 1e-3, 2, 1) == 0
    assert np.array_equal(U[:5], U0[:5])
    mask = np.ones(shape, dtype=bool)
    mask[gz:shape[0] - gz, 3:-3, 3:-3] = False
    assert np.array_equal(U[5:][:, mask], U0[5:][:, mask]) and np.array_equal(T[mask], T0[mask])
    assert np.max(np.abs(U[5:, gz:shape[0] - gz, 3:-3, 3:-3] - U0[5:, gz:shape[0] - gz, 3:-3, 3:-3])) > 1e-4
    for k in range(gz, gz + nz):                                 # EVERY interior cell against the per-cell call
        for j in range(3, 3 + ny):
            for i in range(3, 3 + nx):
                st, Uc, Tc = o.react_cell(om, U0[:, k, j, i], T0[k, j, i], 1e-3, 2, 1)
                assert np.array_equal(Uc, U[:, k, j, i]) and Tc == T[k, j, i], (k, j, i)
