"""Pins of the parts of the oracle that round 1 left held by nothing ("What's weak" 1-2):

* ``xo_max_wavespeed`` -- S written out by hand for one hand-built cell (reading R9: SUM over the active directions,
  INTERIOR cells only);
* ``xo_rhs_cells`` (the sampled-cell checker of the full-size GPU parity test) against ``xo_rhs`` at every interior cell;
* the Roe-type average of reading R5 -- the sqrt(rho) weighting of Gamma~, Y~_s, chi~_s -- written out from its
  definition.  L R = I holds for any average; what the mathematics does fix is pinned by Roe's property U
  (F_b - F_a = A~ (U_b - U_a)): the species and tangential-momentum rows for a three-species mixture (u~, v~, w~, Y~_s)
  and every row for one perfect gas (H~, c~^2).  The weighting of Gamma~ and chi~_s is fixed by nothing in PAPER.md:107
  or in the mathematics, so for those two the pin only guards the DEFINITION against slips; DESIGN.md section 3 lists
  them as "parity unpinned";
* beta_6 of ``xo_wenocu6`` against exact rational arithmetic on smooth data (the case that motivated evaluating it on
  first differences, reading R16).

The gases here are calorically perfect and every thermodynamic quantity is written out in the test from
cp_s = R_s a1_s, e_s = R_s ((a1_s - 1) T + a6_s): nothing is taken from ``workloads.py``'s table evaluation.
"""
from fractions import Fraction as Fr
from pathlib import Path

import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

GOLDEN = Path(__file__).resolve().parent / "golden"

RU = 8.0
W2 = np.array([28.0, 4.0])
GAM2 = np.array([1.4, 5.0 / 3.0])
A6 = np.array([-350.0, 900.0])          # enthalpy constants (K): chi_s = R_s T - Gamma e_s then differs per species


def _nasa7(gam, a6):
    a = np.zeros((len(gam), 7))
    a[:, 0] = gam / (gam - 1.0)
    a[:, 5] = a6
    return a


def _state(rho, vel, T, Y, W=W2, gam=GAM2, a6=A6):
    """conserved vector and the primitives of a calorically perfect mixture, every formula written out"""
    Rs = RU / W
    a1 = gam / (gam - 1.0)
    Rbar = float(np.sum(Y * Rs))
    es = Rs * ((a1 - 1.0) * T + a6)                 # e_s = h_s - R_s T, h_s = R_s (a1 T + a6)
    e = float(np.sum(Y * es))
    cv = float(np.sum(Y * Rs * (a1 - 1.0)))
    Gamma = Rbar / cv
    p = rho * Rbar * T
    k = 0.5 * float(np.dot(vel, vel))
    E = rho * (e + k)
    U = np.array([rho, *(rho * np.asarray(vel)), E, *(rho * Y[:-1])])
    prim = dict(rho=rho, vel=np.asarray(vel, dtype=float), T=T, Y=np.asarray(Y, dtype=float), p=p, Gamma=Gamma,
                c=float(np.sqrt((1.0 + Gamma) * p / rho)), H=(E + p) / rho, chi=Rs * T - Gamma * es)
    return U, prim


# --------------------------------------------------------------------------------------------------------------
# xo_max_wavespeed (Eq. 17; reading R9)
# --------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(5, 4, 6), (7, 5, 1), (1, 6, 4), (9, 1, 1)])
def test_max_wavespeed_is_the_sum_over_active_directions_of_one_hand_built_cell(oracle_mod, dims):
    nx, ny, nz = dims
    dx, dy, dz = 0.1, 0.23, 0.37
    o = oracle_mod.Oracle(nx, ny, nz, dx, dy, dz, W2, _nasa7(GAM2, A6), RU, 0.0, 1e300)
    nzp, nyp, nxp = o.shape
    g = [3 if n > 1 else 0 for n in (nx, ny, nz)]
    Ubg, _ = _state(1.0, (0.0, 0.0, 0.0), 300.0, np.array([0.5, 0.5]))
    U = np.empty((6, nzp, nyp, nxp))
    U[:] = Ubg[:, None, None, None]
    T = np.full((nzp, nyp, nxp), 280.0)
    # the one fast, hot interior cell; all three velocity components non-zero, also along inactive directions
    vel = (30.0, -50.0, 20.0)
    Uh, ph = _state(2.0, vel, 900.0, np.array([0.3, 0.7]))
    kc, jc, ic = g[2] + nz // 2, g[1] + ny // 2, g[0] + nx - 1
    U[:, kc, jc, ic] = Uh
    # a GHOST cell faster and hotter than every interior cell: must not count (xo_max_wavespeed: interior only)
    Ug, _ = _state(0.5, (900.0, 900.0, -900.0), 6000.0, np.array([0.1, 0.9]))
    U[:, 0, 0, 0] = Ug
    active = [n > 1 for n in (nx, ny, nz)]
    S_hand = sum((abs(v) + ph["c"]) / d for v, d, a in zip(vel, (dx, dy, dz), active) if a)
    # the background cell is slower: c0/dx + c0/dy + c0/dz
    _, p0 = _state(1.0, (0.0, 0.0, 0.0), 300.0, np.array([0.5, 0.5]))
    assert S_hand > sum(p0["c"] / d for d, a in zip((dx, dy, dz), active) if a)
    S = o.max_wavespeed(U, T)
    assert o.last_status == 0
    assert abs(S - S_hand) <= 4e-15 * S_hand
    if sum(active) > 1:                                        # the sum differs from the largest single term
        assert S_hand > 1.2 * max((abs(v) + ph["c"]) / d for v, d, a in zip(vel, (dx, dy, dz), active) if a)
    assert abs(T[kc, jc, ic] - 900.0) <= 1e-12 * 900.0         # T of the interior cells is recovered on the way


# --------------------------------------------------------------------------------------------------------------
# xo_rhs_cells == xo_rhs at every interior cell
# --------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("recon", [0, 1])
@pytest.mark.parametrize("visc", [0, 1, 2])
@pytest.mark.parametrize("shape,bc", [((9, 8, 7), (3, 1, 2, 2, 0, 0)), ((12, 1, 1), (1, 1, 0, 0, 0, 0)),
                                      ((6, 11, 1), (0, 0, 2, 1, 0, 0))])
def test_rhs_cells_equals_rhs_at_every_interior_cell(oracle_mod, shape, bc, visc, recon):
    w = wl.random_smooth_box(*shape, nspecies=3, seed=811, bc=bc)
    if 3 in bc:
        w.bc_state = np.tile(w.interior(w.U)[:, 0, 0, 0], (6, 1))
    o = oracle_mod.Oracle.from_workload(w, viscosity=visc, recon=recon)
    U, T = w.U.copy(), w.T_guess.copy()
    r = o.rhs(U, T)                                            # fills the ghosts of U
    assert o.last_status == 0
    nzp, nyp, nxp = w.padded_shape
    kk, jj, ii = np.meshgrid(*(np.arange(3 if n > 1 else 0, (3 if n > 1 else 0) + n) for n in (w.nz, w.ny, w.nx)),
                             indexing="ij")
    idx = ((kk * nyp + jj) * nxp + ii).ravel()
    rc = o.rhs_cells(U, w.T_guess, idx)                        # [cells, Nv], Newton from the same guess
    assert o.last_status == 0
    rf = r.reshape(w.nvars, -1)[:, idx].T
    scale = np.abs(rf).max(axis=0)
    scale[1:4] = scale[1:4].max()                              # an inactive direction's momentum residual is zero
    # bit-identical for LLF / ROE; GLF: the global maxima come from a Newton iteration restarted at the converged T in
    # xo_rhs and at the guess in xo_rhs_cells (last-bit differences of c)
    assert np.max(np.abs(rc - rf) / scale) <= (5e-15 if visc == 2 else 1e-15)


# --------------------------------------------------------------------------------------------------------------
# reading R5: the Roe-type average written out from its definition
# --------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("d", [0, 1, 2])
def test_roe_average_weights_of_reading_R5_written_out(oracle_mod, d):
    o = oracle_mod.Oracle(4, 1, 1, 0.25, 1.0, 1.0, W2, _nasa7(GAM2, A6), RU, 0.0, 1e300)
    # very different densities (weights 1 : 3.65) and compositions, so that an arithmetic mean is far off
    Ua, a = _state(0.3, (40.0, -15.0, 22.0), 450.0, np.array([0.85, 0.15]))
    Ub, b = _state(4.0, (-10.0, 35.0, 5.0), 1300.0, np.array([0.2, 0.8]))
    Pa, Pb = o.cell_primitives(Ua, 400.0), o.cell_primitives(Ub, 1000.0)
    for P, ref in ((Pa, a), (Pb, b)):                          # the cell quantities that enter the average
        assert abs(P.Gamma - ref["Gamma"]) <= 1e-14 * ref["Gamma"] and abs(P.H - ref["H"]) <= 1e-14 * abs(ref["H"])
        assert np.allclose([P.chi[0], P.chi[1]], ref["chi"], rtol=1e-13, atol=0)
    L, R, roe, st = o.eigensystem(Pa, Pb, d)
    assert st == 0
    wa, wb = np.sqrt(a["rho"]), np.sqrt(b["rho"])

    def avg(qa, qb):
        return (wa * qa + wb * qb) / (wa + wb)

    vt, Ht, Gt = avg(a["vel"], b["vel"]), avg(a["H"], b["H"]), avg(a["Gamma"], b["Gamma"])
    Yt, chit = avg(a["Y"], b["Y"]), avg(a["chi"], b["chi"])
    kt = 0.5 * float(vt @ vt)
    c2 = float(Yt @ chit) + Gt * (Ht - kt)                     # the identity that makes L R = I
    assert np.allclose(roe[:3], vt, rtol=1e-14, atol=0)
    assert abs(roe[3] - Ht) <= 1e-14 * abs(Ht)
    assert abs(roe[4] - Gt) <= 1e-14 * Gt
    assert abs(roe[5] - np.sqrt(c2)) <= 1e-14 * np.sqrt(c2)
    # Y~_1 sits in the species row of L; chi~_s follow from the pressure functional pi = (e_0 - l_1) c~^2:
    # pi_0 = chi~_N + Gamma~ k~, pi_5 = chi~_1 - chi~_N
    assert abs(-L[4, 0] - Yt[0]) <= 1e-14
    pi = (np.eye(6)[0] - L[1]) * c2
    chiN = pi[0] - Gt * kt
    assert abs(chiN - chit[1]) <= 1e-12 * abs(chit[1])
    assert abs(pi[5] + chiN - chit[0]) <= 1e-12 * abs(chit[0])
    assert abs(pi[4] - Gt) <= 1e-13 * Gt
    # and the arithmetic means really are far from these (so the pin distinguishes the two readings)
    assert abs(0.5 * (a["Gamma"] + b["Gamma"]) - Gt) > 1e-2 * Gt
    assert abs(0.5 * (a["Y"][0] + b["Y"][0]) - Yt[0]) > 1e-2
    assert abs(0.5 * (a["chi"][0] + b["chi"][0]) - chit[0]) > 1e-2 * abs(chit[0])


# --------------------------------------------------------------------------------------------------------------
# reading R5, the part the mathematics DOES fix: Roe's property U.  With A~ = R diag(lambda) L of the averaged state,
# F(U_b) - F(U_a) = A~ (U_b - U_a) holds row by row exactly when the average is the sqrt(rho)-weighted one:
#   * tangential-momentum rows  Delta(rho u v) = -u~ v~ Delta rho + v~ Delta(rho u) + u~ Delta(rho v)
#   * species rows               Delta(rho u Y_s) = -u~ Y~_s Delta rho + Y~_s Delta(rho u) + u~ Delta(rho Y_s)
#   for ANY equation of state (these rows of A~ hold only u~, v~, w~, Y~_s), and for one calorically perfect gas with
#   a6 = 0 (chi = 0, Gamma = gamma - 1 constant) in ALL rows, which fixes H~ and c~^2 as well (Roe 1981).
# An arithmetic mean of u, Y_s or H fails them at O(1).  What stays a definition is the weighting of Gamma~ and chi~_s.
# --------------------------------------------------------------------------------------------------------------
def _roe_matrix(o, Pa, Pb, d):
    L, R, roe, st = o.eigensystem(Pa, Pb, d)
    assert st == 0
    Nv = L.shape[0]
    un, c = roe[d], roe[5]
    lam = np.full(Nv, un)                                       # fields: u - c, u (entropy, shear x 2, species), u + c
    lam[0], lam[Nv - 1] = un - c, un + c
    return R @ np.diag(lam) @ L


@pytest.mark.parametrize("d", [0, 1, 2])
def test_roe_property_U_fixes_the_weights_of_velocity_and_mass_fractions(oracle_mod, d):
    W3 = np.array([28.0, 4.0, 44.0])
    g3 = np.array([1.4, 5.0 / 3.0, 1.29])
    a63 = np.array([-350.0, 900.0, 120.0])
    o = oracle_mod.Oracle(4, 1, 1, 0.25, 1.0, 1.0, W3, _nasa7(g3, a63), RU, 0.0, 1e300)
    Ua, a = _state(0.3, (40.0, -15.0, 22.0), 450.0, np.array([0.6, 0.15, 0.25]), W3, g3, a63)
    Ub, b = _state(4.0, (-10.0, 35.0, 5.0), 1300.0, np.array([0.1, 0.7, 0.2]), W3, g3, a63)
    Pa, Pb = o.cell_primitives(Ua, 400.0), o.cell_primitives(Ub, 1000.0)
    A = _roe_matrix(o, Pa, Pb, d)
    dU = Ub - Ua
    dF = o.phys_flux(Ub, Pb, d) - o.phys_flux(Ua, Pa, d)
    AdU = A @ dU
    rows = [0] + [1 + q for q in range(3) if q != d] + [5, 6]   # mass, the two tangential momenta, both species
    rowscale = np.abs(A) @ np.abs(dU)                            # each row against the size of its own terms
    assert np.max(np.abs(AdU[rows] - dF[rows]) / rowscale[rows]) <= 1e-13
    # written out: the species and tangential rows of A~ dU with sqrt(rho) weights equal the flux jump ...
    wa, wb = np.sqrt(a["rho"]), np.sqrt(b["rho"])
    ut = (wa * a["vel"] + wb * b["vel"]) / (wa + wb)
    Yt = (wa * a["Y"] + wb * b["Y"]) / (wa + wb)
    for s in range(2):
        row = -ut[d] * Yt[s] * dU[0] + Yt[s] * dU[1 + d] + ut[d] * dU[5 + s]
        assert abs(row - dF[5 + s]) <= 1e-13 * rowscale[5 + s]
    # ... and with arithmetic means they do not (so the property distinguishes the two)
    um, Ym = 0.5 * (a["vel"] + b["vel"]), 0.5 * (a["Y"] + b["Y"])
    row = -um[d] * Ym[0] * dU[0] + Ym[0] * dU[1 + d] + um[d] * dU[5]
    assert abs(row - dF[5]) > 1e-2 * rowscale[5]


@pytest.mark.parametrize("d", [0, 1, 2])
def test_roe_property_U_in_all_rows_for_one_perfect_gas(oracle_mod, d):
    W1, g1, z1 = np.array([28.0]), np.array([1.4]), np.array([0.0])
    o = oracle_mod.Oracle(4, 1, 1, 0.25, 1.0, 1.0, W1, _nasa7(g1, z1), RU, 0.0, 1e300)
    Ua, a = _state(0.3, (40.0, -15.0, 22.0), 450.0, np.array([1.0]), W1, g1, z1)
    Ub, b = _state(4.0, (-10.0, 35.0, 5.0), 1300.0, np.array([1.0]), W1, g1, z1)
    Pa, Pb = o.cell_primitives(Ua, 400.0), o.cell_primitives(Ub, 1000.0)
    A = _roe_matrix(o, Pa, Pb, d)
    dF = o.phys_flux(Ub, Pb, d) - o.phys_flux(Ua, Pa, d)
    assert np.max(np.abs(A @ (Ub - Ua) - dF)) <= 1e-12 * np.abs(dF).max()
    # the energy row fails by O(1) if H~ were the arithmetic mean (c~^2 = (gamma - 1)(H~ - k~) would move with it)
    L, R, roe, _ = o.eigensystem(Pa, Pb, d)
    assert abs(roe[3] - 0.5 * (a["H"] + b["H"])) > 1e-2 * abs(roe[3])


# --------------------------------------------------------------------------------------------------------------
# beta_6 of WENO-CU6 on smooth data against exact rational arithmetic (reading R16)
# --------------------------------------------------------------------------------------------------------------
def _beta6_value_form():
    rows = dict(ln.split("=") for ln in (GOLDEN / "wenocu6_beta6_form.txt").read_text().split("\n")
                if "=" in ln and not ln.startswith("#"))
    return [[int(x) for x in rows[f"row{a}"].split(",")] for a in range(6)]


def _beta6_exact(v, C):
    f = [Fr(float(x)) for x in v]                              # the doubles themselves, exactly
    return sum(C[a][k] * f[a] * f[a + k] for a in range(6) for k in range(6 - a)) / 120960


def test_beta6_on_smooth_data_matches_exact_rational_arithmetic(oracle_mod):
    """A smooth wave at 150 points per wavelength: beta_6 is ~ (cell-to-cell difference)^2 ~ 1e-3 while the value form
    of tests/golden/wenocu6_beta6_form.txt sums terms up to 3.6e7/120960 * v^2 ~ 3e3 -- evaluated in doubles it is off by
    ~1e-12 of that difference, evaluated on first differences (xo_wenocu6) by < 1e-13.  The expected values are exact:
    fractions.Fraction on the very doubles handed to the oracle."""
    C = _beta6_value_form()
    n = 150
    worst_oracle, worst_value_form = 0.0, 0.0
    for j0 in range(0, n, 7):
        x = (j0 + np.arange(6)) / n
        v = 2.0 + np.sin(2 * np.pi * x) + 0.3 * np.cos(6 * np.pi * x)
        D2 = float(np.max(np.diff(v) ** 2))
        exact = _beta6_exact(v, C)
        _, beta, _ = oracle_mod.wenocu6(v)
        worst_oracle = max(worst_oracle, abs(float(Fr(float(beta[3])) - exact)) / D2)
        vf = sum(C[a][k] * v[a] * v[a + k] for a in range(6) for k in range(6 - a)) / 120960.0
        worst_value_form = max(worst_value_form, abs(float(Fr(float(vf)) - exact)) / D2)
    assert worst_oracle <= 2e-13, worst_oracle
    assert worst_value_form > 10 * worst_oracle                # the cancellation the first-difference form avoids


def test_beta6_smooth_golden_values(oracle_mod):
    """the same check against stored exact values (tests/golden/wenocu6_beta6_smooth.txt, written by make_golden.py from
    fractions.Fraction alone)"""
    lines = [ln for ln in (GOLDEN / "wenocu6_beta6_smooth.txt").read_text().splitlines() if ln and ln[0] != "#"]
    assert len(lines) >= 5
    for ln in lines:
        vs, bs = ln.split(";")
        v = np.array([float.fromhex(t) for t in vs.split(",")])
        exact = float.fromhex(bs)
        D2 = float(np.max(np.diff(v) ** 2))
        assert abs(oracle_mod.wenocu6(v)[1][3] - exact) <= 2e-13 * D2
