"""Pins of the oracle's WENO-CU6 reconstruction (PAPER.md:107 names it, ref 34, no formula:
DESIGN.md reading R16)."""
from pathlib import Path

import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl
from helpers import exact_riemann, single_species_workload

GOLDEN = Path(__file__).resolve().parent / "golden"


def _cell_average_poly(f):
    """degree-5 polynomial (numpy, ascending coefficients) whose averages over cells [-2.5,-1.5] .. [2.5,3.5] are f."""
    A = np.array([[((j - 2 + 0.5) ** (k + 1) - (j - 2 - 0.5) ** (k + 1)) / (k + 1) for k in range(6)] for j in range(6)])
    return np.linalg.solve(A, f)


def test_beta6_equals_its_definition_by_quadrature(oracle_mod):
    """beta_6 = sum_l int_{-1/2}^{1/2} (d^l p/dx^l)^2 dx, l = 1..5, evaluated with Gauss-Legendre on the interpolant."""
    rng = np.random.default_rng(6)
    xg, wg = np.polynomial.legendre.leggauss(12)
    xg, wg = 0.5 * xg, 0.5 * wg
    for _ in range(20):
        f = rng.uniform(-2, 3, 6)
        p = np.polynomial.Polynomial(_cell_average_poly(f))
        ref = sum(float(np.sum(wg * p.deriv(l)(xg) ** 2)) for l in range(1, 6))
        _, beta, _ = oracle_mod.wenocu6(f)
        assert abs(beta[3] - ref) <= 1e-10 * ref
        # beta_0..beta_2 are the same measure (l = 1, 2) of the three quadratic interpolants
        for k in range(3):
            A = np.array([[((j + 0.5) ** (m + 1) - (j - 0.5) ** (m + 1)) / (m + 1) for m in range(3)]
                          for j in range(k - 2, k + 1)])
            q = np.polynomial.Polynomial(np.linalg.solve(A, f[k:k + 3]))
            refk = sum(float(np.sum(wg * q.deriv(l)(xg) ** 2)) for l in (1, 2))
            assert abs(beta[k] - refk) <= 1e-11 * max(refk, 1e-30)


def test_beta6_quadratic_form_matches_the_exact_derivation(oracle_mod):
    rows = dict(ln.split("=") for ln in (GOLDEN / "wenocu6_beta6_form.txt").read_text().split("\n")
                if "=" in ln and not ln.startswith("#"))
    C = np.zeros((6, 6))
    for a in range(6):
        for k, val in enumerate(rows[f"row{a}"].split(",")):
            C[a, a + k] = float(val)
    rng = np.random.default_rng(61)
    for _ in range(10):
        f = rng.uniform(-1, 1, 6)
        ref = sum(C[a, b] * f[a] * f[b] for a in range(6) for b in range(a, 6)) / 120960.0
        assert abs(oracle_mod.wenocu6(f)[1][3] - ref) <= 1e-12 * abs(ref)
    # translation invariance, which the oracle's first-difference form relies on: the value form annihilates constants
    assert abs(sum(C[a, b] for a in range(6) for b in range(a, 6))) == 0.0


def test_ideal_weights_give_the_sixth_order_central_flux(oracle_mod):
    """point values of a degree-6 polynomial as the split flux: (h_{i+1/2} - h_{i-1/2})/dx = f'(x_i) exactly."""
    rng = np.random.default_rng(7)
    c = rng.uniform(-1, 1, 7)
    f = np.polynomial.Polynomial(c)
    dx, x0 = 0.37, 0.2
    xs = x0 + dx * np.arange(-3, 4)                            # cells i-3 .. i+3
    v = f(xs)
    hp, _, w = oracle_mod.wenocu6(v[1:7], ideal=True)
    hm, _, _ = oracle_mod.wenocu6(v[0:6], ideal=True)
    assert np.allclose(w, [0.05, 0.45, 0.45, 0.05])
    assert abs((hp - hm) / dx - f.deriv()(x0)) <= 1e-12 * abs(f.deriv()(x0))


def test_nonlinear_weights_sixth_order_on_smooth_data_and_upwind_at_a_jump(oracle_mod):
    errs = []
    for n in (32, 64, 128):
        dx = 1.0 / n
        x = 0.3 + dx * np.arange(-3, 4)
        v = np.sin(2 * np.pi * x) + 2.0
        hp = oracle_mod.wenocu6(v[1:7])[0]
        hm = oracle_mod.wenocu6(v[0:6])[0]
        errs.append(abs((hp - hm) / dx - 2 * np.pi * np.cos(2 * np.pi * 0.3)))
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(orders > 5.5), (errs, orders)
    # a jump between v_{+1} and v_{+2}: the two stencils that cross it lose their weight (completely when the smooth side
    # is flat: alpha ~ d (C + tau/beta) with beta -> eps = 1e-40); what is left is q0, q1 at the ratio 1:9
    val, beta, w = oracle_mod.wenocu6(np.array([1.0, 1.0, 1.0, 1.0, 5.0, 5.0]))
    assert w[2] < 1e-30 and w[3] < 1e-30 and abs(w[0] - 0.1) < 1e-12 and abs(w[1] - 0.9) < 1e-12 and val == 1.0
    val, beta, w = oracle_mod.wenocu6(np.array([1.0, 1.1, 1.2, 1.3, 5.0, 5.1]))
    tau = beta[3] - (beta[0] + 4 * beta[1] + beta[2]) / 6
    a = np.array([0.05, 0.45, 0.45, 0.05]) * (20.0 + tau / (beta + 1e-40))     # the definition, written out
    assert np.allclose(w, a / a.sum(), rtol=1e-13, atol=0)
    assert w[2] + w[3] < 5e-3 and abs(w[0] / w[1] - 1.0 / 9.0) < 1e-3
    q = [(2 * 1.0 - 7 * 1.1 + 11 * 1.2) / 6, (-1.1 + 5 * 1.2 + 2 * 1.3) / 6, (2 * 1.2 + 5 * 1.3 - 5.0) / 6,
         (11 * 1.3 - 7 * 5.0 + 2 * 5.1) / 6]
    assert abs(val - float(np.dot(w, q))) < 1e-12
    # mirrored: jump between v_{-2} and v_{-1}: stencil 0 drops out
    _, _, w = oracle_mod.wenocu6(np.array([5.0, 1.0, 1.0, 1.0, 1.0, 1.0]))
    assert w[0] < 1e-30


def _oracle(oracle_mod, w):
    return oracle_mod.Oracle.from_workload(w, recon=1)


def test_scheme_level_uniform_flow_sod_and_conservation(oracle_mod):
    nx, tend = 400, 0.2
    x = (np.arange(nx) + 0.5) / nx
    rho = np.where(x < 0.5, 1.0, 0.125).reshape(1, 1, nx)
    p = np.where(x < 0.5, 1.0, 0.1).reshape(1, 1, nx)
    w = single_species_workload(nx, rho, np.zeros_like(rho), p, bc=(wl.BC_TRANSMISSIVE,) * 6)
    o = _oracle(oracle_mod, w)
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
    assert np.max(np.abs(pr[plateau] - pstar)) < 3e-3 and np.max(np.abs(u[plateau] - ustar)) < 3e-3
    # uniform 3-D multi-species state: rhs = 0; periodic random box: conservation to round-off
    w3 = wl.random_smooth_box(10, 9, 8, nspecies=3, seed=12)
    o3 = _oracle(oracle_mod, w3)
    U, T = w3.U.copy(), w3.T_guess.copy()
    m0 = w3.interior(U).sum(axis=(1, 2, 3))
    S = o3.max_wavespeed(U, T)
    for _ in range(3):
        o3.rk3_step(U, T, 0.4 / S)
    m1 = w3.interior(U).sum(axis=(1, 2, 3))
    scale = np.abs(m0).copy()
    scale[1:4] = np.abs(w3.interior(U)[0]).sum() * S * w3.dx
    assert np.max(np.abs(m1 - m0) / scale) <= 1e-12


@pytest.mark.parametrize("nsp", [1])
def test_design_order_on_the_advected_density_wave(oracle_mod, nsp):
    errs = []
    for nx in (16, 32, 64):
        x = (np.arange(nx) + 0.5) / nx
        rho = (1.0 + 0.2 * np.sin(2 * np.pi * x)).reshape(1, 1, nx)
        w = single_species_workload(nx, rho, np.ones_like(rho), np.ones_like(rho))
        o = _oracle(oracle_mod, w)
        U, T = w.U.copy(), w.T_guess.copy()
        dx = 1.0 / nx
        nsteps = int(np.ceil(1.0 / (0.4 * dx ** 2 * 4.0)))    # dt ~ dx^2: time error O(dx^6)
        for _ in range(nsteps):
            o.rk3_step(U, T, 1.0 / nsteps)
        errs.append(np.mean(np.abs(w.interior(U)[0, 0, 0] - rho[0, 0])))
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(orders >= 5.5), (errs, orders)
