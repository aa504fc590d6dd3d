"""Seeded synthetic workloads: the input generators shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no Newton T(e), no eigensystem, no WENO, no flux, no RK): it
only manufactures thermodynamically consistent *inputs* -- conserved fields U, a temperature guess, a species
table and boundary data -- in the layout both sides consume (SoA ``U[v][k][j][i]``, i fastest, 3 ghost layers
on every active direction).  It imports neither ``oracle/`` nor the CUDA binding.

The paper's own workloads (PAPER.md:521-527 shock tube; PAPER.md:605-631 shock-bubble interaction, Eq. 32-33)
use real species (N2, O2, Xe, H2, Ar) whose NASA coefficient sets are not in this container and are not to be
written from memory; the generators below take those workloads' *shapes* (two-state Riemann data; planar shock
+ tanh bubble interface in mole fraction, Eq. 32; post-shock state by Rankine-Hugoniot, Eq. 33; zeta = 1e-4
floor; Ma = 2.83) with seeded synthetic NASA-7-style tables and stand in for them (DESIGN.md "Input recipe",
SURVEY.md 8(d)).

The one piece of thermodynamics needed to manufacture a conserved state from (rho, u, T, Y) is the *meaning of
the table*: h_s(T) = R_s (a1 T + a2 T^2/2 + ... + a5 T^5/5 + a6) inside [Tlo, Thi] (NASA
polynomials) with the constant-cp continuation outside it (reading R3).  It is evaluated here with
numpy, forward only (T -> e); the path under test does the inverse (e -> T by Newton, Eq. 21).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Sequence, Tuple

import numpy as np

NG = 3  # ghost width of WENO5: stencil m = i-2 .. i+3 for face i+1/2 (k = 3)

BC_PERIODIC, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_DIRICHLET = 0, 1, 2, 3

SEED_BASE = 24030591 * 10  # seed = SEED_BASE + config index (SURVEY.md 8(d) "Common generator rules")

W10 = (2.016, 32.0, 18.015, 1.008, 16.0, 17.007, 33.006, 34.014, 131.29, 28.014)  # BASELINE.json configs[3]


# ----------------------------------------------------------------------------------------------------------------
# species tables
# ----------------------------------------------------------------------------------------------------------------
@dataclass
class SpeciesTable:
    """N species: molar masses W[N], NASA-7 single-range coefficients nasa7[N][7] (a7 unused), fit range."""

    W: np.ndarray
    nasa7: np.ndarray
    Tlo: float
    Thi: float
    Ru: float

    @property
    def n(self) -> int:
        return int(self.W.shape[0])

    @property
    def Rs(self) -> np.ndarray:
        return self.Ru / self.W

    # --- forward evaluation of the table (input manufacture only) ---
    def cp_over_R(self, T: np.ndarray) -> np.ndarray:
        """cp_s/R_s at temperature array T -> shape (N,) + T.shape; frozen outside [Tlo, Thi]."""
        Tc = np.clip(np.asarray(T, dtype=np.float64), self.Tlo, self.Thi)
        a = self.nasa7
        out = np.empty((self.n,) + Tc.shape)
        for s in range(self.n):
            out[s] = a[s, 0] + Tc * (a[s, 1] + Tc * (a[s, 2] + Tc * (a[s, 3] + Tc * a[s, 4])))
        return out

    def h_over_R(self, T: np.ndarray) -> np.ndarray:
        """h_s/R_s (units of kelvin) -> (N,) + T.shape, linear continuation outside the fit range."""
        T = np.asarray(T, dtype=np.float64)
        Tc = np.clip(T, self.Tlo, self.Thi)
        a = self.nasa7
        cp = self.cp_over_R(T)
        out = np.empty((self.n,) + Tc.shape)
        for s in range(self.n):
            poly = Tc * (a[s, 0] + Tc * (a[s, 1] / 2 + Tc * (a[s, 2] / 3 + Tc * (a[s, 3] / 4 + Tc * a[s, 4] / 5))))
            out[s] = poly + a[s, 5] + cp[s] * (T - Tc)
        return out

    def mixture_R(self, Y: np.ndarray) -> np.ndarray:
        return np.tensordot(self.Rs, Y, axes=(0, 0))

    def mixture_W_from_X(self, X: np.ndarray) -> np.ndarray:
        return np.tensordot(self.W, X, axes=(0, 0))

    def X_to_Y(self, X: np.ndarray) -> np.ndarray:
        """mole -> mass fractions: Y_s = X_s W_s / sum_t X_t W_t."""
        shp = (self.n,) + (1,) * (X.ndim - 1)
        num = X * self.W.reshape(shp)
        return num / num.sum(axis=0)

    def frozen_gamma(self, Y: np.ndarray, T: np.ndarray) -> np.ndarray:
        shp = (self.n,) + (1,) * (np.ndim(T))
        cp = (Y * self.Rs.reshape(shp) * self.cp_over_R(T)).sum(axis=0)
        return cp / (cp - self.mixture_R(Y))

    def internal_energy(self, Y: np.ndarray, T: np.ndarray) -> np.ndarray:
        """e(T, Y) = sum_s Y_s h_s(T) - Rbar T  (Eq. 21 middle line), forward direction."""
        shp = (self.n,) + (1,) * (np.ndim(T))
        h = (Y * self.Rs.reshape(shp) * self.h_over_R(T)).sum(axis=0)
        return h - self.mixture_R(Y) * T


def calorically_perfect_table(W: Sequence[float], gamma: Sequence[float], Ru: float = 1.0,
                              a6: Optional[Sequence[float]] = None) -> SpeciesTable:
    """a1 = gamma/(gamma-1), a2..a5 = 0; unlimited fit range."""
    W = np.asarray(W, dtype=np.float64)
    g = np.asarray(gamma, dtype=np.float64)
    a = np.zeros((W.shape[0], 7))
    a[:, 0] = g / (g - 1.0)
    if a6 is not None:
        a[:, 5] = np.asarray(a6, dtype=np.float64)
    return SpeciesTable(W=W, nasa7=a, Tlo=0.0, Thi=1e300, Ru=float(Ru))


def synthetic_nasa7_table(W: Sequence[float], Ru: float, rng: np.random.Generator,
                          formation: bool = False) -> SpeciesTable:
    """Seeded synthetic NASA-7-style species (BASELINE.json configs[1]).

    a1 ~ U[2.5, 4.0]; r ~ U[0.05, 0.30]; beta ~ U[0, 1]; theta = T/3000;
    s(theta) = (1-beta) theta + beta (4 theta - 6 theta^2 + 4 theta^3 - theta^4)   (monotone on [0, 1]);
    cp/R = a1 + Delta s(theta), Delta chosen so cp(3000 K)/cp(200 K) = 1 + r exactly.
    a6 makes h_s(298.15 K) = 0; with ``formation=True`` a6 gets an extra U[-2000, 2000] K so that the
    formation-enthalpy (chi_s) terms are exercised.
    """
    W = np.asarray(W, dtype=np.float64)
    n = W.shape[0]
    a1 = rng.uniform(2.5, 4.0, n)
    r = rng.uniform(0.05, 0.30, n)
    beta = rng.uniform(0.0, 1.0, n)

    def s_of(theta):
        return (1 - beta) * theta + beta * (4 * theta - 6 * theta ** 2 + 4 * theta ** 3 - theta ** 4)

    delta = r * a1 / (s_of(1.0) - (1 + r) * s_of(1.0 / 15.0))
    a = np.zeros((n, 7))
    a[:, 0] = a1
    a[:, 1] = delta * (1 + 3 * beta) / 3000.0
    a[:, 2] = -6 * delta * beta / 3000.0 ** 2
    a[:, 3] = 4 * delta * beta / 3000.0 ** 3
    a[:, 4] = -delta * beta / 3000.0 ** 4
    tab = SpeciesTable(W=W, nasa7=a, Tlo=200.0, Thi=3000.0, Ru=float(Ru))
    a[:, 5] = -tab.h_over_R(np.float64(298.15))
    if formation:
        a[:, 5] += rng.uniform(-2000.0, 2000.0, n)
    return tab


# ----------------------------------------------------------------------------------------------------------------
# workload container
# ----------------------------------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    table: SpeciesTable
    bc: Tuple[int, int, int, int, int, int]
    U: np.ndarray                      # [Nv, nzp, nyp, nxp] padded, ghosts edge-replicated (refilled by the path)
    T_guess: np.ndarray                # [nzp, nyp, nxp] Newton starting guess
    bc_state: Optional[np.ndarray] = None   # [6, Nv] conserved Dirichlet states
    cfl: float = 0.5                   # PAPER.md:135 (CFL <= 0.5)
    steps: int = 1
    notes: dict = field(default_factory=dict)
    ng: int = NG                       # ghost width of the arrays: 3, or 4 for WENO7 (see ``with_ghost_width``)

    @property
    def nspecies(self) -> int:
        return self.table.n

    @property
    def nvars(self) -> int:
        return self.table.n + 4

    @property
    def padded_shape(self) -> Tuple[int, int, int]:
        return tuple(self.U.shape[1:])

    @property
    def interior_cells(self) -> int:
        return self.nx * self.ny * self.nz

    def interior(self, A: np.ndarray) -> np.ndarray:
        """View of the interior cells of a padded [..., nzp, nyp, nxp] array."""
        gx = self.ng if self.nx > 1 else 0
        gy = self.ng if self.ny > 1 else 0
        gz = self.ng if self.nz > 1 else 0
        return A[..., gz:gz + self.nz, gy:gy + self.ny, gx:gx + self.nx]


def padded_dims(nx: int, ny: int, nz: int) -> Tuple[int, int, int]:
    """A direction with one interior cell is inactive: no ghosts, no sweep (SURVEY.md 8 notation)."""
    return (nz + 2 * NG if nz > 1 else 1, ny + 2 * NG if ny > 1 else 1, nx + 2 * NG if nx > 1 else 1)


def _pad(A: np.ndarray, nx: int, ny: int, nz: int, ng: int = NG) -> np.ndarray:
    """interior [..., nz, ny, nx] -> padded, edge-replicated ghosts."""
    pw = [(0, 0)] * (A.ndim - 3) + [(ng, ng) if n > 1 else (0, 0) for n in (nz, ny, nx)]
    return np.ascontiguousarray(np.pad(A, pw, mode="edge"))


def with_ghost_width(w: "Workload", ng: int) -> "Workload":
    """The same workload with ``ng`` ghost layers per active direction (WENO7 needs 4: stencil i-3..i+4)."""
    import dataclasses

    return dataclasses.replace(w, U=_pad(np.ascontiguousarray(w.interior(w.U)), w.nx, w.ny, w.nz, ng),
                               T_guess=_pad(np.ascontiguousarray(w.interior(w.T_guess)), w.nx, w.ny, w.nz, ng), ng=ng)


def conserved_from_primitive(table: SpeciesTable, rho, u, v, w, T, Y) -> np.ndarray:
    """(rho, u, v, w, T, Y[N]) -> U[Nv] = (rho, rho u, rho v, rho w, E, rho Y_1..rho Y_{N-1})  (Eq. 2)."""
    rho = np.asarray(rho, dtype=np.float64)
    e = table.internal_energy(Y, T)
    n = table.n
    U = np.empty((n + 4,) + rho.shape)
    U[0] = rho
    U[1] = rho * u
    U[2] = rho * v
    U[3] = rho * w
    U[4] = rho * (e + 0.5 * (u * u + v * v + w * w))
    for s in range(n - 1):
        U[5 + s] = rho * Y[s]
    return U


def _finish(name, nx, ny, nz, dx, dy, dz, table, bc, Uint, Tint, rng, bc_state=None, steps=1, notes=None,
            guess_jitter=0.02) -> Workload:
    U = _pad(Uint, nx, ny, nz)
    Tg = Tint * (1.0 + guess_jitter * rng.uniform(-1.0, 1.0, Tint.shape))
    Tg = _pad(Tg, nx, ny, nz)
    return Workload(name=name, nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, table=table, bc=tuple(bc), U=U,
                    T_guess=Tg, bc_state=bc_state, steps=steps, notes=notes or {})


# ----------------------------------------------------------------------------------------------------------------
# config 1: 1-D two-species shock tube
# ----------------------------------------------------------------------------------------------------------------
def config1_shock_tube(nx: int = 400, axis: int = 0, seed: Optional[int] = None, y_floor: float = 0.0) -> Workload:
    """BASELINE.json configs[0]; shape of the paper's inert shock tube.

    ``axis`` lays the tube along x (0), y (1) or z (2) -- used by direction-consistency tests.  ``y_floor`` > 0 keeps both
    mass fractions inside [y_floor, 1 - y_floor] (the role of zeta in the paper's Eq. 32): without it
    the tanh tails hold cells with Y ~ 1e-16, where the positivity limiter's decision rests on round-off.
    """
    rng = np.random.default_rng(SEED_BASE + 1 if seed is None else seed)
    table = calorically_perfect_table(W=(28.0, 4.0), gamma=(1.4, 5.0 / 3.0), Ru=1.0)
    dx = 1.0 / nx
    x = (np.arange(nx) + 0.5) * dx
    left = x < 0.5
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    YA = 0.5 * (1.0 - np.tanh((x - 0.5) / (2.0 * dx)))
    if y_floor > 0.0:
        YA = np.clip(YA, y_floor, 1.0 - y_floor)
    Y = np.stack([YA, 1.0 - YA])
    rho = rho * (1.0 + 1e-3 * rng.uniform(-1.0, 1.0, nx))
    T = p / (rho * table.mixture_R(Y))
    z = np.zeros(nx)
    Ui = conserved_from_primitive(table, rho, z, z, z, T, Y)          # [Nv, nx]
    dims = [1, 1, 1]
    dims[axis] = nx
    shape = (dims[2], dims[1], dims[0])
    Ui = Ui.reshape((table.n + 4,) + shape)
    Ti = T.reshape(shape)
    d = [1.0, 1.0, 1.0]
    d[axis] = dx
    bc = [BC_TRANSMISSIVE] * 6
    return _finish("config1_shock_tube_1d_2sp", dims[0], dims[1], dims[2], d[0], d[1], d[2], table, bc, Ui, Ti, rng,
                   steps=200)


# ----------------------------------------------------------------------------------------------------------------
# configs 2-4: shock-bubble interaction
# ----------------------------------------------------------------------------------------------------------------
def _rankine_hugoniot(gamma: float, Ma: float, rho0: float, p0: float):
    """PAPER.md:626-630, Eq. 33 (with gamma of the ambient gas)."""
    c0 = np.sqrt(gamma * p0 / rho0)
    rho1 = rho0 * (gamma + 1.0) * Ma ** 2 / (2.0 + (gamma - 1.0) * Ma ** 2)
    u1 = Ma * c0 * (1.0 - rho0 / rho1)
    p1 = p0 * (1.0 + 2.0 * gamma / (gamma + 1.0) * (Ma ** 2 - 1.0))
    return rho1, u1, p1


def _legendre(l: int, x: np.ndarray) -> np.ndarray:
    p0, p1 = np.ones_like(x), x
    if l == 0:
        return p0
    for n in range(1, l):
        p0, p1 = p1, ((2 * n + 1) * x * p1 - n * p0) / (n + 1)
    return p1


def _shock_bubble(name, cfg_index, nx, ny, nz, Lx, Ly, Lz, table, X_amb, X_bub, Ma, x_shock, centre, R0, bc,
                  surface, minors=None, steps=1, seed=None, rng=None) -> Workload:
    """Planar shock + tanh-smoothed bubble interface in mole fraction (Eq. 32-33)."""
    n = table.n
    dx, dy, dz = Lx / nx, Ly / ny, (Lz / nz if nz > 1 else 1.0)
    x = (np.arange(nx) + 0.5) * dx
    y = (np.arange(ny) + 0.5) * dy
    z = (np.arange(nz) + 0.5) * dz if nz > 1 else np.array([centre[2]])
    Z, Yc, X = np.meshgrid(z, y, x, indexing="ij")
    rx, ry, rz = X - centre[0], Yc - centre[1], Z - centre[2]
    r = np.sqrt(rx * rx + ry * ry + rz * rz)
    Rsurf = R0 * (1.0 + surface(rx, ry, rz, r))
    d = r - Rsurf                                             # signed distance (radial) to the perturbed surface
    zeta = 1e-4
    phi = 0.5 * ((1.0 - 2.0 * zeta) * np.tanh(d / (2.0 * dx)) + 1.0)   # X of the ambient gas, Eq. 32

    X_amb = np.asarray(X_amb, dtype=np.float64)
    X_bub = np.asarray(X_bub, dtype=np.float64)
    Xf = X_amb.reshape(n, 1, 1, 1) * phi + X_bub.reshape(n, 1, 1, 1) * (1.0 - phi)
    Yf = table.X_to_Y(Xf)
    if minors is not None:
        idx, y_in, y_out = minors
        ym = np.zeros_like(Yf)
        for q, s in enumerate(idx):
            ym[s] = (1.0 - phi) * y_in[q] + phi * y_out[q]
        Yf = Yf * (1.0 - ym.sum(axis=0)) + ym                 # majors renormalised

    # quiescent gas: rho0 = 1, p0 = 1 in the ambient mixture; Ru was chosen so that this is T0 = 300 K
    Y_amb = Yf[:, 0, 0, -1]                                   # far downstream corner = pure ambient (+ minors)
    p0 = 1.0
    T0 = p0 / (1.0 * table.mixture_R(Y_amb))
    gam = float(table.frozen_gamma(Y_amb, np.float64(T0)))
    rho1, u1, p1 = _rankine_hugoniot(gam, Ma, 1.0, p0)
    T1 = p1 / (rho1 * table.mixture_R(Y_amb))

    post = X < x_shock
    for s in range(n):
        Yf[s] = np.where(post, Y_amb[s], Yf[s])
    p = np.where(post, p1, p0)
    T = np.where(post, T1, T0)
    rho = p / (table.mixture_R(Yf) * T)
    u = np.where(post, u1, 0.0)
    zero = np.zeros_like(u)
    Ui = conserved_from_primitive(table, rho, u, zero, zero, T, Yf)

    bc_state = np.zeros((6, n + 4))
    st = conserved_from_primitive(table, np.float64(rho1), np.float64(u1), 0.0, 0.0, np.float64(T1), Y_amb)
    bc_state[:] = st
    return _finish(name, nx, ny, nz, dx, dy, dz, table, bc, Ui, T, rng, bc_state=bc_state, steps=steps,
                   notes={"Ma": Ma, "gamma_ambient": gam, "T0": float(T0), "post_shock": (rho1, u1, p1)})


def config2_shock_bubble_2d(nx: int = 2048, ny: int = 1024, seed: Optional[int] = None) -> Workload:
    """BASELINE.json configs[1]: 2-D, 3 thermally perfect species, Ma 1.22; reduced sizes keep the set-up."""
    rng = np.random.default_rng(SEED_BASE + 2 if seed is None else seed)
    W = (28.0, 4.0, 146.0)
    table = synthetic_nasa7_table(W, Ru=28.0 / 300.0, rng=rng)
    modes = np.arange(2, 17)
    signs = rng.choice([-1.0, 1.0], modes.size)
    phases = rng.uniform(0.0, 2 * np.pi, modes.size)
    amp = 0.01 * signs / (modes * np.sum(1.0 / modes))       # sum |a_m| = 0.01

    def surface(rx, ry, rz, r):
        ang = np.arctan2(ry, rx)
        out = np.zeros_like(ang)
        for a, m, ph in zip(amp, modes, phases):
            out += a * np.cos(m * ang + ph)
        return out

    bc = (BC_DIRICHLET, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_REFLECTIVE, BC_PERIODIC, BC_PERIODIC)
    return _shock_bubble("config2_shock_bubble_2d_3sp", 2, nx, ny, 1, 2.0, 1.0, 1.0, table, (1, 0, 0), (0, 0.95, 0.05),
                         1.22, 0.3, (0.6, 0.5, 0.0), 0.2, bc, surface, steps=500, rng=rng)


def config3_shock_bubble_3d(n: int = 256, seed: Optional[int] = None) -> Workload:
    """BASELINE.json configs[2]: 3-D, 4 species, Ma 2.83, periodic y/z."""
    rng = np.random.default_rng(SEED_BASE + 3 if seed is None else seed)
    W = (28.0, 32.0, 4.0, 131.3)
    table = synthetic_nasa7_table(W, Ru=28.84 / 300.0, rng=rng)
    nh = 24
    axes = rng.normal(size=(nh, 3))
    axes /= np.linalg.norm(axes, axis=1, keepdims=True)
    coef = rng.normal(size=nh)
    degs = 2 + (np.arange(nh) % 7)                            # l cycling 2..8

    def raw(nxv, nyv, nzv):
        out = np.zeros_like(nxv)
        for a, l, ax in zip(coef, degs, axes):
            out += a * _legendre(int(l), np.clip(nxv * ax[0] + nyv * ax[1] + nzv * ax[2], -1.0, 1.0))
        return out

    probe = rng.normal(size=(4096, 3))                        # resolution-independent normalisation sample
    probe /= np.linalg.norm(probe, axis=1, keepdims=True)
    scale = 0.01 / np.max(np.abs(raw(probe[:, 0], probe[:, 1], probe[:, 2])))

    def surface(rx, ry, rz, r):
        rr = np.maximum(r, 1e-300)
        return scale * raw(rx / rr, ry / rr, rz / rr)

    bc = (BC_DIRICHLET, BC_TRANSMISSIVE, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC, BC_PERIODIC)
    return _shock_bubble("config3_shock_bubble_3d_4sp", 3, n, n, n, 1.0, 1.0, 1.0, table, (0.79, 0.21, 0, 0),
                         (0, 0, 0.37, 0.63), 2.83, 0.15, (0.4, 0.5, 0.5), 0.125, bc, surface, steps=200, rng=rng)


def table10(seed: Optional[int] = None, formation: bool = False, Ru: float = 28.014 / 300.0) -> SpeciesTable:
    """The 10-species table shared by configs 4 and 5 (own seed so that both configs get the same table)."""
    rng = np.random.default_rng(SEED_BASE + 40 if seed is None else seed)
    return synthetic_nasa7_table(W10, Ru=Ru, rng=rng, formation=formation)


def config4_shock_bubble_3d_10sp(nx: int = 512, ny: int = 256, nz: int = 256, seed: Optional[int] = None) -> Workload:
    """BASELINE.json configs[3] -- the configuration the headline metric is quoted on."""
    rng = np.random.default_rng(SEED_BASE + 4 if seed is None else seed)
    table = table10()
    X_amb = np.zeros(10)
    X_amb[9] = 1.0
    X_bub = np.zeros(10)
    X_bub[[0, 1, 8]] = np.array([2.0, 1.0, 7.0]) / 10.0      # 2:1:7 mole mixture of species 1:2:9
    idx = [2, 3, 4, 5, 6, 7]                                  # species 3-8: minor, log-uniform in [1e-8, 1e-4]
    y_in = 10.0 ** rng.uniform(-8.0, -4.0, len(idx))
    y_out = 10.0 ** rng.uniform(-8.0, -4.0, len(idx))
    bc = (BC_DIRICHLET, BC_TRANSMISSIVE, BC_REFLECTIVE, BC_REFLECTIVE, BC_REFLECTIVE, BC_REFLECTIVE)
    return _shock_bubble("config4_shock_bubble_3d_10sp", 4, nx, ny, nz, 2.0, 1.0, 1.0, table, X_amb, X_bub, 2.83, 0.3,
                         (0.6, 0.5, 0.5), 0.15, bc, lambda rx, ry, rz, r: 0.0 * r, minors=(idx, y_in, y_out),
                         steps=100, rng=rng)


# ----------------------------------------------------------------------------------------------------------------
# config 5: random-state stress test
# ----------------------------------------------------------------------------------------------------------------
def _box_filter_periodic(A: np.ndarray) -> np.ndarray:
    """One pass of a periodic 3x3x3 box filter over the last three axes (separable)."""
    for ax in (-1, -2, -3):
        if A.shape[ax] > 1:
            A = (np.roll(A, 1, axis=ax) + A + np.roll(A, -1, axis=ax)) / 3.0
    return A


def config5_random_states(nx: int = 640, ny: int = 384, nz: int = 384, seed: Optional[int] = None,
                          formation: bool = False) -> Workload:
    """BASELINE.json configs[4]: periodic box of smoothed random states, 10 species."""
    rng = np.random.default_rng(SEED_BASE + 5 if seed is None else seed)
    shape = (nz, ny, nx)
    tab1 = table10(formation=formation, Ru=1.0)
    rho = 10.0 ** rng.uniform(-1.0, 1.0, shape)
    p = 10.0 ** rng.uniform(-1.0, 2.0, shape)
    Y = rng.standard_gamma(0.5, (10,) + shape)                # Dirichlet(0.5 * 1) = normalised Gamma(0.5) draws
    Y /= Y.sum(axis=0)
    Wbar = 1.0 / np.tensordot(1.0 / tab1.W, Y, axes=(0, 0))
    t_unit = p * Wbar / rho                                   # T * Ru
    Ru = float(np.median(t_unit) / 1000.0)                    # median T = 1000 K before filtering
    table = table10(formation=formation, Ru=Ru)
    T = t_unit / Ru
    c = np.sqrt(table.frozen_gamma(Y, T) * table.mixture_R(Y) * T)
    u = rng.uniform(-2.0, 2.0, shape) * c
    v = rng.uniform(-2.0, 2.0, shape) * c if ny > 1 else np.zeros(shape)
    w = rng.uniform(-2.0, 2.0, shape) * c if nz > 1 else np.zeros(shape)
    Ui = conserved_from_primitive(table, rho, u, v, w, T, Y)
    del Y, u, v, w, c
    for _ in range(3):
        for k in range(Ui.shape[0]):
            Ui[k] = _box_filter_periodic(Ui[k])
    d = 1.0 / 384.0
    bc = (BC_PERIODIC,) * 6
    # the guess: the pre-filter T is no longer the state's T; a flat 1000 K +-2% guess keeps Newton at 3-5 steps
    Tg = np.full(shape, 1000.0)
    return _finish("config5_random_10sp", nx, ny, nz, d, d if ny > 1 else 1.0, d if nz > 1 else 1.0, table, bc, Ui, Tg,
                   rng, steps=1, notes={"Ru": Ru})


def config5_random_states_device(nx: int = 640, ny: int = 384, nz: int = 384, device="cuda:0", seed: Optional[int] = None):
    """BASELINE.json configs[4] at its stated size, generated ON THE DEVICE with torch (94 M cells x 14 variables take
    minutes with numpy on the host, seconds here).  Same recipe as ``config5_random_states`` -- log-uniform rho and p,
    Dirichlet(0.5) mass fractions, velocities in +-2 local sound speeds, Ru such that the median T is 1000 K, three
    passes of a periodic 3x3x3 box filter on the conserved variables -- with torch's seeded CUDA generator, so the
    numbers differ from the numpy variant's.  Returns a ``Workload`` whose ``U`` / ``T_guess`` are padded torch tensors
    on ``device`` (ghosts unfilled: the path fills them); the oracle side of the parity test receives a sub-block copied
    to the host (``periodic_subblock_arrays``)."""
    import torch

    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(SEED_BASE + 5 if seed is None else seed)
    shape = (nz, ny, nx)
    f64 = dict(dtype=torch.float64, device=dev)

    def uniform(lo, hi):
        return lo + (hi - lo) * torch.rand(shape, generator=gen, **f64)

    tab1 = table10(Ru=1.0)
    rho = 10.0 ** uniform(-1.0, 1.0)
    p = 10.0 ** uniform(-1.0, 2.0)
    Y = torch._standard_gamma(torch.full((10,) + shape, 0.5, **f64), generator=gen)   # Dirichlet = normalised Gamma
    Y /= Y.sum(dim=0, keepdim=True)
    Wt = torch.tensor(tab1.W, **f64).reshape(10, 1, 1, 1)
    Wbar = 1.0 / (Y / Wt).sum(dim=0)
    t_unit = p * Wbar / rho                                   # T * Ru
    Ru = float(torch.median(t_unit.reshape(-1)).item() / 1000.0)
    table = table10(Ru=Ru)
    T = t_unit / Ru
    del t_unit, p, Wbar
    # forward evaluation of the table (input generation only): cp/R, h/R per species with the constant-cp continuation
    a = torch.tensor(table.nasa7, **f64)
    Rs = torch.tensor(table.Rs, **f64)
    Tc = T.clamp(table.Tlo, table.Thi)
    cp_mix = torch.zeros(shape, **f64)
    h_mix = torch.zeros(shape, **f64)
    R_mix = torch.zeros(shape, **f64)
    for s_ in range(10):
        cpR = a[s_, 0] + Tc * (a[s_, 1] + Tc * (a[s_, 2] + Tc * (a[s_, 3] + Tc * a[s_, 4])))
        hR = Tc * (a[s_, 0] + Tc * (a[s_, 1] / 2 + Tc * (a[s_, 2] / 3 + Tc * (a[s_, 3] / 4 + Tc * a[s_, 4] / 5)))) + a[s_, 5]
        hR = hR + cpR * (T - Tc)
        cp_mix += Y[s_] * Rs[s_] * cpR
        h_mix += Y[s_] * Rs[s_] * hR
        R_mix += Y[s_] * Rs[s_]
    del Tc, cpR, hR
    c = torch.sqrt(cp_mix / (cp_mix - R_mix) * R_mix * T)
    e = h_mix - R_mix * T
    del cp_mix, h_mix, R_mix, T
    U = torch.empty((14,) + shape, **f64)
    U[0] = rho
    k2 = torch.zeros(shape, **f64)
    for q, n_ in enumerate((nx, ny, nz)):
        vel = uniform(-2.0, 2.0) * c if n_ > 1 else torch.zeros(shape, **f64)
        U[1 + q] = rho * vel
        k2 += vel * vel
    U[4] = rho * (e + 0.5 * k2)
    for s_ in range(9):
        U[5 + s_] = rho * Y[s_]
    del Y, e, k2, vel, c, rho
    for _ in range(3):
        for k in range(14):
            A = U[k]
            for ax in (-1, -2, -3):
                if A.shape[ax] > 1:
                    A = (torch.roll(A, 1, dims=ax) + A + torch.roll(A, -1, dims=ax)) / 3.0
            U[k] = A
    gx, gy, gz = (NG if n_ > 1 else 0 for n_ in (nx, ny, nz))
    Up = torch.zeros((14, nz + 2 * gz, ny + 2 * gy, nx + 2 * gx), **f64)
    Up[:, gz:gz + nz, gy:gy + ny, gx:gx + nx] = U
    del U
    Tg = torch.full(Up.shape[1:], 1000.0, **f64) * (1.0 + 0.02 * (2.0 * torch.rand(Up.shape[1:], generator=gen, **f64) - 1.0))
    d = 1.0 / 384.0
    return Workload(name="config5_random_10sp_device", nx=nx, ny=ny, nz=nz, dx=d, dy=d if ny > 1 else 1.0,
                    dz=d if nz > 1 else 1.0, table=table, bc=(BC_PERIODIC,) * 6, U=Up, T_guess=Tg, steps=1,
                    notes={"Ru": Ru})


def periodic_subblock_arrays(wl: Workload, Ui: np.ndarray, Ti: np.ndarray) -> Workload:
    """A stand-alone transmissive workload from an already cut interior block Ui [Nv, n, n, n], Ti [n, n, n]."""
    n = Ui.shape[-1]
    return Workload(name=wl.name + "_subblock", nx=n, ny=n, nz=n, dx=wl.dx, dy=wl.dy, dz=wl.dz, table=wl.table,
                    bc=(BC_TRANSMISSIVE,) * 6, U=_pad(np.ascontiguousarray(Ui), n, n, n),
                    T_guess=_pad(np.ascontiguousarray(Ti), n, n, n), steps=1)


def periodic_subblock(wl: Workload, origin: Tuple[int, int, int], size: int, margin: int) -> Workload:
    """Cut the (size + 2 margin)^3 block around ``origin`` (interior index of the inner block's first cell, x y z)
    out of a periodic workload, with periodic wrap, as a stand-alone workload with transmissive ends.  After one
    RK3 step the inner size^3 cells depend only on data inside the cut when margin >= 9 (3 stages x 3 cells)."""
    n = size + 2 * margin
    ix = (np.arange(n) + origin[0] - margin) % wl.nx
    iy = (np.arange(n) + origin[1] - margin) % wl.ny
    iz = (np.arange(n) + origin[2] - margin) % wl.nz
    Ui = wl.interior(wl.U)[:, iz][:, :, iy][:, :, :, ix]
    Ti = wl.interior(wl.T_guess)[iz][:, iy][:, :, ix]
    bc = (BC_TRANSMISSIVE,) * 6
    sub = Workload(name=wl.name + "_subblock", nx=n, ny=n, nz=n, dx=wl.dx, dy=wl.dy, dz=wl.dz, table=wl.table, bc=bc,
                   U=_pad(np.ascontiguousarray(Ui), n, n, n), T_guess=_pad(np.ascontiguousarray(Ti), n, n, n),
                   steps=1, notes={"origin": origin, "size": size, "margin": margin})
    return sub


# ----------------------------------------------------------------------------------------------------------------
# small generic states used by tests
# ----------------------------------------------------------------------------------------------------------------
def random_smooth_box(nx: int, ny: int, nz: int, nspecies: int, seed: int, bc=(BC_PERIODIC,) * 6,
                      formation: bool = True, amplitude: float = 0.3) -> Workload:
    """Smooth, strictly positive random periodic state on a small box (low-order Fourier modes), N species with a
    formation-enthalpy table -- the general-purpose small parity / invariance input."""
    rng = np.random.default_rng(seed)
    W = rng.uniform(2.0, 140.0, nspecies)
    table = synthetic_nasa7_table(W, Ru=float(np.mean(W)) / 300.0, rng=rng, formation=formation)
    shape = (nz, ny, nx)
    zc = (np.arange(nz) + 0.5) / nz
    yc = (np.arange(ny) + 0.5) / ny
    xc = (np.arange(nx) + 0.5) / nx
    Z, Yc, X = np.meshgrid(zc, yc, xc, indexing="ij")

    def wave():
        out = np.zeros(shape)
        for _ in range(4):
            kx, ky, kz = rng.integers(0, 3, 3)
            if nx == 1:
                kx = 0
            if ny == 1:
                ky = 0
            if nz == 1:
                kz = 0
            out += rng.uniform(-1, 1) * np.sin(2 * np.pi * (kx * X + ky * Yc + kz * Z) + rng.uniform(0, 2 * np.pi))
        return out / 4.0

    rho = np.exp(amplitude * 2.0 * wave())
    T = 900.0 * np.exp(amplitude * 2.0 * wave())
    Yr = np.stack([np.exp(2.0 * wave()) for _ in range(nspecies)])
    Yr /= Yr.sum(axis=0)
    c = np.sqrt(table.frozen_gamma(Yr, T) * table.mixture_R(Yr) * T)
    u = 0.8 * c * wave() * 2
    v = 0.8 * c * wave() * 2 if ny > 1 else np.zeros(shape)
    w = 0.8 * c * wave() * 2 if nz > 1 else np.zeros(shape)
    Ui = conserved_from_primitive(table, rho, u, v, w, T, Yr)
    d = (1.0 / nx, 1.0 / ny if ny > 1 else 1.0, 1.0 / nz if nz > 1 else 1.0)
    bc_state = None
    if BC_DIRICHLET in bc:
        bc_state = np.tile(Ui.reshape(nspecies + 4, -1)[:, :1].T, (6, 1))
    return _finish(f"random_smooth_{nx}x{ny}x{nz}_{nspecies}sp", nx, ny, nz, d[0], d[1], d[2], table, bc, Ui, T, rng,
                   bc_state=bc_state)


def rough_box(nx: int, ny: int, nz: int, nspecies: int = 4, seed: int = 3, bc=(BC_PERIODIC,) * 6) -> Workload:
    """Cell-to-cell random composition (species 1 absent from 30 % of the cells), density and temperature with moderate
    velocities: the unlimited scheme undershoots Y by several per cent here, so this is the input on which the
    positivity-preserving flux blending is active at many faces."""
    rng = np.random.default_rng(seed)
    table = synthetic_nasa7_table(rng.uniform(2, 60, nspecies), Ru=0.1, rng=rng, formation=True)
    shape = (nz, ny, nx)
    Y = rng.standard_gamma(0.3, (nspecies,) + shape)
    Y /= Y.sum(axis=0)
    Y[0][rng.uniform(size=shape) < 0.3] = 0.0
    Y /= Y.sum(axis=0)
    rho = 10 ** rng.uniform(-0.5, 0.5, shape)
    T = 10 ** rng.uniform(2.5, 3.2, shape)
    c = np.sqrt(table.frozen_gamma(Y, T) * table.mixture_R(Y) * T)
    u = [rng.uniform(-0.5, 0.5, shape) * c if m > 1 else np.zeros(shape) for m in (nx, ny, nz)]
    Ui = conserved_from_primitive(table, rho, u[0], u[1], u[2], T, Y)
    d = [1.0 / m if m > 1 else 1.0 for m in (nx, ny, nz)]
    bc_state = np.tile(Ui.reshape(nspecies + 4, -1)[:, :1].T, (6, 1)) if BC_DIRICHLET in bc else None
    return _finish(f"rough_{nx}x{ny}x{nz}_{nspecies}sp", nx, ny, nz, d[0], d[1], d[2], table, bc, Ui, T, rng,
                   bc_state=bc_state)


# ----------------------------------------------------------------------------------------------------------------
# transport fits for the viscous / diffusive terms (Eq. 29)
# ----------------------------------------------------------------------------------------------------------------
@dataclass
class TransportFits:
    """ln eta = a_0 + a_1 ln T + a_2 (ln T)^2 + a_3 (ln T)^3 for mu_s [N,4], kappa_s [N,4] and the binary D_st at p_ref
    [N,N,4] (symmetric).  The paper fits these to kinetic-theory values of real species (collision-integral tables,
    PAPER.md:155-178), which are not in this container; these are seeded synthetic fits of the same SHAPE: power laws
    mu ~ T^0.7, kappa ~ T^0.75, D ~ T^1.7 with seeded quadratic / cubic corrections in ln T."""

    mu: np.ndarray
    kappa: np.ndarray
    D: np.ndarray
    p_ref: float


def synthetic_transport(table: SpeciesTable, seed: int, mu0: float = 2e-3, T0: float = 300.0, p_ref: float = 1.0,
                        rho0: float = 1.0) -> TransportFits:
    """mu0: viscosity scale at T0 in the workload's units (rho ~ 1, p ~ 1, lengths ~ 1: mu0 = 2e-3 puts the cell Reynolds
    number of the test boxes at O(10)); kappa_s = mu_s cp_s(T0) / Pr_s, D_st = mu / (rho0 Sc_st) at (T0, p_ref)."""
    rng = np.random.default_rng(seed)
    n = table.n
    lnT0 = np.log(T0)

    def fit(val0, expo):
        a = np.zeros(4)
        a[2], a[3] = rng.uniform(-0.02, 0.02), rng.uniform(-0.002, 0.002)
        a[1] = expo - 2 * a[2] * lnT0 - 3 * a[3] * lnT0 ** 2     # d ln eta / d ln T = expo at T0
        a[0] = np.log(val0) - (a[1] * lnT0 + a[2] * lnT0 ** 2 + a[3] * lnT0 ** 3)
        return a

    mus = mu0 * rng.uniform(0.5, 2.0, n)
    cp0 = table.Rs * table.cp_over_R(np.float64(min(max(T0, table.Tlo), table.Thi)))
    mu = np.stack([fit(mus[s], 0.7 + rng.uniform(-0.05, 0.05)) for s in range(n)])
    kappa = np.stack([fit(mus[s] * cp0[s] / rng.uniform(0.65, 0.8), 0.75 + rng.uniform(-0.05, 0.05)) for s in range(n)])
    D = np.zeros((n, n, 4))
    for s in range(n):
        for t in range(s + 1, n):
            D[s, t] = D[t, s] = fit(0.5 * (mus[s] + mus[t]) / (rho0 * rng.uniform(0.6, 1.1)), 1.7 + rng.uniform(-0.05, 0.05))
    return TransportFits(mu=mu, kappa=kappa, D=D, p_ref=float(p_ref))


# ----------------------------------------------------------------------------------------------------------------
# a seeded synthetic reaction mechanism (Eq. 8-12)
# ----------------------------------------------------------------------------------------------------------------
@dataclass
class Mechanism:
    nu_r: np.ndarray          # [NR, N] reactant coefficients nu'
    nu_p: np.ndarray          # [NR, N] product coefficients nu''
    A: np.ndarray             # [NR] Arrhenius pre-exponential factor, temperature exponent, activation energy (Eq. 11)
    B: np.ndarray
    E: np.ndarray
    third: np.ndarray         # [NR] 1: third-body reaction
    eff: np.ndarray           # [NR, N] third-body efficiencies
    p_atm: float              # the standard pressure of Eq. 12 in the workload's units


def reacting_table(seed: int = 0, Ru: float = 8.0):
    """Eight species built from two elements of mass 1.008 and 16.0 -- compositions (2,0) (0,2) (2,1) (1,0) (0,1) (1,1)
    (1,2) (2,2) -- plus an inert ninth of mass 28.0: molar masses that conserve mass in every element-balanced reaction.
    Seeded synthetic NASA-7 coefficients with formation-enthalpy and entropy constants (a6, a7).  -> (table, comp [9, 2])"""
    comp = np.array([(2, 0), (0, 2), (2, 1), (1, 0), (0, 1), (1, 1), (1, 2), (2, 2), (0, 0)])
    W = comp @ np.array([1.008, 16.0])
    W[8] = 28.0
    rng = np.random.default_rng(SEED_BASE + 900 + seed)
    table = synthetic_nasa7_table(W, Ru=Ru, rng=rng, formation=False)
    table.nasa7[:, 5] += rng.uniform(-1500.0, 1500.0, 9) * (np.arange(9) != 8)   # formation enthalpies / R (K)
    # entropy constants: S_s/R_s = O(1) around 1000 K, so that the equilibrium constants of Eq. 12 are moderate
    table.nasa7[:, 6] = -table.nasa7[:, 0] * np.log(1000.0) + rng.uniform(-1.0, 1.0, 9)
    return table, comp


def synthetic_mechanism(table: SpeciesTable, comp: np.ndarray, n_reactions: int, seed: int, rate: float = 50.0,
                        p_atm: Optional[float] = None, T_act: float = 1500.0) -> Mechanism:
    """Element-balanced reversible reactions drawn at random from ALL the balanced ones of the forms A + B <=> C + D and
    A + B (+ M) <=> C (+ M) among the reactive species (enumerated from the composition table -- no real mechanism is
    written out), with seeded Arrhenius parameters: A such that the forward rate is ~ `rate` per unit time at
    concentration ~ 0.05 and 1000 K, B in [-1, 1], E/Ru in [0, T_act] K; a third of the three-body ones get seeded
    third-body efficiencies in [0.5, 3]."""
    rng = np.random.default_rng(SEED_BASE + 950 + seed)
    n = table.n
    if p_atm is None:
        p_atm = table.Ru * 1000.0 * 0.05      # p0/(Ru T) = the typical concentration at 1000 K
    reactive = [s for s in range(n) if comp[s].sum() > 0]
    cands = []
    for i, a in enumerate(reactive):
        for b in reactive[i:]:
            lhs = comp[a] + comp[b]
            for c in reactive:                                    # A + B (+M) <=> C (+M)
                if c not in (a, b) and np.array_equal(comp[c], lhs):
                    cands.append(((a, b), (c,), 1))
            for j, c in enumerate(reactive):                      # A + B <=> C + D
                for d_ in reactive[j:]:
                    if {a, b} != {c, d_} and (a, b) < (c, d_) and np.array_equal(comp[c] + comp[d_], lhs):
                        cands.append(((a, b), (c, d_), 0))
    pick = rng.permutation(len(cands))[:n_reactions]
    nr = len(pick)
    nu_r, nu_p = np.zeros((nr, n), dtype=np.int64), np.zeros((nr, n), dtype=np.int64)
    third, eff = np.zeros(nr, dtype=np.int64), np.ones((nr, n))
    A, B, E = np.zeros(nr), rng.uniform(-1.0, 1.0, nr), table.Ru * rng.uniform(0.0, T_act, nr)
    for r, q in enumerate(pick):
        lhs, rhs, tb = cands[q]
        for s in lhs:
            nu_r[r, s] += 1
        for s in rhs:
            nu_p[r, s] += 1
        third[r] = tb
        if tb:
            eff[r] = rng.uniform(0.5, 3.0, n)
        A[r] = rate / 0.05 / (0.5 if tb else 1.0) * rng.uniform(0.3, 3.0) / (1000.0 ** B[r] * np.exp(-E[r] / (table.Ru * 1000.0)))
    return Mechanism(nu_r=nu_r, nu_p=nu_p, A=A, B=B, E=E, third=third, eff=eff, p_atm=float(p_atm))


def reacting_box(nx: int, ny: int, nz: int, seed: int, bc=(BC_PERIODIC,) * 6, smooth: bool = False) -> Workload:
    """random (or smooth periodic) composition / temperature / density field on the nine-species reacting table: the input
    of the reaction-step tests and of bench.py --workload react"""
    table, _ = reacting_table()
    rng = np.random.default_rng(seed)
    shape = (nx, ny, nz)
    shp = (nz, ny, nx)
    if smooth:
        z, y, x = np.meshgrid((np.arange(nz) + 0.5) / nz, (np.arange(ny) + 0.5) / ny, (np.arange(nx) + 0.5) / nx, indexing="ij")
        ph = lambda: np.sin(2 * np.pi * (x * (nx > 1) + y * (ny > 1) + z * (nz > 1)) + rng.uniform(0, 6))   # noqa: E731
        Y = np.stack([np.exp(0.8 * ph()) for _ in range(9)])
        Y /= Y.sum(axis=0)
        T = 1100.0 + 250.0 * ph()
        rho = 1.0 + 0.2 * ph()
        c = np.sqrt(table.frozen_gamma(Y, T) * table.mixture_R(Y) * T)
        vel = [0.3 * c * ph() if m > 1 else np.zeros(shp) for m in shape]
    else:
        Y = rng.dirichlet(0.7 * np.ones(9), size=shp).transpose(3, 0, 1, 2)
        Y[3][rng.uniform(size=shp) < 0.2] = 0.0                  # a species absent from a fifth of the cells
        Y /= Y.sum(axis=0)
        T = rng.uniform(700, 2200, shp)
        rho = 10 ** rng.uniform(-0.4, 0.4, shp)
        vel = [rng.normal(size=shp) * 30 if m > 1 else np.zeros(shp) for m in shape]
    Ui = conserved_from_primitive(table, rho, vel[0], vel[1], vel[2], T, Y)
    d = [1.0 / m if m > 1 else 1.0 for m in shape]
    return _finish("reacting_box", nx, ny, nz, d[0], d[1], d[2], table, bc, Ui, T, rng)
