"""Test-side helpers: independent closed forms and textbook routines the oracle is pinned against."""
from __future__ import annotations

import numpy as np

from paper_2403_05910_b200 import workloads as wl


def make_oracle(oracle_mod, w, **kw):
    return oracle_mod.Oracle.from_workload(w, **kw)


def rel_err_per_var(a: np.ndarray, b: np.ndarray, scale=None) -> np.ndarray:
    """Reading R14: per variable v, max|a_v - b_v| / max(max|b_v|, tiny); a, b shaped [Nv, ...]."""
    nv = a.shape[0]
    a2, b2 = a.reshape(nv, -1), b.reshape(nv, -1)
    num = np.abs(a2 - b2).max(axis=1)
    den = np.abs(b2).max(axis=1) if scale is None else np.asarray(scale, dtype=np.float64)
    return num / np.maximum(den, 1e-300)


def state_scales(U: np.ndarray, c_max: float) -> np.ndarray:
    """R14 scales for conserved variables: momentum components use max|rho|*c so that an identically zero
    velocity component does not divide by zero."""
    nv = U.shape[0]
    s = np.abs(U.reshape(nv, -1)).max(axis=1)
    s[1:4] = np.abs(U[0]).max() * c_max
    return s


# ---------------------------------------------------------------------------------------------------------------
# exact Riemann solution for a calorically perfect gas (textbook: two-rarefaction/shock pressure function, Newton)
# ---------------------------------------------------------------------------------------------------------------
def exact_riemann(rhoL, uL, pL, rhoR, uR, pR, gamma, xi):
    """Sample the exact solution at similarity coordinates xi = (x - x0)/t. Returns rho, u, p arrays."""
    g = gamma
    cL, cR = np.sqrt(g * pL / rhoL), np.sqrt(g * pR / rhoR)

    def fK(p, rhoK, pK, cK):
        if p > pK:  # shock
            A, B = 2.0 / ((g + 1) * rhoK), (g - 1) / (g + 1) * pK
            f = (p - pK) * np.sqrt(A / (p + B))
            df = np.sqrt(A / (p + B)) * (1 - 0.5 * (p - pK) / (p + B))
        else:  # rarefaction
            f = 2 * cK / (g - 1) * ((p / pK) ** ((g - 1) / (2 * g)) - 1)
            df = 1.0 / (rhoK * cK) * (p / pK) ** (-(g + 1) / (2 * g))
        return f, df

    p = 0.5 * (pL + pR)
    for _ in range(100):
        fl, dfl = fK(p, rhoL, pL, cL)
        fr, dfr = fK(p, rhoR, pR, cR)
        dp = (fl + fr + uR - uL) / (dfl + dfr)
        p = max(p - dp, 1e-14)
        if abs(dp) < 1e-15 * p:
            break
    pstar = p
    ustar = 0.5 * (uL + uR) + 0.5 * (fK(p, rhoR, pR, cR)[0] - fK(p, rhoL, pL, cL)[0])

    rho, u, pp = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    for q, s in enumerate(xi):
        if s <= ustar:  # left of contact
            if pstar > pL:
                SL = uL - cL * np.sqrt((g + 1) / (2 * g) * pstar / pL + (g - 1) / (2 * g))
                if s < SL:
                    r, v, pr = rhoL, uL, pL
                else:
                    r = rhoL * ((pstar / pL + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * pstar / pL + 1))
                    v, pr = ustar, pstar
            else:
                SHL = uL - cL
                cs = cL * (pstar / pL) ** ((g - 1) / (2 * g))
                STL = ustar - cs
                if s < SHL:
                    r, v, pr = rhoL, uL, pL
                elif s > STL:
                    r, v, pr = rhoL * (pstar / pL) ** (1 / g), ustar, pstar
                else:
                    v = 2 / (g + 1) * (cL + (g - 1) / 2 * uL + s)
                    cc = 2 / (g + 1) * (cL + (g - 1) / 2 * (uL - s))
                    r = rhoL * (cc / cL) ** (2 / (g - 1))
                    pr = pL * (cc / cL) ** (2 * g / (g - 1))
        else:
            if pstar > pR:
                SR = uR + cR * np.sqrt((g + 1) / (2 * g) * pstar / pR + (g - 1) / (2 * g))
                if s > SR:
                    r, v, pr = rhoR, uR, pR
                else:
                    r = rhoR * ((pstar / pR + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * pstar / pR + 1))
                    v, pr = ustar, pstar
            else:
                SHR = uR + cR
                cs = cR * (pstar / pR) ** ((g - 1) / (2 * g))
                STR = ustar + cs
                if s > SHR:
                    r, v, pr = rhoR, uR, pR
                elif s < STR:
                    r, v, pr = rhoR * (pstar / pR) ** (1 / g), ustar, pstar
                else:
                    v = 2 / (g + 1) * (-cR + (g - 1) / 2 * uR + s)
                    cc = 2 / (g + 1) * (cR - (g - 1) / 2 * (uR - s))
                    r = rhoR * (cc / cR) ** (2 / (g - 1))
                    pr = pR * (cc / cR) ** (2 * g / (g - 1))
        rho[q], u[q], pp[q] = r, v, pr
    return rho, u, pp, pstar, ustar


def single_species_workload(nx, rho, u, p, gamma=1.4, bc=(wl.BC_PERIODIC,) * 6, ny=1, nz=1, axis=0):
    """N = 1 calorically perfect gas with Ru = W = 1; rho, u, p arrays of the interior shape (nz, ny, nx)."""
    table = wl.calorically_perfect_table(W=(1.0,), gamma=(gamma,), Ru=1.0)
    rho = np.asarray(rho, dtype=np.float64)
    T = p / rho
    Y = np.ones((1,) + rho.shape)
    vel = [np.zeros_like(rho)] * 3
    vel[axis] = u
    U = wl.conserved_from_primitive(table, rho, vel[0], vel[1], vel[2], T, Y)
    dims = rho.shape[::-1]
    d = [1.0 / n if n > 1 else 1.0 for n in dims]
    rng = np.random.default_rng(7)
    return wl._finish("single_species", dims[0], dims[1], dims[2], d[0], d[1], d[2], table, bc, U, T, rng,
                      guess_jitter=0.0)
