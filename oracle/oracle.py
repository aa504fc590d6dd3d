"""ctypes marshalling for oracle/xf_oracle.c (no arithmetic of the method here).  TEST INFRASTRUCTURE ONLY."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path
from typing import Optional

import numpy as np

_HERE = Path(__file__).resolve().parent
_SO = _HERE / "libxf_oracle.so"
MAXN = 16
MAXNV = MAXN + 4


class OConfig(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
        ("N", C.c_int), ("Ru", C.c_double),
        ("W", C.c_double * MAXN), ("a", (C.c_double * 7) * MAXN),
        ("Tlo", C.c_double), ("Thi", C.c_double),
        ("bc", C.c_int * 6), ("bc_state", (C.c_double * MAXNV) * 6),
        ("rtol", C.c_double), ("maxit", C.c_int), ("ideal_weights", C.c_int), ("viscosity", C.c_int),
        ("lam_glob", (C.c_double * 3) * 3), ("recon", C.c_int), ("positivity", C.c_int), ("pp_dt", C.c_double),
    ]


class OTransport(C.Structure):
    _fields_ = [("mu", (C.c_double * 4) * MAXN), ("kappa", (C.c_double * 4) * MAXN),
                ("D", ((C.c_double * 4) * MAXN) * MAXN), ("p_ref", C.c_double)]


def make_transport(tr) -> OTransport:
    """tr: an object with mu[N,4], kappa[N,4], D[N,N,4], p_ref (workloads.TransportFits)."""
    o = OTransport()
    n = tr.mu.shape[0]
    for s in range(n):
        for q in range(4):
            o.mu[s][q] = tr.mu[s, q]
            o.kappa[s][q] = tr.kappa[s, q]
            for t in range(n):
                o.D[s][t][q] = tr.D[s, t, q]
    o.p_ref = float(tr.p_ref)
    return o


MAXR = 64


class OMechanism(C.Structure):
    _fields_ = [("NR", C.c_int), ("nu_r", (C.c_int * MAXN) * MAXR), ("nu_p", (C.c_int * MAXN) * MAXR),
                ("A", C.c_double * MAXR), ("B", C.c_double * MAXR), ("E", C.c_double * MAXR),
                ("third", C.c_int * MAXR), ("eff", (C.c_double * MAXN) * MAXR), ("p_atm", C.c_double)]


def make_mechanism(m) -> OMechanism:
    """m: workloads.Mechanism (nu_r, nu_p [NR,N] int, A, B, E [NR], third [NR], eff [NR,N], p_atm)"""
    o = OMechanism()
    nr, n = m.nu_r.shape
    assert nr <= MAXR
    o.NR = nr
    for r in range(nr):
        o.A[r], o.B[r], o.E[r], o.third[r] = float(m.A[r]), float(m.B[r]), float(m.E[r]), int(m.third[r])
        for s in range(n):
            o.nu_r[r][s], o.nu_p[r][s], o.eff[r][s] = int(m.nu_r[r, s]), int(m.nu_p[r, s]), float(m.eff[r, s])
    o.p_atm = float(m.p_atm)
    return o


class OPrim(C.Structure):
    _fields_ = [
        ("rho", C.c_double), ("vel", C.c_double * 3), ("Y", C.c_double * MAXN), ("e", C.c_double),
        ("T", C.c_double), ("p", C.c_double), ("Rbar", C.c_double), ("Cv", C.c_double), ("Gamma", C.c_double),
        ("c", C.c_double), ("H", C.c_double), ("chi", C.c_double * MAXN), ("iters", C.c_int), ("status", C.c_int),
    ]


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (plain C, no fast-math, no FMA contraction, OpenMP on outer loops)."""
    src = _HERE / "xf_oracle.c"
    hdr = _HERE / "xf_oracle.h"
    if not force and _SO.exists() and _SO.stat().st_mtime >= max(src.stat().st_mtime, hdr.stat().st_mtime):
        return _SO
    tmp = _SO.with_suffix(f".so.tmp{os.getpid()}")
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall",
           "-o", str(tmp), str(src), "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _SO)
    return _SO


_lib = None
os.environ.setdefault("OMP_WAIT_POLICY", "passive")  # idle oracle threads must not spin against the tests


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_SO))
        dp = C.POINTER(C.c_double)
        cp = C.POINTER(OConfig)
        pp = C.POINTER(OPrim)
        L.xo_padded_cells.restype = C.c_long
        L.xo_padded_cells.argtypes = [cp]
        L.xo_species_thermo.argtypes = [cp, C.c_int, C.c_double, dp, dp, dp]
        L.xo_species_thermo.restype = None
        L.xo_mixture.argtypes = [cp, dp, C.c_double, dp, dp, dp]
        L.xo_mixture.restype = None
        L.xo_cell_primitives.argtypes = [cp, dp, C.c_double, pp]
        L.xo_cell_primitives.restype = None
        L.xo_primitives.argtypes = [cp, dp, dp, dp, dp, dp]
        L.xo_phys_flux.argtypes = [cp, dp, pp, C.c_int, dp]
        L.xo_phys_flux.restype = None
        L.xo_eigensystem.argtypes = [cp, pp, pp, C.c_int, dp, dp, dp]
        L.xo_weno5.argtypes = [dp, C.c_int]
        L.xo_weno5.restype = C.c_double
        L.xo_wenocu6.argtypes = [dp, C.c_int, dp, dp]
        L.xo_wenocu6.restype = C.c_double
        L.xo_weno7.argtypes = [dp, C.c_int, dp, dp]
        L.xo_weno7.restype = C.c_double
        L.xo_stencil_cells.argtypes = [cp]
        L.xo_positivity_blend.argtypes = [cp, C.c_int, dp, pp, dp, pp, C.c_double, dp]
        L.xo_positivity_blend.restype = C.c_double
        L.xo_face_flux.argtypes = [cp, C.c_int, dp, pp, dp]
        L.xo_fill_ghosts.argtypes = [cp, dp]
        L.xo_fill_ghosts.restype = None
        L.xo_rhs.argtypes = [cp, dp, dp, dp]
        L.xo_rhs_nofill.argtypes = [cp, dp, dp, dp]
        L.xo_rhs_cells.argtypes = [cp, dp, dp, C.c_long, C.POINTER(C.c_long), dp]
        L.xo_rk3_step.argtypes = [cp, dp, dp, C.c_double]
        L.xo_max_wavespeed.argtypes = [cp, dp, dp, C.POINTER(C.c_int)]
        L.xo_max_wavespeed.restype = C.c_double
        mp = C.POINTER(OMechanism)
        L.xo_qss_alpha.argtypes = [C.c_double]
        L.xo_qss_alpha.restype = C.c_double
        L.xo_reaction_rates.argtypes = [cp, mp, C.c_double, dp, C.c_double, dp, dp]
        L.xo_reaction_rates.restype = None
        L.xo_react_cell.argtypes = [cp, mp, dp, dp, C.c_double, C.c_int, C.c_int]
        L.xo_react.argtypes = [cp, mp, dp, dp, C.c_double, C.c_int, C.c_int]
        tp = C.POINTER(OTransport)
        L.xo_transport_cell.argtypes = [cp, tp, C.c_double, dp, C.c_double, dp, dp, dp, dp]
        L.xo_transport_cell.restype = None
        L.xo_viscous_face_flux.argtypes = [cp, tp, dp, dp, C.c_long, C.c_int, dp, dp]
        L.xo_viscous_face_flux.restype = None
        L.xo_viscous_rhs.argtypes = [cp, tp, dp, dp, dp]
        L.xo_rhs_ns.argtypes = [cp, tp, dp, dp, dp]
        L.xo_rk3_step_ns.argtypes = [cp, tp, dp, dp, C.c_double]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def wenocu6(v, ideal: bool = False):
    """-> (value at +1/2, [beta0, beta1, beta2, beta6], [four normalised weights])"""
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.shape == (6,)
    beta, w = np.zeros(4), np.zeros(4)
    val = float(lib().xo_wenocu6(_dp(v), int(ideal), _dp(beta), _dp(w)))
    return val, beta, w


def weno7(v, ideal: bool = False):
    """-> (value at +1/2, [beta0..beta3], [four normalised weights]); v = v_{-3}..v_{+3}"""
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.shape == (7,)
    beta, w = np.zeros(4), np.zeros(4)
    val = float(lib().xo_weno7(_dp(v), int(ideal), _dp(beta), _dp(w)))
    return val, beta, w


def weno5(v, ideal: bool = False) -> float:
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert v.shape == (5,)
    return float(lib().xo_weno5(_dp(v), int(ideal)))


class Oracle:
    """One oracle context: grid, species table and boundary data (mirrors xf_config of include/xf.h)."""

    def __init__(self, nx, ny, nz, dx, dy, dz, W, nasa7, Ru, Tlo, Thi, bc=(0,) * 6, bc_state=None,
                 rtol: float = 1e-13, maxit: int = 50, ideal_weights: bool = False, viscosity: int = 0, recon: int = 0,
                 positivity: bool = False, pp_dt: float = 0.0, ng: Optional[int] = None):
        W = np.asarray(W, dtype=np.float64)
        nasa7 = np.asarray(nasa7, dtype=np.float64)
        n = W.shape[0]
        assert 1 <= n <= MAXN and nasa7.shape == (n, 7)
        cfg = OConfig()
        ng = (4 if recon == 2 else 3) if ng is None else int(ng)
        assert ng >= (4 if recon == 2 else 3)
        cfg.nx, cfg.ny, cfg.nz, cfg.ng = int(nx), int(ny), int(nz), ng
        cfg.dx, cfg.dy, cfg.dz = float(dx), float(dy), float(dz)
        cfg.N, cfg.Ru = n, float(Ru)
        for s in range(n):
            cfg.W[s] = W[s]
            for q in range(7):
                cfg.a[s][q] = nasa7[s, q]
        cfg.Tlo, cfg.Thi = float(Tlo), float(Thi)
        for q in range(6):
            cfg.bc[q] = int(bc[q])
        if bc_state is not None:
            bs = np.asarray(bc_state, dtype=np.float64)
            for q in range(6):
                for v in range(n + 4):
                    cfg.bc_state[q][v] = bs[q, v]
        cfg.rtol, cfg.maxit, cfg.ideal_weights = float(rtol), int(maxit), int(ideal_weights)
        cfg.viscosity = int(viscosity)   # 0 LLF, 1 ROE, 2 GLF (xf_oracle.h)
        cfg.recon = int(recon)           # 0 WENO5-JS, 1 WENO-CU6, 2 WENO7
        cfg.positivity, cfg.pp_dt = int(positivity), float(pp_dt)
        self.cfg = cfg
        self.ng = ng
        self.N = n
        self.Nv = n + 4
        self.cells = int(lib().xo_padded_cells(C.byref(cfg)))
        self.shape = (nz + 2 * ng if nz > 1 else 1, ny + 2 * ng if ny > 1 else 1, nx + 2 * ng if nx > 1 else 1)

    @classmethod
    def from_workload(cls, wl, **kw) -> "Oracle":
        t = wl.table
        kw.setdefault("ng", getattr(wl, "ng", 3))
        return cls(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, t.W, t.nasa7, t.Ru, t.Tlo, t.Thi, wl.bc, wl.bc_state, **kw)

    # ---- per-cell pieces (for the pins) ----
    def species_thermo(self, s: int, T: float):
        cp, h, e = C.c_double(), C.c_double(), C.c_double()
        lib().xo_species_thermo(C.byref(self.cfg), s, float(T), C.byref(cp), C.byref(h), C.byref(e))
        return cp.value, h.value, e.value

    def mixture(self, Y, T: float):
        Y = np.ascontiguousarray(Y, dtype=np.float64)
        R, e, cv = C.c_double(), C.c_double(), C.c_double()
        lib().xo_mixture(C.byref(self.cfg), _dp(Y), float(T), C.byref(R), C.byref(e), C.byref(cv))
        return R.value, e.value, cv.value

    def cell_primitives(self, Ucell, Tguess: float) -> OPrim:
        Ucell = np.ascontiguousarray(Ucell, dtype=np.float64)
        P = OPrim()
        lib().xo_cell_primitives(C.byref(self.cfg), _dp(Ucell), float(Tguess), C.byref(P))
        return P

    def phys_flux(self, Ucell, P: OPrim, d: int) -> np.ndarray:
        Ucell = np.ascontiguousarray(Ucell, dtype=np.float64)
        F = np.zeros(self.Nv)
        lib().xo_phys_flux(C.byref(self.cfg), _dp(Ucell), C.byref(P), d, _dp(F))
        return F

    def eigensystem(self, PA: OPrim, PB: OPrim, d: int):
        L = np.zeros((self.Nv, self.Nv))
        R = np.zeros((self.Nv, self.Nv))
        roe = np.zeros(6)
        st = lib().xo_eigensystem(C.byref(self.cfg), C.byref(PA), C.byref(PB), d, _dp(L), _dp(R), _dp(roe))
        return L, R, roe, st

    def positivity_blend(self, d: int, Ua, Pa: OPrim, Ub, Pb: OPrim, kappa: float, Fhat):
        """-> (theta, blended flux); Fhat is not modified"""
        Ua = np.ascontiguousarray(Ua, dtype=np.float64)
        Ub = np.ascontiguousarray(Ub, dtype=np.float64)
        F = np.array(Fhat, dtype=np.float64)
        th = lib().xo_positivity_blend(C.byref(self.cfg), d, _dp(Ua), C.byref(Pa), _dp(Ub), C.byref(Pb), float(kappa), _dp(F))
        return float(th), F

    def face_flux(self, d: int, Ust, Tguess) -> np.ndarray:
        """Ust[S][Nv]: the S = 6 (8 for WENO7) stencil cells; primitives by Newton from Tguess[S]."""
        Ust = np.ascontiguousarray(Ust, dtype=np.float64)
        S = int(lib().xo_stencil_cells(C.byref(self.cfg)))
        assert Ust.shape[0] == S
        prims = (OPrim * S)()
        for m in range(S):
            lib().xo_cell_primitives(C.byref(self.cfg), _dp(Ust[m]), float(Tguess[m]), C.byref(prims[m]))
        F = np.zeros(self.Nv)
        lib().xo_face_flux(C.byref(self.cfg), d, _dp(Ust), prims, _dp(F))
        return F

    # ---- whole-field calls; U [Nv, nzp, nyp, nxp], T [nzp, nyp, nxp], modified in place like the C-ABI ----
    def _chk(self, U, T=None):
        assert U.dtype == np.float64 and U.flags["C_CONTIGUOUS"] and U.size == self.Nv * self.cells
        if T is not None:
            assert T.dtype == np.float64 and T.flags["C_CONTIGUOUS"] and T.size == self.cells

    def fill_ghosts(self, U):
        self._chk(U)
        lib().xo_fill_ghosts(C.byref(self.cfg), _dp(U))

    def primitives(self, U, T, p=None, c=None):
        self._chk(U, T)
        it = C.c_double()
        st = lib().xo_primitives(C.byref(self.cfg), _dp(U), _dp(T), _dp(p) if p is not None else None,
                                 _dp(c) if c is not None else None, C.byref(it))
        return st, it.value

    def rhs(self, U, T, fill: bool = True) -> np.ndarray:
        self._chk(U, T)
        out = np.zeros_like(U)
        fn = lib().xo_rhs if fill else lib().xo_rhs_nofill
        self.last_status = fn(C.byref(self.cfg), _dp(U), _dp(T), _dp(out))
        return out

    def rhs_cells(self, U, Tguess, idx) -> np.ndarray:
        """rhs at padded linear cell indices ``idx`` (U must have filled ghosts) -> [len(idx), Nv]."""
        self._chk(U, Tguess)
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        out = np.zeros((idx.shape[0], self.Nv))
        self.last_status = lib().xo_rhs_cells(C.byref(self.cfg), _dp(U), _dp(Tguess), idx.shape[0],
                                               idx.ctypes.data_as(C.POINTER(C.c_long)), _dp(out))
        return out

    def rk3_step(self, U, T, dt: float) -> int:
        self._chk(U, T)
        return lib().xo_rk3_step(C.byref(self.cfg), _dp(U), _dp(T), float(dt))

    # ---- viscous / diffusive terms (xf_oracle.h: readings R19-R23); tr = make_transport(workloads.TransportFits) ----
    def transport_cell(self, tr: OTransport, rho: float, Y, T: float):
        """-> (mu, kappa, rho D_sm [N], h_s [N])"""
        Y = np.ascontiguousarray(Y, dtype=np.float64)
        mu, ka = C.c_double(), C.c_double()
        rD, h = np.zeros(self.N), np.zeros(self.N)
        lib().xo_transport_cell(C.byref(self.cfg), C.byref(tr), float(rho), _dp(Y), float(T), C.byref(mu), C.byref(ka),
                                _dp(rD), _dp(h))
        return mu.value, ka.value, rD, h

    def viscous_face_flux(self, tr: OTransport, U, T, ia: int, d: int):
        """-> (F_v [Nv] at the face above padded cell ia in direction d, J_s.n [N])"""
        self._chk(U, T)
        F, J = np.zeros(self.Nv), np.zeros(self.N)
        lib().xo_viscous_face_flux(C.byref(self.cfg), C.byref(tr), _dp(U), _dp(T), int(ia), int(d), _dp(F), _dp(J))
        return F, J

    def viscous_rhs(self, tr: OTransport, U, T) -> np.ndarray:
        """div F_v at interior cells from ghost-filled U and the converged T of every padded cell"""
        self._chk(U, T)
        out = np.zeros_like(U)
        lib().xo_viscous_rhs(C.byref(self.cfg), C.byref(tr), _dp(U), _dp(T), _dp(out))
        return out

    def rhs_ns(self, tr: OTransport, U, T) -> np.ndarray:
        self._chk(U, T)
        out = np.zeros_like(U)
        self.last_status = lib().xo_rhs_ns(C.byref(self.cfg), C.byref(tr), _dp(U), _dp(T), _dp(out))
        return out

    def rk3_step_ns(self, tr: OTransport, U, T, dt: float) -> int:
        self._chk(U, T)
        return lib().xo_rk3_step_ns(C.byref(self.cfg), C.byref(tr), _dp(U), _dp(T), float(dt))

    # ---- reaction step (xf_oracle.h: readings R24-R30); m = make_mechanism(workloads.Mechanism) ----
    def reaction_rates(self, m: OMechanism, rho: float, Y, T: float):
        """-> (q [N], d [N]): production and destruction rates of Y_s"""
        Y = np.ascontiguousarray(Y, dtype=np.float64)
        q, d = np.zeros(self.N), np.zeros(self.N)
        lib().xo_reaction_rates(C.byref(self.cfg), C.byref(m), float(rho), _dp(Y), float(T), _dp(q), _dp(d))
        return q, d

    def react_cell(self, m: OMechanism, Ucell, T: float, dt: float, n_sub: int = 1, n_corr: int = 1):
        """-> (status, Ucell after the reaction step, T)"""
        Uc = np.array(Ucell, dtype=np.float64)
        Tk = np.array([T], dtype=np.float64)
        st = lib().xo_react_cell(C.byref(self.cfg), C.byref(m), _dp(Uc), _dp(Tk), float(dt), int(n_sub), int(n_corr))
        return st, Uc, float(Tk[0])

    def react(self, m: OMechanism, U, T, dt: float, n_sub: int = 1, n_corr: int = 1) -> int:
        self._chk(U, T)
        return lib().xo_react(C.byref(self.cfg), C.byref(m), _dp(U), _dp(T), float(dt), int(n_sub), int(n_corr))

    def max_wavespeed(self, U, T) -> float:
        self._chk(U, T)
        st = C.c_int()
        S = lib().xo_max_wavespeed(C.byref(self.cfg), _dp(U), _dp(T), C.byref(st))
        self.last_status = st.value
        return float(S)
