import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

os.environ.setdefault("OMP_WAIT_POLICY", "passive")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle

    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def oracle_ld(tmp_path_factory, oracle_mod):
    """A LONG-DOUBLE build of oracle/xf_oracle.c, produced by text substitution (double -> long double, libm calls and
    literals suffixed): the oracle's own arithmetic in 80 bits, used to measure the round-off floor of the fp64 oracle
    (tests/test_oracle_roundoff_floor.py) and the conditioning of the positivity limiter.  Nothing of the CUDA path is
    involved.  Returns rhs_cells(w, U_filled, Tguess, idx, **config) -> long-double [len(idx), Nv]."""
    import ctypes as C
    import re
    import subprocess

    import numpy as np

    LD = np.longdouble
    if np.finfo(LD).eps >= np.finfo(np.float64).eps:
        pytest.skip("no extended-precision long double on this platform")
    MAXN, MAXNV = 16, 20
    src_dir = Path(oracle_mod.__file__).resolve().parent
    out = tmp_path_factory.mktemp("oracle_ld")
    lit = re.compile(r"(?<![\w.])(\d+\.\d*(?:[eE][-+]?\d+)?|\d+[eE][-+]?\d+)(?![\w.])")
    for name in ("xf_oracle.c", "xf_oracle.h"):
        t = (src_dir / name).read_text()
        t = re.sub(r"\bdouble\b", "long double", t)
        for f in ("sqrt", "fabs", "fmax", "fmin", "exp", "log", "pow"):
            t = re.sub(rf"\b{f}\(", f"{f}l(", t)
        t = lit.sub(r"\1L", t)
        (out / name).write_text(t)
    so = out / "libxf_oracle_ld.so"
    subprocess.run(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", str(so),
                    str(out / "xf_oracle.c"), "-lm"], check=True)
    ld = C.c_longdouble

    class Cfg(C.Structure):   # xo_config of oracle/xf_oracle.h with every double widened
        _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
                    ("dx", ld), ("dy", ld), ("dz", ld), ("N", C.c_int), ("Ru", ld),
                    ("W", ld * MAXN), ("a", (ld * 7) * MAXN), ("Tlo", ld), ("Thi", ld),
                    ("bc", C.c_int * 6), ("bc_state", (ld * MAXNV) * 6),
                    ("rtol", ld), ("maxit", C.c_int), ("ideal_weights", C.c_int), ("viscosity", C.c_int),
                    ("lam_glob", (ld * 3) * 3), ("recon", C.c_int), ("positivity", C.c_int), ("pp_dt", ld)]

    lib = C.CDLL(str(so))
    lib.xo_rhs_cells.argtypes = [C.POINTER(Cfg), C.c_void_p, C.c_void_p, C.c_long, C.c_void_p, C.c_void_p]

    def rhs_cells(w, U_filled, Tguess, idx, viscosity=0, recon=0, positivity=False, pp_dt=0.0):
        """long-double rhs at the sampled cells; the INPUTS are the doubles of the fp64 run, converted exactly"""
        cfg = Cfg()
        cfg.nx, cfg.ny, cfg.nz, cfg.ng = w.nx, w.ny, w.nz, getattr(w, "ng", 3)
        cfg.dx, cfg.dy, cfg.dz = w.dx, w.dy, w.dz
        t = w.table
        cfg.N, cfg.Ru = t.n, t.Ru
        for s in range(t.n):
            cfg.W[s] = t.W[s]
            for q in range(7):
                cfg.a[s][q] = t.nasa7[s, q]
        cfg.Tlo, cfg.Thi = t.Tlo, t.Thi
        cfg.rtol, cfg.maxit = 1e-17, 60
        cfg.viscosity, cfg.recon, cfg.positivity, cfg.pp_dt = int(viscosity), int(recon), int(positivity), pp_dt
        Ul = np.ascontiguousarray(U_filled, dtype=LD)
        Tl = np.ascontiguousarray(Tguess, dtype=LD)
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        outl = np.zeros((idx.shape[0], t.n + 4), dtype=LD)
        st = lib.xo_rhs_cells(C.byref(cfg), Ul.ctypes.data, Tl.ctypes.data, idx.shape[0], idx.ctypes.data,
                              outl.ctypes.data)
        assert st in (0, 5)          # rtol 1e-17 is below what even 80 bits resolve: "not converged" means "to round-off"
        return outl

    return rhs_cells
