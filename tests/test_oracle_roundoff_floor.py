"""The oracle's own round-off floor, measured against a LONG-DOUBLE build of the very same source.

Why: reading R14 normalises the error of a residual row by that row's largest magnitude.  For a partial density that is
present only where nothing moves yet (config 2's bubble gas at t = 0), or a trace species (config 4), the row's own
residual can be smaller than the round-off it inherits from the O(rho c) characteristic fluxes the mass flux is assembled
from: Fhat_{rho Y_s} = Y~_s s + g_s, and s = g_0 + g_1 + g_{Nv-1} cancels to eps rho c in quiescent gas.  That floor
belongs to the ARITHMETIC, not to an implementation: this test shows the fp64 oracle missing its own 80-bit build by more
than 1e-12 of the row's own scale on such rows, and by < 2e-13 on the scale DESIGN.md section 11 derives,
max(own scale, max Y_s x density-row scale) -- the scale tests/test_gpu_parity.py uses at full size.

The long-double library is produced from oracle/xf_oracle.c by text substitution (double -> long double, libm calls and
literals suffixed; fixture `oracle_ld` of tests/conftest.py); nothing of the CUDA path is involved.
"""
import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

LD = np.longdouble
pytestmark = pytest.mark.skipif(np.finfo(LD).eps >= np.finfo(np.float64).eps,
                                reason="no extended-precision long double on this platform")


def _samples(w, rng, n_rand, x_bands):
    gz, gy, gx = (3 if w.nz > 1 else 0), (3 if w.ny > 1 else 0), (3 if w.nx > 1 else 0)
    nzp, nyp, nxp = w.padded_shape
    i = [rng.integers(0, w.nx, n_rand)]
    for lo, hi, cnt in x_bands:                                # cells around the shock / across the bubble
        i.append(rng.integers(int(lo * w.nx), max(int(hi * w.nx), int(lo * w.nx) + 1), cnt))
    i = np.concatenate(i)
    j = rng.integers(0, w.ny, i.size)
    k = rng.integers(0, w.nz, i.size)
    return ((k + gz).astype(np.int64) * nyp + (j + gy)) * nxp + (i + gx)


@pytest.mark.parametrize("name", ["config2_full", "config4_reduced"])
def test_fp64_oracle_against_its_long_double_build(oracle_mod, oracle_ld, name):
    rng = np.random.default_rng(wl.SEED_BASE + 77)
    if name == "config2_full":
        w = wl.config2_shock_bubble_2d(2048, 1024)
        idx = _samples(w, rng, 1500, [(0.14, 0.16, 1000), (0.19, 0.41, 2500)])   # shock at x = 0.3 of [0, 2]; bubble
    else:
        w = wl.config4_shock_bubble_3d_10sp(128, 64, 64)
        idx = _samples(w, rng, 1500, [(0.14, 0.16, 1000), (0.22, 0.38, 2500)])
    orc = oracle_mod.Oracle.from_workload(w)
    U = w.U.copy()
    orc.fill_ghosts(U)
    r64 = orc.rhs_cells(U, w.T_guess, idx)
    assert orc.last_status == 0
    r80 = oracle_ld(w, U, w.T_guess, idx)
    nv = w.nvars
    err = np.abs(r64.astype(LD) - r80).max(axis=0).astype(np.float64)
    own = np.abs(r80).max(axis=0).astype(np.float64)
    own[1:4] = own[1:4].max()
    Ymax = (np.abs(w.interior(w.U)[5:]) / w.interior(w.U)[0]).reshape(nv - 5, -1).max(axis=1)
    scale = own.copy()
    scale[5:] = np.maximum(own[5:], Ymax * own[0])
    print(name, "fp64 oracle vs long double, own scale:", err / own)
    print(name, "fp64 oracle vs long double, R14 scale:", err / scale)
    assert (err / scale).max() < 2e-13                         # the floor on the scale the parity tests use
    assert (err / own)[:5].max() < 2e-13                       # rho, momentum, E: own scale is fine
    if name == "config2_full":
        # the bubble gas (row 6) is quiescent at t = 0: on its OWN scale the fp64 oracle is off by more than the 1e-12 bar
        assert (err / own)[6] > 1e-12
