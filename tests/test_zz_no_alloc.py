"""-m gpu test of the no-allocation entry point xf_convective_rhs_noalloc (include/xf.h): the residual evaluation on the
library's file-scope `static __device__` scratch array instead of a caller-provided workspace.

The existing path (xf_convective_rhs with a workspace) is the reference here: same kernels, same inputs, so the two
residuals must agree within the tests' per-RHS bar (1e-12 of each row's maximum, tests/test_gpu_parity.py) -- and, the
arithmetic being the same instruction stream, bit for bit.  Calls come in a row on the SAME shared scratch, with
different problems between them, so that a result that depended on what the previous call left there would show.

This file sorts last on purpose (`pytest --collect-only`): the suite runs with `pytest -x`.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2403_05910_b200 import workloads as wl

pytestmark = pytest.mark.gpu

RHS_TOL = 1e-12


def _err(a, b):
    nv = a.shape[0]
    a2, b2 = a.reshape(nv, -1), b.reshape(nv, -1)
    den = np.abs(b2).max(axis=1)
    den[1:4] = den[1:4].max()
    return np.abs(a2 - b2).max(axis=1) / np.maximum(den, 1e-300)


class _Pair:
    """One context, one device state, and both ways of evaluating its residual."""

    def __init__(self, w, **kw):
        from gpu_helpers import GpuRun

        self.g = GpuRun(w, **kw)
        self.w = w

    def reference(self):
        self.g.reset()
        return self.g.rhs()                                   # xf_convective_rhs with a torch-allocated workspace

    def noalloc(self, stream=None):
        g = self.g
        g.reset()
        out = g.torch.zeros_like(g.U)
        g.ctx.xf_convective_rhs_noalloc(g.U, g.T, out, stream)
        assert g.ctx.xf_status() == 0
        return out.cpu().numpy()

    def close(self):
        self.g.close()


def _check(p):
    ref = p.reference()
    got = p.noalloc()
    assert np.abs(ref).max() > 0.0
    err = _err(p.w.interior(got), p.w.interior(ref))
    assert err.max() < RHS_TOL, err
    assert np.array_equal(got, ref)                           # same kernels on the same data: bit for bit


def test_two_calls_in_a_row_match_the_workspace_path():
    """Calls back to back on the shared scratch, with different problems (3-D N = 4 with every boundary kind, a smaller
    2-D N = 3 one, then the first again, then the first with other data): each equals the existing path's residual."""
    a = _Pair(wl.random_smooth_box(36, 30, 22, nspecies=4, seed=11, bc=(3, 1, 2, 2, 0, 0)))
    b = _Pair(wl.random_smooth_box(70, 36, 1, nspecies=3, seed=12, bc=(1, 1, 0, 0, 0, 0)))
    a.g.ctx.xf_noalloc_prepare()
    _check(a)
    _check(a)                                                 # two calls in a row, same problem
    _check(b)                                                 # the scratch now holds the larger problem's leftovers
    _check(a)
    w2 = wl.random_smooth_box(36, 30, 22, nspecies=4, seed=99, bc=(3, 1, 2, 2, 0, 0))
    a.w.U[...] = w2.U                                         # same context, other data
    a.w.T_guess[...] = w2.T_guess
    _check(a)
    a.close()
    b.close()


def test_odd_extents_and_other_options():
    """The fallback kernels (odd extents: no TMA), WENO-CU6 with ROE viscosity, and the limiter on rough data."""
    p = _Pair(wl.random_smooth_box(21, 19, 17, nspecies=5, seed=13, bc=(1, 2, 2, 1, 0, 0)), reconstruction=1, viscosity=1)
    _check(p)
    _check(p)
    p.close()
    w = wl.rough_box(34, 28, 1, nspecies=4, seed=3)
    q = _Pair(w, positivity=True)
    q.g.ctx.xf_set_rhs_dt(1e-3 * w.dx)
    _check(q)
    _check(q)
    q.close()


def test_viscous_context_uses_the_scratch_for_the_cell_table_too():
    """A context with a transport table: the residual includes div F_v and the cell table of the viscous kernels sits in
    the static scratch behind the primitives."""
    w = wl.random_smooth_box(30, 26, 20, nspecies=4, seed=21, bc=(0,) * 6)
    tr = wl.synthetic_transport(w.table, seed=4)
    p = _Pair(w, transport=tr)
    _check(p)
    _check(p)
    p.close()


def test_calls_on_a_side_stream_and_no_device_memory_is_taken():
    """The entry point on a non-default stream, and what it is for: after one warm call (kernel modules loaded), further
    calls leave the device's free memory exactly where it was."""
    import torch

    p = _Pair(wl.random_smooth_box(40, 24, 18, nspecies=10, seed=31, bc=(0,) * 6))
    ref = p.reference()
    g = p.g
    out = torch.zeros_like(g.U)
    side = torch.cuda.Stream()
    g.reset()
    torch.cuda.synchronize()
    g.ctx.xf_convective_rhs_noalloc(g.U, g.T, out, side.cuda_stream)      # warm call
    side.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        g.reset()                                             # T is in/out (the Newton guess): the same start as the reference
        torch.cuda.synchronize()
        g.ctx.xf_convective_rhs_noalloc(g.U, g.T, out, side.cuda_stream)
        side.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert g.ctx.xf_status() == 0
    assert np.array_equal(out.cpu().numpy(), ref)
    p.close()


def test_problems_beyond_the_static_scratch_are_rejected_with_a_clear_error():
    import torch

    from paper_2403_05910_b200 import xf

    cap = int(xf.lib().xf_noalloc_scratch_bytes())
    assert cap == 64 << 20
    # 1-D, N = 2: N + 4 = 6 scratch fields per padded cell -> just above the cap
    nx = cap // (6 * 8) + 64
    w = wl.random_smooth_box(nx, 1, 1, nspecies=2, seed=5)
    ctx = xf.Context.from_workload(w)
    assert ctx.rhs_workspace_bytes > cap
    U = torch.from_numpy(w.U.copy()).cuda()
    T = torch.from_numpy(w.T_guess.copy()).cuda()
    out = torch.full_like(U, 7.0)
    with pytest.raises(xf.XfError) as ei:
        ctx.xf_convective_rhs_noalloc(U, T, out)
    assert ei.value.code == xf.XF_ETOOBIG
    assert "static scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                           # nothing was launched
    assert np.array_equal(U.cpu().numpy(), w.U)               # not even the ghost fill
    # the same problem still runs through the workspace path
    ctx.xf_convective_rhs(U, T, out, ctx.workspace())
    assert ctx.xf_status() == 0
    ctx.close()
    # and the largest size that fits is accepted
    nx_ok = cap // (6 * 8) - 6
    w = wl.random_smooth_box(nx_ok, 1, 1, nspecies=2, seed=5)
    p = _Pair(w)
    assert p.g.ctx.rhs_workspace_bytes <= cap
    _check(p)
    p.close()
