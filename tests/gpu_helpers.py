"""Helpers of the -m gpu parity tests: move a seeded workload to the device and call the C-ABI binding."""
from __future__ import annotations

import numpy as np


class GpuRun:
    """Device copies of one workload + an xf Context.  All compute goes through the C-ABI binding."""

    def __init__(self, w, **kw):
        import torch

        from paper_2403_05910_b200 import xf

        self.torch = torch
        self.w = w
        self.ctx = xf.Context.from_workload(w, **kw)
        self.U = torch.from_numpy(w.U.copy()).cuda()
        self.T = torch.from_numpy(w.T_guess.copy()).cuda()
        self.work = self.ctx.workspace()
        self.S = torch.zeros(1, dtype=torch.float64, device="cuda")

    def reset(self, U=None, T=None):
        self.U.copy_(self.torch.from_numpy(self.w.U if U is None else U))
        self.T.copy_(self.torch.from_numpy(self.w.T_guess if T is None else T))

    def rhs(self) -> np.ndarray:
        """One xf_convective_rhs on the current device state -> host [Nv, nzp, nyp, nxp] (ghost entries zeroed)."""
        out = self.torch.zeros_like(self.U)
        self.ctx.xf_convective_rhs(self.U, self.T, out, self.work)
        assert self.ctx.xf_status() == 0
        return out.cpu().numpy()

    def max_wavespeed(self) -> float:
        self.ctx.xf_max_wavespeed(self.U, self.T, self.S)
        return float(self.S.item())

    def step(self, dt: float):
        self.ctx.xf_rk3_step(self.U, self.T, dt, self.work)

    def host_U(self) -> np.ndarray:
        return self.U.cpu().numpy()

    def host_T(self) -> np.ndarray:
        return self.T.cpu().numpy()

    def close(self):
        self.ctx.close()
