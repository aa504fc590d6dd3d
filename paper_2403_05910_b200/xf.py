"""Thin ctypes binding of libxf.so (include/xf.h): argument marshalling only -- every step of the path runs in the
CUDA kernels of csrc/.  PyTorch supplies device memory and streams; there is no CPU fallback: if the library is
missing or no CUDA device is present, loading / ``xf_create`` fails loudly.

Function names follow the C ABI (``xf_create``, ``xf_primitives``, ``xf_convective_rhs``, ``xf_rk3_step``,
``xf_max_wavespeed`` ...); ``Context`` is a small RAII convenience around them.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional, Sequence

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libxf.so"

XF_OK, XF_EINVAL, XF_ECUDA, XF_ENOMEM, XF_ENONPHYSICAL, XF_ENOCONV, XF_ETOOBIG = 0, -1, -2, -3, -4, -5, -6
XF_BC_PERIODIC, XF_BC_TRANSMISSIVE, XF_BC_REFLECTIVE, XF_BC_DIRICHLET, XF_BC_EXCHANGE = 0, 1, 2, 3, 4
XF_VISC_LLF, XF_VISC_ROE, XF_VISC_GLF = 0, 1, 2
XF_RECON_WENO5, XF_RECON_WENOCU6, XF_RECON_WENO7 = 0, 1, 2
XF_MAX_SPECIES = 16

# every symbol include/xf.h declares (tests check that the library exports all of them)
ABI_SYMBOLS = (
    "xf_create", "xf_destroy", "xf_num_vars", "xf_padded_cells", "xf_rhs_workspace_bytes", "xf_workspace_bytes",
    "xf_fill_ghosts", "xf_primitives", "xf_convective_rhs", "xf_rk3_step", "xf_rk3_step_cfl", "xf_step_cfl",
    "xf_max_wavespeed", "xf_set_rhs_dt", "xf_viscous_rhs", "xf_fill_ghosts_dir", "xf_halo_doubles", "xf_pack_halo",
    "xf_unpack_halo", "xf_rk3_stage", "xf_set_mechanism", "xf_react",
    "xf_status", "xf_newton_mean_iterations", "xf_launch_count", "xf_convective_rhs_host", "xf_rk3_steps_host",
    "xf_probe_fp64_peak", "xf_probe_fp64_sustained", "xf_strerror", "xf_timing_enable", "xf_timing_read",
    "xf_noalloc_scratch_bytes", "xf_noalloc_prepare", "xf_convective_rhs_noalloc",
)
KERNEL_KINDS = ("ghost_fill", "primitives", "sweep_x", "sweep_y", "sweep_z", "max_wavespeed", "transport",
                "viscous", "react")  # XF_K_* of xf.h


class XfConfig(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
        ("nspecies", C.c_int), ("Ru", C.c_double),
        ("W", C.POINTER(C.c_double)), ("nasa7", C.POINTER(C.c_double)),
        ("Tlo", C.c_double), ("Thi", C.c_double),
        ("bc", C.c_int * 6), ("bc_state", C.POINTER(C.c_double)),
        ("newton_rtol", C.c_double), ("newton_maxit", C.c_int), ("device", C.c_int), ("viscosity", C.c_int), ("reconstruction", C.c_int),
        ("positivity", C.c_int), ("transport", C.POINTER(C.c_double)),
    ]


class XfError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} ({code})")


_lib = None


def lib() -> C.CDLL:
    """Load libxf.so (built in-tree by ``paper_2403_05910_b200.build``).  Raises if it is not there."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2403_05910_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(str(LIB_PATH))
        vp, dp, ctx = C.c_void_p, C.c_void_p, C.c_void_p
        L.xf_create.argtypes = [C.POINTER(ctx), C.POINTER(XfConfig)]
        L.xf_destroy.argtypes = [ctx]
        for name in ("xf_num_vars", "xf_padded_cells", "xf_rhs_workspace_bytes", "xf_workspace_bytes"):
            getattr(L, name).argtypes = [ctx]
            getattr(L, name).restype = C.c_size_t
        L.xf_fill_ghosts.argtypes = [ctx, dp, vp]
        L.xf_primitives.argtypes = [ctx, dp, dp, dp, dp, vp]
        L.xf_convective_rhs.argtypes = [ctx, dp, dp, dp, vp, vp]
        L.xf_noalloc_scratch_bytes.argtypes = []
        L.xf_noalloc_scratch_bytes.restype = C.c_size_t
        L.xf_noalloc_prepare.argtypes = [ctx]
        L.xf_convective_rhs_noalloc.argtypes = [ctx, dp, dp, dp, vp]
        L.xf_set_rhs_dt.argtypes = [ctx, C.c_double]
        L.xf_viscous_rhs.argtypes = [ctx, dp, dp, dp, vp, vp]
        ip = C.POINTER(C.c_int)
        ddp = C.POINTER(C.c_double)
        L.xf_set_mechanism.argtypes = [ctx, C.c_int, ip, ip, ddp, ddp, ddp, ip, ddp, C.c_double]
        L.xf_react.argtypes = [ctx, dp, dp, C.c_double, C.c_int, C.c_int, vp]
        L.xf_fill_ghosts_dir.argtypes = [ctx, dp, C.c_int, vp]
        L.xf_halo_doubles.argtypes = [ctx, C.c_int]
        L.xf_halo_doubles.restype = C.c_size_t
        L.xf_pack_halo.argtypes = [ctx, dp, dp, C.c_int, C.c_int, dp, vp]
        L.xf_unpack_halo.argtypes = [ctx, dp, dp, C.c_int, C.c_int, dp, vp]
        L.xf_rk3_stage.argtypes = [ctx, C.c_int, dp, dp, dp, dp, C.c_double, vp, vp]
        L.xf_rk3_step.argtypes = [ctx, dp, dp, C.c_double, vp, vp]
        L.xf_rk3_step_cfl.argtypes = [ctx, dp, dp, C.c_double, dp, vp, vp]
        L.xf_step_cfl.argtypes = [ctx, dp, dp, C.c_double, dp, vp, vp]
        L.xf_max_wavespeed.argtypes = [ctx, dp, dp, dp, vp]
        L.xf_status.argtypes = [ctx, vp]
        L.xf_newton_mean_iterations.argtypes = [ctx, vp, C.POINTER(C.c_double)]
        L.xf_launch_count.argtypes = [ctx]
        L.xf_launch_count.restype = C.c_long
        L.xf_convective_rhs_host.argtypes = [ctx, dp, dp, dp]
        L.xf_rk3_steps_host.argtypes = [ctx, dp, dp, C.c_double, C.c_int, C.POINTER(C.c_double)]
        L.xf_probe_fp64_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.xf_probe_fp64_sustained.argtypes = [C.c_int, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.xf_timing_enable.argtypes = [ctx, C.c_int]
        L.xf_timing_read.argtypes = [ctx, vp, C.POINTER(C.c_double), C.POINTER(C.c_long)]
        L.xf_strerror.argtypes = [C.c_int]
        L.xf_strerror.restype = C.c_char_p
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().xf_strerror(int(code)).decode()


def _check(code: int, where: str) -> None:
    if code != XF_OK:
        raise XfError(code, where)


def _ptr(t) -> int:
    """Device (torch.Tensor) or host (numpy.ndarray) fp64 contiguous buffer -> raw address; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.dtype == np.float64 and t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    import torch

    assert isinstance(t, torch.Tensor) and t.is_contiguous()
    assert t.dtype in (torch.float64, torch.uint8)
    return t.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch

        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def xf_probe_fp64_peak(device: int = 0, iters: int = 4096):
    """-> (TFLOP/s, ms) of the register-resident fp64 FMA probe kernel."""
    tf, ms = C.c_double(), C.c_double()
    _check(lib().xf_probe_fp64_peak(int(device), int(iters), C.byref(tf), C.byref(ms)), "xf_probe_fp64_peak")
    return tf.value, ms.value


def xf_probe_fp64_sustained(device: int = 0, seconds: float = 1.5):
    """-> (TFLOP/s, ms) of the same probe launched back to back for at least ``seconds``."""
    tf, ms = C.c_double(), C.c_double()
    _check(lib().xf_probe_fp64_sustained(int(device), float(seconds), C.byref(tf), C.byref(ms)), "xf_probe_fp64_sustained")
    return tf.value, ms.value


class Context:
    """Owns one ``xf_ctx``.  Methods are the C-ABI calls with the context bound; tensors are caller-owned."""

    def __init__(self, nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, W: Sequence[float], nasa7, Ru: float,
                 Tlo: float, Thi: float, bc=(0,) * 6, bc_state=None, newton_rtol: float = 0.0, newton_maxit: int = 0,
                 device: int = 0, viscosity: int = XF_VISC_LLF, reconstruction: int = XF_RECON_WENO5,
                 positivity: bool = False, ng: Optional[int] = None, transport=None):
        W = np.ascontiguousarray(W, dtype=np.float64)
        nasa7 = np.ascontiguousarray(nasa7, dtype=np.float64)
        n = int(W.shape[0])
        assert nasa7.shape == (n, 7)
        cfg = XfConfig()
        ng = (4 if int(reconstruction) == XF_RECON_WENO7 else 3) if ng is None else int(ng)
        cfg.nx, cfg.ny, cfg.nz, cfg.ng = int(nx), int(ny), int(nz), ng
        cfg.dx, cfg.dy, cfg.dz = float(dx), float(dy), float(dz)
        cfg.nspecies, cfg.Ru = n, float(Ru)
        cfg.W = W.ctypes.data_as(C.POINTER(C.c_double))
        cfg.nasa7 = nasa7.ctypes.data_as(C.POINTER(C.c_double))
        cfg.Tlo, cfg.Thi = float(Tlo), float(Thi)
        for q in range(6):
            cfg.bc[q] = int(bc[q])
        bs = None
        if bc_state is not None:
            bs = np.ascontiguousarray(bc_state, dtype=np.float64)
            assert bs.shape == (6, n + 4)
            cfg.bc_state = bs.ctypes.data_as(C.POINTER(C.c_double))
        cfg.newton_rtol, cfg.newton_maxit, cfg.device = float(newton_rtol), int(newton_maxit), int(device)
        cfg.viscosity = int(viscosity)
        cfg.reconstruction = int(reconstruction)
        cfg.positivity = int(bool(positivity))
        tr = None
        if transport is not None:   # an object with mu [N,4], kappa [N,4], D [N,N,4], p_ref (workloads.TransportFits)
            tr = np.ascontiguousarray(np.concatenate([np.asarray(transport.mu, dtype=np.float64).ravel(),
                                                      np.asarray(transport.kappa, dtype=np.float64).ravel(),
                                                      np.asarray(transport.D, dtype=np.float64).ravel(),
                                                      [float(transport.p_ref)]]))
            assert tr.shape[0] == 8 * n + 4 * n * n + 1
            cfg.transport = tr.ctypes.data_as(C.POINTER(C.c_double))
        self._h = C.c_void_p()
        _check(lib().xf_create(C.byref(self._h), C.byref(cfg)), "xf_create")
        self.device = int(device)
        self.N, self.Nv = n, n + 4
        self.cells = int(lib().xf_padded_cells(self._h))
        self.ng = ng
        self.shape = tuple(m + 2 * ng if m > 1 else 1 for m in (nz, ny, nx))
        self.interior_cells = int(nx) * int(ny) * int(nz)
        self.rhs_workspace_bytes = int(lib().xf_rhs_workspace_bytes(self._h))
        self.workspace_bytes = int(lib().xf_workspace_bytes(self._h))

    @classmethod
    def from_workload(cls, wl, **kw) -> "Context":
        t = wl.table
        kw.setdefault("ng", getattr(wl, "ng", 3))
        return cls(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, t.W, t.nasa7, t.Ru, t.Tlo, t.Thi, wl.bc, wl.bc_state, **kw)

    def close(self) -> None:
        h = getattr(self, "_h", None)
        if h is not None and h.value and _lib is not None:   # at interpreter shutdown the module globals may be gone
            _lib.xf_destroy(h)
        self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # ---- device-memory helpers (plumbing) ----
    def empty_fields(self, nfields: Optional[int] = None):
        import torch

        shape = self.shape if nfields is None else (nfields,) + self.shape
        return torch.empty(shape, dtype=torch.float64, device=f"cuda:{self.device}")

    def workspace(self, rhs_only: bool = False):
        import torch

        nbytes = self.rhs_workspace_bytes if rhs_only else self.workspace_bytes
        return torch.empty(nbytes // 8, dtype=torch.float64, device=f"cuda:{self.device}")

    # ---- the C-ABI calls ----
    def xf_fill_ghosts(self, U, stream=None) -> None:
        _check(lib().xf_fill_ghosts(self._h, _ptr(U), _stream(stream)), "xf_fill_ghosts")

    def xf_primitives(self, U, T, p=None, c=None, stream=None) -> None:
        _check(lib().xf_primitives(self._h, _ptr(U), _ptr(T), _ptr(p), _ptr(c), _stream(stream)), "xf_primitives")

    def xf_convective_rhs(self, U, T, rhs, work, stream=None) -> None:
        assert work.numel() * work.element_size() >= self.rhs_workspace_bytes
        _check(lib().xf_convective_rhs(self._h, _ptr(U), _ptr(T), _ptr(rhs), _ptr(work), _stream(stream)),
               "xf_convective_rhs")

    def xf_noalloc_prepare(self) -> None:
        _check(lib().xf_noalloc_prepare(self._h), "xf_noalloc_prepare")

    def xf_convective_rhs_noalloc(self, U, T, rhs, stream=None) -> None:
        """xf_convective_rhs on the library's static device scratch (include/xf.h): no workspace, no allocation."""
        _check(lib().xf_convective_rhs_noalloc(self._h, _ptr(U), _ptr(T), _ptr(rhs), _stream(stream)),
               "xf_convective_rhs_noalloc")

    def xf_set_mechanism(self, m) -> None:
        """m: an object with nu_r, nu_p [NR, N] (int), A, B, E [NR], third [NR], eff [NR, N], p_atm (workloads.Mechanism)"""
        i32 = lambda a: np.ascontiguousarray(a, dtype=np.int32)       # noqa: E731
        f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)     # noqa: E731
        nu_r, nu_p, third, A, B, E, eff = i32(m.nu_r), i32(m.nu_p), i32(m.third), f64(m.A), f64(m.B), f64(m.E), f64(m.eff)
        assert nu_r.shape == nu_p.shape == eff.shape == (A.shape[0], self.N)
        ip, ddp = C.POINTER(C.c_int), C.POINTER(C.c_double)
        _check(lib().xf_set_mechanism(self._h, int(A.shape[0]), nu_r.ctypes.data_as(ip), nu_p.ctypes.data_as(ip),
                                      A.ctypes.data_as(ddp), B.ctypes.data_as(ddp), E.ctypes.data_as(ddp),
                                      third.ctypes.data_as(ip), eff.ctypes.data_as(ddp), float(m.p_atm)), "xf_set_mechanism")

    def xf_react(self, U, T, dt: float, n_sub: int = 1, n_corr: int = 1, stream=None) -> None:
        _check(lib().xf_react(self._h, _ptr(U), _ptr(T), float(dt), int(n_sub), int(n_corr), _stream(stream)), "xf_react")

    def xf_fill_ghosts_dir(self, U, d: int, stream=None) -> None:
        _check(lib().xf_fill_ghosts_dir(self._h, _ptr(U), int(d), _stream(stream)), "xf_fill_ghosts_dir")

    def xf_halo_doubles(self, d: int) -> int:
        return int(lib().xf_halo_doubles(self._h, int(d)))

    def xf_pack_halo(self, U, T, d: int, side: int, buf, stream=None) -> None:
        assert buf.numel() >= self.xf_halo_doubles(d)
        _check(lib().xf_pack_halo(self._h, _ptr(U), _ptr(T), int(d), int(side), _ptr(buf), _stream(stream)), "xf_pack_halo")

    def xf_unpack_halo(self, U, T, d: int, side: int, buf, stream=None) -> None:
        assert buf.numel() >= self.xf_halo_doubles(d)
        _check(lib().xf_unpack_halo(self._h, _ptr(U), _ptr(T), int(d), int(side), _ptr(buf), _stream(stream)),
               "xf_unpack_halo")

    def xf_rk3_stage(self, stage: int, Un, Uin, Uout, T, dt: float, work, stream=None) -> None:
        assert work.numel() * work.element_size() >= self.workspace_bytes
        _check(lib().xf_rk3_stage(self._h, int(stage), _ptr(Un), _ptr(Uin), _ptr(Uout), _ptr(T), float(dt), _ptr(work),
                                  _stream(stream)), "xf_rk3_stage")

    def xf_viscous_rhs(self, U, T, rhs, work, stream=None) -> None:
        assert work.numel() * work.element_size() >= self.rhs_workspace_bytes
        _check(lib().xf_viscous_rhs(self._h, _ptr(U), _ptr(T), _ptr(rhs), _ptr(work), _stream(stream)), "xf_viscous_rhs")

    def xf_set_rhs_dt(self, dt: float) -> None:
        _check(lib().xf_set_rhs_dt(self._h, float(dt)), "xf_set_rhs_dt")

    def xf_rk3_step(self, U, T, dt: float, work, stream=None) -> None:
        assert work.numel() * work.element_size() >= self.workspace_bytes
        _check(lib().xf_rk3_step(self._h, _ptr(U), _ptr(T), float(dt), _ptr(work), _stream(stream)), "xf_rk3_step")

    def xf_rk3_step_cfl(self, U, T, cfl: float, S_dev, work, stream=None) -> None:
        assert work.numel() * work.element_size() >= self.workspace_bytes
        _check(lib().xf_rk3_step_cfl(self._h, _ptr(U), _ptr(T), float(cfl), _ptr(S_dev), _ptr(work), _stream(stream)),
               "xf_rk3_step_cfl")

    def xf_step_cfl(self, U, T, cfl: float, S_dev, work, stream=None) -> None:
        assert work.numel() * work.element_size() >= self.workspace_bytes
        _check(lib().xf_step_cfl(self._h, _ptr(U), _ptr(T), float(cfl), _ptr(S_dev), _ptr(work), _stream(stream)),
               "xf_step_cfl")

    def xf_max_wavespeed(self, U, T, S_dev, stream=None) -> None:
        _check(lib().xf_max_wavespeed(self._h, _ptr(U), _ptr(T), _ptr(S_dev), _stream(stream)), "xf_max_wavespeed")

    def xf_status(self, stream=None) -> int:
        return int(lib().xf_status(self._h, _stream(stream)))

    def xf_newton_mean_iterations(self, stream=None) -> float:
        m = C.c_double()
        _check(lib().xf_newton_mean_iterations(self._h, _stream(stream), C.byref(m)), "xf_newton_mean_iterations")
        return m.value

    def xf_launch_count(self) -> int:
        return int(lib().xf_launch_count(self._h))

    def xf_timing_enable(self, max_records: int) -> None:
        _check(lib().xf_timing_enable(self._h, int(max_records)), "xf_timing_enable")

    def xf_timing_read(self, stream=None) -> dict:
        """-> {kernel kind: (total ms, records)} since the last read."""
        n = len(KERNEL_KINDS)
        ms, cnt = (C.c_double * n)(), (C.c_long * n)()
        _check(lib().xf_timing_read(self._h, _stream(stream), ms, cnt), "xf_timing_read")
        return {k: (ms[q], cnt[q]) for q, k in enumerate(KERNEL_KINDS)}

    def xf_convective_rhs_host(self, U_host: np.ndarray, T_host: np.ndarray, rhs_host: np.ndarray) -> None:
        _check(lib().xf_convective_rhs_host(self._h, _ptr(U_host), _ptr(T_host), _ptr(rhs_host)),
               "xf_convective_rhs_host")

    def xf_rk3_steps_host(self, U_host: np.ndarray, T_host: np.ndarray, cfl: float, nsteps: int) -> float:
        t = C.c_double()
        _check(lib().xf_rk3_steps_host(self._h, _ptr(U_host), _ptr(T_host), float(cfl), int(nsteps), C.byref(t)),
               "xf_rk3_steps_host")
        return t.value
