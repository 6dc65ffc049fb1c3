"""Thin ctypes binding of libburgers.so (include/burgers.h) -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; this module only turns
torch tensors / numpy arrays into pointers and sizes.  There is NO CPU fallback: if the
library has not been built (``python -m paper_2601_12204_b200.build``) importing this module
raises, and calling a device entry point with a non-CUDA tensor raises.

Device calls take torch CUDA tensors (``u`` [B][N] contiguous, ``nu``/``dt`` [B]) and enqueue on
the current torch stream; ``*_host`` calls take numpy arrays (host memory) and return when the
result is back in host memory.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libburgers.so")

OK = 0
ERR_NULL, ERR_SHAPE, ERR_ENUM, ERR_VALUE, ERR_WORKSPACE, ERR_CUDA, ERR_PLAN = -1, -2, -3, -4, -5, -6, -7
ERR_LIMIT = -8
BC_PERIODIC, BC_DIRICHLET = 0, 1
SCHEME_EULER, SCHEME_RK4 = 0, 1
OP_EXPLICIT, OP_BTCS, OP_CFL, OP_NEWTON, OP_GS = 0, 1, 2, 3, 4
PLAN_AUTO, PLAN_RESIDENT, PLAN_TILED, PLAN_THOMAS, PLAN_HYBRID, PLAN_LONG, PLAN_LONG_GENERAL = 0, 1, 2, 3, 4, 5, 6

EXPORTS = [
    "burgers_explicit_f32", "burgers_explicit_f64", "burgers_explicit_plan_f32",
    "burgers_explicit_plan_f64", "burgers_explicit_traj_f32", "burgers_explicit_traj_f64", "burgers_explicit_adaptive_f32", "burgers_explicit_adaptive_f64", "burgers_explicit_adjoint_f32", "burgers_explicit_adjoint_f64",
    "burgers_adjoint_workspace_bytes", "burgers_explicit_adjoint_ckpt_f32", "burgers_explicit_adjoint_ckpt_f64",
    "burgers_adjoint_ckpt_workspace_bytes", "burgers_explicit_adjoint_scheme_f32", "burgers_explicit_adjoint_scheme_f64",
    "burgers_adjoint_scheme_workspace_bytes", "burgers_btcs_f32", "burgers_btcs_f64", "burgers_btcs_plan_f32",
    "burgers_btcs_plan_f64", "burgers_btcs_traj_f32", "burgers_btcs_traj_f64", "burgers_btcs_adjoint_f32", "burgers_btcs_adjoint_f64",
    "burgers_btcs_adjoint_workspace_bytes", "burgers_btcs_gs_f32", "burgers_btcs_gs_f64", "burgers_newton_f32", "burgers_newton_f64", "burgers_newton_traj_f32", "burgers_newton_traj_f64", "dt_from_cfl_f32", "dt_from_cfl_f64", "burgers_explicit_host_f32",
    "burgers_explicit_host_f64", "burgers_btcs_host_f32", "burgers_btcs_host_f64",
    "burgers_newton_host_f32", "burgers_newton_host_f64", "dt_from_cfl_host_f32", "dt_from_cfl_host_f64",
    "burgers_solve_host_f32", "burgers_solve_host_f64", "burgers_workspace_bytes", "burgers_plan_query",
    "burgers_launch_count", "burgers_pipe_peak", "burgers_strerror", "burgers_version",
    "burgers_noalloc_scratch_bytes", "burgers_noalloc_init", "burgers_btcs_noalloc",
    "burgers_newton_adjoint_f32", "burgers_newton_adjoint_f64", "burgers_newton_adjoint_workspace_bytes",
    "burgers_btcs_adjoint_ckpt_f32", "burgers_btcs_adjoint_ckpt_f64", "burgers_newton_adjoint_ckpt_f32",
    "burgers_newton_adjoint_ckpt_f64", "burgers_implicit_adjoint_ckpt_workspace_bytes",
]

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_2601_12204_b200.build` "
        "(there is no CPU fallback)")

_lib = ctypes.CDLL(LIB_PATH)

_p, _i64, _f64, _int, _sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int, ctypes.c_size_t
for _sfx in ("f32", "f64"):
    getattr(_lib, f"burgers_explicit_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _int, _p, _sz, _p]
    getattr(_lib, f"burgers_explicit_plan_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _int, _int, _int, _int, _p, _sz, _p]
    getattr(_lib, f"burgers_btcs_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _p, _sz, _p]
    getattr(_lib, f"burgers_explicit_traj_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _int, _i64, _p, _p, _sz, _p]
    getattr(_lib, f"burgers_explicit_traj_{_sfx}").restype = _int
    getattr(_lib, f"burgers_explicit_adaptive_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _f64, _i64, _i64, _int, _int, _p, _p, _p, _sz, _p]
    getattr(_lib, f"burgers_explicit_adaptive_{_sfx}").restype = _int
    getattr(_lib, f"burgers_explicit_adjoint_{_sfx}").argtypes = [_p, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _p, _sz, _p]
    getattr(_lib, f"burgers_explicit_adjoint_{_sfx}").restype = _int
    getattr(_lib, f"burgers_explicit_adjoint_ckpt_{_sfx}").argtypes = [_p, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _i64, _p, _sz, _p]
    getattr(_lib, f"burgers_explicit_adjoint_ckpt_{_sfx}").restype = _int
    getattr(_lib, f"burgers_explicit_adjoint_scheme_{_sfx}").argtypes = [_p, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _int, _i64, _p, _sz, _p]
    getattr(_lib, f"burgers_explicit_adjoint_scheme_{_sfx}").restype = _int
    getattr(_lib, f"burgers_btcs_adjoint_{_sfx}").argtypes = [_p, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _p, _sz, _p]
    getattr(_lib, f"burgers_btcs_adjoint_{_sfx}").restype = _int
    getattr(_lib, f"burgers_newton_adjoint_{_sfx}").argtypes = [_p, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _f64, _f64, _int,
                                                               _p, _sz, _p]
    getattr(_lib, f"burgers_newton_adjoint_{_sfx}").restype = _int
    getattr(_lib, f"burgers_btcs_adjoint_ckpt_{_sfx}").argtypes = [_p, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _i64, _p, _sz, _p]
    getattr(_lib, f"burgers_btcs_adjoint_ckpt_{_sfx}").restype = _int
    getattr(_lib, f"burgers_newton_adjoint_ckpt_{_sfx}").argtypes = [_p, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _f64, _f64,
                                                                    _int, _i64, _p, _sz, _p]
    getattr(_lib, f"burgers_newton_adjoint_ckpt_{_sfx}").restype = _int
    getattr(_lib, f"burgers_btcs_traj_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _i64, _p, _p, _sz, _p]
    getattr(_lib, f"burgers_btcs_traj_{_sfx}").restype = _int
    getattr(_lib, f"burgers_btcs_gs_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _f64, _int, _p, _p, _sz, _p]
    getattr(_lib, f"burgers_btcs_gs_{_sfx}").restype = _int
    getattr(_lib, f"burgers_btcs_plan_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _int, _p, _sz, _p]
    getattr(_lib, f"dt_from_cfl_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _f64, _int, _p, _p]
    getattr(_lib, f"burgers_newton_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _f64, _f64, _int, _p, _int, _p, _sz, _p]
    getattr(_lib, f"burgers_newton_{_sfx}").restype = _int
    getattr(_lib, f"burgers_newton_traj_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _f64, _f64, _int, _p, _i64, _p, _p, _sz, _p]
    getattr(_lib, f"burgers_newton_traj_{_sfx}").restype = _int
    getattr(_lib, f"burgers_newton_host_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _f64, _f64, _int, _p]
    getattr(_lib, f"burgers_newton_host_{_sfx}").restype = _int
    getattr(_lib, f"burgers_explicit_host_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int, _int]
    getattr(_lib, f"burgers_btcs_host_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _p, _i64, _int]
    getattr(_lib, f"dt_from_cfl_host_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _f64, _int, _p]
    getattr(_lib, f"burgers_solve_host_{_sfx}").argtypes = [_p, _i64, _i64, _f64, _p, _f64, _i64, _int, _int, _int, _p]
    getattr(_lib, f"burgers_solve_host_{_sfx}").restype = _int
    for _n in ("burgers_explicit_", "burgers_explicit_plan_", "burgers_btcs_", "burgers_btcs_plan_",
               "dt_from_cfl_", "burgers_explicit_host_", "burgers_btcs_host_", "dt_from_cfl_host_"):
        getattr(_lib, _n + _sfx).restype = _int
_lib.burgers_workspace_bytes.argtypes = [_int, _int, _i64, _i64, _int, _int, _int]
_lib.burgers_workspace_bytes.restype = _sz
_lib.burgers_adjoint_workspace_bytes.argtypes = [_int, _i64, _i64, _int, _i64]
_lib.burgers_adjoint_workspace_bytes.restype = _sz
_lib.burgers_adjoint_ckpt_workspace_bytes.argtypes = [_int, _i64, _i64, _int, _i64, _i64]
_lib.burgers_adjoint_ckpt_workspace_bytes.restype = _sz
_lib.burgers_adjoint_scheme_workspace_bytes.argtypes = [_int, _i64, _i64, _int, _int, _i64, _i64]
_lib.burgers_adjoint_scheme_workspace_bytes.restype = _sz
_lib.burgers_btcs_adjoint_workspace_bytes.argtypes = [_int, _i64, _i64, _int, _i64]
_lib.burgers_btcs_adjoint_workspace_bytes.restype = _sz
_lib.burgers_newton_adjoint_workspace_bytes.argtypes = [_int, _i64, _i64, _int, _i64]
_lib.burgers_newton_adjoint_workspace_bytes.restype = _sz
_lib.burgers_implicit_adjoint_ckpt_workspace_bytes.argtypes = [_int, _int, _i64, _i64, _int, _i64, _i64]
_lib.burgers_implicit_adjoint_ckpt_workspace_bytes.restype = _sz
_lib.burgers_plan_query.argtypes = [_int, _int, _i64, _i64, _int, _int]
_lib.burgers_plan_query.restype = _int
_lib.burgers_launch_count.argtypes = [_int, _int, _i64, _i64, _int, _int, _int, _int, _i64]
_lib.burgers_launch_count.restype = _i64
_lib.burgers_pipe_peak.argtypes = [_int, _i64, _p, _p, ctypes.POINTER(ctypes.c_double)]
_lib.burgers_pipe_peak.restype = _int
_lib.burgers_noalloc_scratch_bytes.argtypes = []
_lib.burgers_noalloc_scratch_bytes.restype = _sz
_lib.burgers_noalloc_init.argtypes = []
_lib.burgers_noalloc_init.restype = _int
_lib.burgers_btcs_noalloc.argtypes = [_int, _p, _i64, _i64, _f64, _p, _p, _i64, _int, _p]
_lib.burgers_btcs_noalloc.restype = _int
_lib.burgers_strerror.argtypes = [_int]
_lib.burgers_strerror.restype = ctypes.c_char_p
_lib.burgers_version.argtypes = []
_lib.burgers_version.restype = _int


class BurgersError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} (status {status})")


def raw():
    """The ctypes library handle (tests of the raw C ABI: error codes, symbols)."""
    return _lib


def strerror(status: int) -> str:
    return _lib.burgers_strerror(int(status)).decode()


def version() -> int:
    return int(_lib.burgers_version())


def workspace_bytes(op, is_f64, B, N, bc, scheme=0, plan=PLAN_AUTO) -> int:
    return int(_lib.burgers_workspace_bytes(op, int(bool(is_f64)), B, N, bc, scheme, plan))


def plan_query(op, is_f64, B, N, bc, scheme=0) -> int:
    return int(_lib.burgers_plan_query(op, int(bool(is_f64)), B, N, bc, scheme))


def launch_count(op, is_f64, B, N, bc, scheme=0, plan=PLAN_AUTO, tblock=0, n_steps=0) -> int:
    return int(_lib.burgers_launch_count(op, int(bool(is_f64)), B, N, bc, scheme, plan, tblock, n_steps))


def _check(st, where):
    if st != OK:
        raise BurgersError(st, where)


# ------------------------------------------------------------------ device (torch) entry points
def _dev(t, name, dtype=None):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA torch tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"{name} must have dtype {dtype}")
    return t


def _sfx(t):
    import torch
    if t.dtype == torch.float32:
        return "f32"
    if t.dtype == torch.float64:
        return "f64"
    raise TypeError("u must be float32 or float64")


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _shape(u):
    if u.dim() == 1:
        return 1, u.shape[0]
    if u.dim() != 2:
        raise ValueError("u must be [B][N] or [N]")
    return u.shape[0], u.shape[1]


def _check_vecs(B, **vecs):
    """Every per-trajectory array (nu, dt, iters_out, ...) must hold exactly B elements: a short one would be
    read or written out of bounds on the device."""
    for name, t in vecs.items():
        if t is not None and t.numel() != B:
            raise ValueError(f"{name} must have length B = {B}, got {t.numel()}")


def _ws(ws, need, device):
    import torch
    if need == 0:
        return None, 0, ws
    if ws is None:
        ws = torch.empty(need, dtype=torch.uint8, device=device)
    _dev(ws, "ws")
    return ctypes.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size(), ws


def alloc_workspace(op, u, bc, scheme=0, plan=PLAN_AUTO):
    """A uint8 CUDA tensor big enough for `op` on `u` (None when no scratch is needed)."""
    import torch
    B, N = _shape(u)
    need = workspace_bytes(op, u.dtype == torch.float64, B, N, bc, scheme, plan)
    return torch.empty(need, dtype=torch.uint8, device=u.device) if need else None


def burgers_explicit(u, L, nu, dt, n_steps, bc, scheme, ws=None, plan=PLAN_AUTO, tblock=0, ppt=0):
    """In-place explicit time stepping of u [B][N] (include/burgers.h: burgers_explicit_*)."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    need = workspace_bytes(OP_EXPLICIT, u.dtype == torch.float64, B, N, bc, scheme, plan)
    wsp, wsb, ws = _ws(ws, need, u.device)
    fn = getattr(_lib, f"burgers_explicit_plan_{sfx}")
    st = fn(u.data_ptr(), B, N, float(L), nu.data_ptr(), dt.data_ptr(), int(n_steps), int(bc),
            int(scheme), int(plan), int(tblock), int(ppt), wsp, wsb, _stream())
    _check(st, f"burgers_explicit_{sfx}")
    return u


def burgers_explicit_traj(u, L, nu, dt, n_steps, bc, scheme, snap_every, snaps=None, ws=None):
    """Explicit time stepping with trajectory output (include/burgers.h: burgers_explicit_traj_*).
    Returns (u, snaps) with snaps [n_steps // snap_every][B][N]."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    ns = int(n_steps) // int(snap_every) if snap_every >= 1 else 0
    if snaps is None:
        snaps = torch.empty((max(ns, 1), B, N), dtype=u.dtype, device=u.device)
    _dev(snaps, "snaps", u.dtype)
    if snaps.numel() < ns * B * N:
        raise ValueError("snaps is too small")
    need = workspace_bytes(OP_EXPLICIT, u.dtype == torch.float64, B, N, bc, scheme)
    wsp, wsb, ws = _ws(ws, need, u.device)
    st = getattr(_lib, f"burgers_explicit_traj_{sfx}")(u.data_ptr(), B, N, float(L), nu.data_ptr(), dt.data_ptr(),
                                                       int(n_steps), int(bc), int(scheme), int(snap_every),
                                                       snaps.data_ptr(), wsp, wsb, _stream())
    _check(st, f"burgers_explicit_traj_{sfx}")
    return u, snaps[:ns]


def burgers_explicit_adaptive(u, L, nu, C, n_outer, m_steps, bc, scheme, ws=None):
    """Explicit stepping with the CFL time step recomputed every m_steps steps (include/burgers.h:
    burgers_explicit_adaptive_*).  Returns (u, t, dt_last): t = simulated time per trajectory (float64)."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu)
    dt = torch.empty(B, dtype=u.dtype, device=u.device)
    t = torch.zeros(B, dtype=torch.float64, device=u.device)
    need = workspace_bytes(OP_EXPLICIT, u.dtype == torch.float64, B, N, bc, scheme)
    wsp, wsb, ws = _ws(ws, need, u.device)
    st = getattr(_lib, f"burgers_explicit_adaptive_{sfx}")(u.data_ptr(), B, N, float(L), nu.data_ptr(), float(C),
                                                           int(n_outer), int(m_steps), int(bc), int(scheme),
                                                           dt.data_ptr(), t.data_ptr(), wsp, wsb, _stream())
    _check(st, f"burgers_explicit_adaptive_{sfx}")
    return u, t, dt


def burgers_explicit_adjoint(u0, lam, L, nu, dt, n_steps, bc, ws=None, segment=0, scheme=SCHEME_EULER):
    """lam <- (du^N/du^0)^T lam for n_steps forward-Euler or RK4 steps from u0 (include/burgers.h:
    burgers_explicit_adjoint_scheme_*; segment = checkpoint interval, 0 = automatic); u0 is not modified."""
    import torch
    _dev(u0, "u0"); sfx = _sfx(u0)
    _dev(lam, "lam", u0.dtype); _dev(nu, "nu", u0.dtype); _dev(dt, "dt", u0.dtype)
    B, N = _shape(u0)
    _check_vecs(B, nu=nu, dt=dt)
    if lam.numel() != u0.numel():
        raise ValueError("lam must have the shape of u0")
    need = int(_lib.burgers_adjoint_scheme_workspace_bytes(int(u0.dtype == torch.float64), B, N, int(bc), int(scheme),
                                                           int(n_steps), int(segment)))
    wsp, wsb, ws = _ws(ws, need, u0.device)
    st = getattr(_lib, f"burgers_explicit_adjoint_scheme_{sfx}")(u0.data_ptr(), lam.data_ptr(), B, N, float(L),
                                                                 nu.data_ptr(), dt.data_ptr(), int(n_steps), int(bc),
                                                                 int(scheme), int(segment), wsp, wsb, _stream())
    _check(st, f"burgers_explicit_adjoint_{sfx}")
    return lam


def burgers_btcs_adjoint(u0, lam, L, nu, dt, n_steps, bc, ws=None, segment=0):
    """lam <- (du^N/du^0)^T lam for n_steps BTCS steps from u0 (include/burgers.h: burgers_btcs_adjoint_ckpt_*;
    segment = 0: automatic checkpointing)."""
    import torch
    _dev(u0, "u0"); sfx = _sfx(u0)
    _dev(lam, "lam", u0.dtype); _dev(nu, "nu", u0.dtype); _dev(dt, "dt", u0.dtype)
    B, N = _shape(u0)
    _check_vecs(B, nu=nu, dt=dt)
    if lam.numel() != u0.numel():
        raise ValueError("lam must have the shape of u0")
    need = int(_lib.burgers_implicit_adjoint_ckpt_workspace_bytes(OP_BTCS, int(u0.dtype == torch.float64), B, N, int(bc),
                                                                  int(n_steps), int(segment)))
    wsp, wsb, ws = _ws(ws, need, u0.device)
    st = getattr(_lib, f"burgers_btcs_adjoint_ckpt_{sfx}")(u0.data_ptr(), lam.data_ptr(), B, N, float(L), nu.data_ptr(),
                                                           dt.data_ptr(), int(n_steps), int(bc), int(segment), wsp, wsb,
                                                           _stream())
    _check(st, f"burgers_btcs_adjoint_{sfx}")
    return lam


def burgers_newton_adjoint(u0, lam, L, nu, dt, n_steps, bc, theta=1.0, tol=1e-13, max_iter=50, ws=None, segment=0):
    """lam <- (du^N/du^0)^T lam for n_steps Newton / theta-scheme steps from u0 (include/burgers.h:
    burgers_newton_adjoint_*; the forward sweep is iterated to tol)."""
    import torch
    _dev(u0, "u0"); sfx = _sfx(u0)
    _dev(lam, "lam", u0.dtype); _dev(nu, "nu", u0.dtype); _dev(dt, "dt", u0.dtype)
    B, N = _shape(u0)
    _check_vecs(B, nu=nu, dt=dt)
    if lam.numel() != u0.numel():
        raise ValueError("lam must have the shape of u0")
    need = int(_lib.burgers_implicit_adjoint_ckpt_workspace_bytes(OP_NEWTON, int(u0.dtype == torch.float64), B, N, int(bc),
                                                                  int(n_steps), int(segment)))
    wsp, wsb, ws = _ws(ws, need, u0.device)
    st = getattr(_lib, f"burgers_newton_adjoint_ckpt_{sfx}")(u0.data_ptr(), lam.data_ptr(), B, N, float(L), nu.data_ptr(),
                                                             dt.data_ptr(), int(n_steps), int(bc), float(theta), float(tol),
                                                             int(max_iter), int(segment), wsp, wsb, _stream())
    _check(st, f"burgers_newton_adjoint_{sfx}")
    return lam


def burgers_btcs_traj(u, L, nu, dt, n_steps, bc, snap_every, snaps=None, ws=None):
    """BTCS time stepping with trajectory output (include/burgers.h: burgers_btcs_traj_*)."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    ns = int(n_steps) // int(snap_every) if snap_every >= 1 else 0
    if snaps is None:
        snaps = torch.empty((max(ns, 1), B, N), dtype=u.dtype, device=u.device)
    _dev(snaps, "snaps", u.dtype)
    if snaps.numel() < ns * B * N:
        raise ValueError("snaps is too small")
    need = workspace_bytes(OP_BTCS, u.dtype == torch.float64, B, N, bc, 0)
    wsp, wsb, ws = _ws(ws, need, u.device)
    st = getattr(_lib, f"burgers_btcs_traj_{sfx}")(u.data_ptr(), B, N, float(L), nu.data_ptr(), dt.data_ptr(),
                                                   int(n_steps), int(bc), int(snap_every), snaps.data_ptr(),
                                                   wsp, wsb, _stream())
    _check(st, f"burgers_btcs_traj_{sfx}")
    return u, snaps[:ns]


def burgers_btcs(u, L, nu, dt, n_steps, bc, ws=None, plan=PLAN_AUTO):
    """In-place BTCS time stepping of u [B][N] (include/burgers.h: burgers_btcs_*)."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    need = workspace_bytes(OP_BTCS, u.dtype == torch.float64, B, N, bc, 0, plan)
    wsp, wsb, ws = _ws(ws, need, u.device)
    fn = getattr(_lib, f"burgers_btcs_plan_{sfx}")
    st = fn(u.data_ptr(), B, N, float(L), nu.data_ptr(), dt.data_ptr(), int(n_steps), int(bc),
            int(plan), wsp, wsb, _stream())
    _check(st, f"burgers_btcs_{sfx}")
    return u


def noalloc_scratch_bytes() -> int:
    return int(_lib.burgers_noalloc_scratch_bytes())


def burgers_btcs_noalloc(u, L, nu, dt, n_steps, bc):
    """In-place BTCS time stepping with the library's built-in scratch array: no allocation anywhere
    (include/burgers.h: burgers_btcs_noalloc; BurgersError(ERR_LIMIT) beyond noalloc_scratch_bytes())."""
    import torch
    _dev(u, "u")
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    st = _lib.burgers_btcs_noalloc(int(u.dtype == torch.float64), u.data_ptr(), B, N, float(L), nu.data_ptr(),
                                   dt.data_ptr(), int(n_steps), int(bc), _stream())
    _check(st, "burgers_btcs_noalloc")
    return u


def burgers_btcs_gs(u, L, nu, dt, n_steps, bc, tol=1e-6, max_iter=1000, iters_out=None, ws=None):
    """In-place BTCS with a Gauss-Seidel inner solver (include/burgers.h: burgers_btcs_gs_*)."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    ip = None
    if iters_out is not None:
        _dev(iters_out, "iters_out", torch.int64)
        _check_vecs(B, iters_out=iters_out)
        ip = ctypes.c_void_p(iters_out.data_ptr())
    need = workspace_bytes(OP_GS, u.dtype == torch.float64, B, N, bc)
    wsp, wsb, ws = _ws(ws, need, u.device)
    st = getattr(_lib, f"burgers_btcs_gs_{sfx}")(u.data_ptr(), B, N, float(L), nu.data_ptr(), dt.data_ptr(),
                                                 int(n_steps), int(bc), float(tol), int(max_iter), ip, wsp, wsb,
                                                 _stream())
    _check(st, f"burgers_btcs_gs_{sfx}")
    return u


def burgers_newton(u, L, nu, dt, n_steps, bc, tol=1e-6, max_iter=50, iters_out=None, ws=None, plan=PLAN_AUTO,
                   theta=1.0):
    """In-place implicit central-convection theta-scheme by Newton-Raphson (include/burgers.h:
    burgers_newton_*; theta = 1: the paper's BTCS Eq.11, 1/2: Crank-Nicolson).  iters_out: optional
    int64 CUDA tensor [B] receiving the iteration totals."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    ip = None
    if iters_out is not None:
        _dev(iters_out, "iters_out", torch.int64)
        _check_vecs(B, iters_out=iters_out)
        ip = ctypes.c_void_p(iters_out.data_ptr())
    need = workspace_bytes(OP_NEWTON, u.dtype == torch.float64, B, N, bc, 0, plan)
    wsp, wsb, ws = _ws(ws, need, u.device)
    st = getattr(_lib, f"burgers_newton_{sfx}")(u.data_ptr(), B, N, float(L), nu.data_ptr(), dt.data_ptr(),
                                                int(n_steps), int(bc), float(theta), float(tol), int(max_iter), ip,
                                                int(plan), wsp, wsb, _stream())
    _check(st, f"burgers_newton_{sfx}")
    return u


def burgers_newton_traj(u, L, nu, dt, n_steps, bc, snap_every, tol=1e-6, max_iter=50, iters_out=None, snaps=None, ws=None,
                        theta=1.0):
    """Newton / theta-scheme stepping with trajectory output (include/burgers.h: burgers_newton_traj_*).
    Returns (u, snaps) with snaps [n_steps // snap_every][B][N]."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype); _dev(dt, "dt", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu, dt=dt)
    ns = int(n_steps) // int(snap_every) if snap_every >= 1 else 0
    if snaps is None:
        snaps = torch.empty((max(ns, 1), B, N), dtype=u.dtype, device=u.device)
    _dev(snaps, "snaps", u.dtype)
    if snaps.numel() < ns * B * N:
        raise ValueError("snaps is too small")
    ip = None
    if iters_out is not None:
        _dev(iters_out, "iters_out", torch.int64)
        _check_vecs(B, iters_out=iters_out)
        ip = ctypes.c_void_p(iters_out.data_ptr())
    need = workspace_bytes(OP_NEWTON, u.dtype == torch.float64, B, N, bc)
    wsp, wsb, ws = _ws(ws, need, u.device)
    st = getattr(_lib, f"burgers_newton_traj_{sfx}")(u.data_ptr(), B, N, float(L), nu.data_ptr(), dt.data_ptr(),
                                                     int(n_steps), int(bc), float(theta), float(tol), int(max_iter), ip,
                                                     int(snap_every), snaps.data_ptr(), wsp, wsb, _stream())
    _check(st, f"burgers_newton_traj_{sfx}")
    return u, snaps[:ns]


def dt_from_cfl(u, L, nu, C, bc, out=None):
    """dt[b] = C min(dx/max|u_b|, dx^2/(2 nu_b)) (include/burgers.h: dt_from_cfl_*)."""
    import torch
    _dev(u, "u"); sfx = _sfx(u)
    _dev(nu, "nu", u.dtype)
    B, N = _shape(u)
    _check_vecs(B, nu=nu)
    if out is None:
        out = torch.empty(B, dtype=u.dtype, device=u.device)
    _dev(out, "out", u.dtype)
    st = getattr(_lib, f"dt_from_cfl_{sfx}")(u.data_ptr(), B, N, float(L), nu.data_ptr(), float(C),
                                             int(bc), out.data_ptr(), _stream())
    _check(st, f"dt_from_cfl_{sfx}")
    return out


PEAK_KINDS = ("ffma_chain", "ffma_3reg", "fadd_2reg", "dfma_chain", "dfma_3reg", "dadd_2reg", "dfma_select_mix")


def pipe_peak(kind, iters, sink):
    """One launch of the FP-pipe micro-benchmark `kind` (index into PEAK_KINDS) on the current stream
    (include/burgers.h: burgers_pipe_peak); returns the lane-instructions it executes.  The caller times it."""
    _dev(sink, "sink")
    n = ctypes.c_double(0.0)
    _check(_lib.burgers_pipe_peak(int(kind), int(iters), sink.data_ptr(), _stream(), ctypes.byref(n)),
           "burgers_pipe_peak")
    return n.value


# ------------------------------------------------------------------ host (numpy) entry points
def _host(a, name, dtype=None):
    if not isinstance(a, np.ndarray) or not a.flags.c_contiguous:
        raise TypeError(f"{name} must be a C-contiguous numpy array")
    if dtype is not None and a.dtype != dtype:
        raise TypeError(f"{name} must have dtype {dtype}")
    return a


def _hshape(u, **vecs):
    B, N = (1, u.shape[0]) if u.ndim == 1 else u.shape
    for name, a in vecs.items():
        if a.size != B:
            raise ValueError(f"{name} must have length B = {B}, got {a.size}")
    return B, N


def _hsfx(a):
    if a.dtype == np.float32:
        return "f32"
    if a.dtype == np.float64:
        return "f64"
    raise TypeError("u must be float32 or float64")


def burgers_explicit_host(u, L, nu, dt, n_steps, bc, scheme):
    """Host-buffer explicit stepping: u (numpy, [B][N]) is updated in place."""
    _host(u, "u"); sfx = _hsfx(u); _host(nu, "nu", u.dtype); _host(dt, "dt", u.dtype)
    B, N = _hshape(u, nu=nu, dt=dt)
    st = getattr(_lib, f"burgers_explicit_host_{sfx}")(u.ctypes.data, B, N, float(L), nu.ctypes.data,
                                                       dt.ctypes.data, int(n_steps), int(bc), int(scheme))
    _check(st, f"burgers_explicit_host_{sfx}")
    return u


def burgers_btcs_host(u, L, nu, dt, n_steps, bc):
    _host(u, "u"); sfx = _hsfx(u); _host(nu, "nu", u.dtype); _host(dt, "dt", u.dtype)
    B, N = _hshape(u, nu=nu, dt=dt)
    st = getattr(_lib, f"burgers_btcs_host_{sfx}")(u.ctypes.data, B, N, float(L), nu.ctypes.data,
                                                   dt.ctypes.data, int(n_steps), int(bc))
    _check(st, f"burgers_btcs_host_{sfx}")
    return u


def burgers_solve_host(u, L, nu, C, n_steps, bc, op=OP_EXPLICIT, scheme=0, return_dt=False):
    """The whole hot path on host buffers in one call (include/burgers.h: burgers_solve_host_*): dt from the
    CFL number C on the device, then n_steps of the explicit scheme or of BTCS; u is updated in place."""
    _host(u, "u"); sfx = _hsfx(u); _host(nu, "nu", u.dtype)
    B, N = _hshape(u, nu=nu)
    dt = np.empty(B, dtype=u.dtype) if return_dt else None
    st = getattr(_lib, f"burgers_solve_host_{sfx}")(u.ctypes.data, B, N, float(L), nu.ctypes.data, float(C),
                                                    int(n_steps), int(bc), int(op), int(scheme),
                                                    dt.ctypes.data if return_dt else None)
    _check(st, f"burgers_solve_host_{sfx}")
    return (u, dt) if return_dt else u


def burgers_newton_host(u, L, nu, dt, n_steps, bc, tol=1e-6, max_iter=50, return_iters=False, theta=1.0):
    _host(u, "u"); sfx = _hsfx(u); _host(nu, "nu", u.dtype); _host(dt, "dt", u.dtype)
    B, N = _hshape(u, nu=nu, dt=dt)
    iters = np.zeros(B, dtype=np.int64)
    st = getattr(_lib, f"burgers_newton_host_{sfx}")(u.ctypes.data, B, N, float(L), nu.ctypes.data, dt.ctypes.data,
                                                     int(n_steps), int(bc), float(theta), float(tol), int(max_iter),
                                                     iters.ctypes.data)
    _check(st, f"burgers_newton_host_{sfx}")
    return (u, iters) if return_iters else u


def dt_from_cfl_host(u, L, nu, C, bc):
    _host(u, "u"); sfx = _hsfx(u); _host(nu, "nu", u.dtype)
    B, N = _hshape(u, nu=nu)
    out = np.empty(B, dtype=u.dtype)
    st = getattr(_lib, f"dt_from_cfl_host_{sfx}")(u.ctypes.data, B, N, float(L), nu.ctypes.data, float(C),
                                                  int(bc), out.ctypes.data)
    _check(st, f"dt_from_cfl_host_{sfx}")
    return out
