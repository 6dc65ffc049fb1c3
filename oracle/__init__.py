"""CPU oracle for the Burgers hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front-end of ``oracle/burgers_oracle.c`` (plain scalar fp64 C restating
PAPER.md Eq.1-8, 21-24 in the readings listed in DESIGN.md).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; the product
(``paper_2601_12204_b200``) never does and shares no code with it.

All functions take and return fp64 numpy arrays.  For fp32 workloads the caller
rounds the inputs (u0, nu, dt) to fp32 first and widens them again, so that
both sides see identical input values.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "burgers_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

PERIODIC, DIRICHLET = 0, 1
EULER, RK4 = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no FMA contraction, OpenMP)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
           "-shared", "-std=c11", "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    i64, f64, ci = ctypes.c_int64, ctypes.c_double, ctypes.c_int
    p = ctypes.c_void_p
    lib.oracle_rhs.argtypes = [p, p, i64, f64, f64, ci, ci, f64]
    lib.oracle_rhs.restype = None
    lib.oracle_explicit.argtypes = [p, i64, i64, f64, p, p, i64, ci, ci, ci, f64, ci]
    lib.oracle_explicit.restype = ci
    lib.oracle_explicit_long.argtypes = [p, i64, f64, f64, f64, i64, ci, ci]
    lib.oracle_explicit_long.restype = ci
    lib.oracle_btcs_rows.argtypes = [p, i64, f64, f64, f64, ci, ci, f64, p, p, p, p]
    lib.oracle_btcs_rows.restype = None
    lib.oracle_thomas.argtypes = [i64, p, p, p, p, p]
    lib.oracle_thomas.restype = ci
    lib.oracle_cyclic.argtypes = [i64, p, p, p, p, p]
    lib.oracle_cyclic.restype = ci
    lib.oracle_btcs.argtypes = [p, i64, i64, f64, p, p, i64, ci, ci, f64, ci]
    lib.oracle_btcs.restype = ci
    lib.oracle_dt_from_cfl.argtypes = [p, i64, i64, f64, p, f64, ci, p]
    lib.oracle_dt_from_cfl.restype = ci
    lib.oracle_newton_residual.argtypes = [p, p, i64, f64, f64, f64, f64, ci, ci, f64, p]
    lib.oracle_newton_residual.restype = None
    lib.oracle_newton_jacobian.argtypes = [p, i64, f64, f64, f64, f64, ci, ci, f64, p, p, p]
    lib.oracle_newton_jacobian.restype = None
    lib.oracle_newton_btcs.argtypes = [p, i64, i64, f64, p, p, f64, i64, ci, f64, ci, ci, f64, p, ci]
    lib.oracle_newton_btcs.restype = ci
    lib.oracle_btcs_gs.argtypes = [p, i64, i64, f64, p, p, i64, ci, f64, ci, ci, f64, p, ci]
    lib.oracle_btcs_gs.restype = ci
    lib.oracle_explicit_adjoint.argtypes = [p, p, i64, i64, f64, p, p, i64, ci, ci, f64, ci]
    lib.oracle_explicit_adjoint.restype = ci
    lib.oracle_rk4_adjoint.argtypes = [p, p, i64, i64, f64, p, p, i64, ci, ci, f64, ci]
    lib.oracle_rk4_adjoint.restype = ci
    lib.oracle_btcs_adjoint.argtypes = [p, p, i64, i64, f64, p, p, i64, ci, ci, f64, ci]
    lib.oracle_btcs_adjoint.restype = ci
    lib.oracle_newton_adjoint.argtypes = [p, p, i64, i64, f64, p, p, f64, i64, ci, f64, ci, ci, f64, ci]
    lib.oracle_newton_adjoint.restype = ci
    lib.oracle_max_threads.argtypes = []
    lib.oracle_max_threads.restype = ci
    _lib = lib
    return lib


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data)


def _per_traj(x, B) -> np.ndarray:
    a = _f64(x).reshape(-1)
    if a.size == 1 and B != 1:
        a = np.full(B, float(a[0]))
    if a.size != B:
        raise ValueError("per-trajectory array must have length B")
    return np.ascontiguousarray(a)


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def default_threads() -> int:
    return max(1, min(max_threads(), os.cpu_count() or 1))


def rhs(u, L, nu, bc, adv=None) -> np.ndarray:
    """F(u) of one trajectory (D2)."""
    u = _f64(u).reshape(-1)
    F = np.empty_like(u)
    _load().oracle_rhs(_ptr(u), _ptr(F), u.size, float(L), float(nu), int(bc),
                       int(adv is not None), float(adv or 0.0))
    return F


def explicit(u0, L, nu, dt, n_steps, bc, scheme, adv=None, threads=None) -> np.ndarray:
    """Explicit time stepping (D3); u0 is [B][N] (or [N]); returns a new array."""
    u = _f64(u0).copy()
    shape = u.shape
    u = u.reshape(-1, shape[-1])
    B, N = u.shape
    nu_a, dt_a = _per_traj(nu, B), _per_traj(dt, B)
    rc = _load().oracle_explicit(_ptr(u), B, N, float(L), _ptr(nu_a), _ptr(dt_a),
                                 int(n_steps), int(bc), int(scheme),
                                 int(adv is not None), float(adv or 0.0),
                                 int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_explicit: bad arguments")
    return u.reshape(shape)


def explicit_long(u0, L, nu, dt, n_steps, bc, threads=None) -> np.ndarray:
    """Forward Euler on one long grid, spatial loop split over threads."""
    u = _f64(u0).reshape(-1).copy()
    rc = _load().oracle_explicit_long(_ptr(u), u.size, float(L), float(nu), float(dt),
                                      int(n_steps), int(bc),
                                      int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_explicit_long: bad arguments")
    return u


def btcs_rows(u, L, nu, dt, bc, adv=None):
    """(sub, diag, sup, rhs) of the BTCS system assembled from u^n (D4)."""
    u = _f64(u).reshape(-1)
    out = [np.empty_like(u) for _ in range(4)]
    _load().oracle_btcs_rows(_ptr(u), u.size, float(L), float(nu), float(dt), int(bc),
                             int(adv is not None), float(adv or 0.0),
                             *[_ptr(o) for o in out])
    return tuple(out)


def thomas(sub, diag, sup, rhs) -> np.ndarray:
    sub, diag, sup, rhs = map(_f64, (sub, diag, sup, rhs))
    x = np.empty_like(rhs)
    if _load().oracle_thomas(rhs.size, _ptr(sub), _ptr(diag), _ptr(sup), _ptr(rhs),
                             _ptr(x)) != 0:
        raise MemoryError
    return x


def cyclic(sub, diag, sup, rhs) -> np.ndarray:
    sub, diag, sup, rhs = map(_f64, (sub, diag, sup, rhs))
    x = np.empty_like(rhs)
    if _load().oracle_cyclic(rhs.size, _ptr(sub), _ptr(diag), _ptr(sup), _ptr(rhs),
                             _ptr(x)) != 0:
        raise MemoryError
    return x


def btcs(u0, L, nu, dt, n_steps, bc, adv=None, threads=None) -> np.ndarray:
    """BTCS time stepping (D4-D7); returns a new array."""
    u = _f64(u0).copy()
    shape = u.shape
    u = u.reshape(-1, shape[-1])
    B, N = u.shape
    nu_a, dt_a = _per_traj(nu, B), _per_traj(dt, B)
    rc = _load().oracle_btcs(_ptr(u), B, N, float(L), _ptr(nu_a), _ptr(dt_a),
                             int(n_steps), int(bc), int(adv is not None),
                             float(adv or 0.0), int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_btcs: bad arguments")
    return u.reshape(shape)


def dt_from_cfl(u, L, nu, C, bc) -> np.ndarray:
    """dt_b = C min(dx/max|u_b|, dx^2/(2 nu_b)) (D8)."""
    u = _f64(u)
    u2 = u.reshape(-1, u.shape[-1])
    B, N = u2.shape
    nu_a = _per_traj(nu, B)
    out = np.empty(B, dtype=np.float64)
    rc = _load().oracle_dt_from_cfl(_ptr(u2), B, N, float(L), _ptr(nu_a), float(C),
                                    int(bc), _ptr(out))
    if rc != 0:
        raise ValueError("oracle_dt_from_cfl: bad arguments")
    return out


def newton_residual(w, un, L, nu, dt, bc, adv=None, theta=1.0) -> np.ndarray:
    """Residual F(w) of Eq.11 (theta-weighted, D11) for one trajectory."""
    w, un = _f64(w).reshape(-1), _f64(un).reshape(-1)
    F = np.empty_like(w)
    _load().oracle_newton_residual(_ptr(w), _ptr(un), w.size, float(L), float(nu), float(dt), float(theta), int(bc),
                                   int(adv is not None), float(adv or 0.0), _ptr(F))
    return F


def newton_jacobian(w, L, nu, dt, bc, adv=None, theta=1.0):
    """(sub, diag, sup) of the tridiagonal Jacobian of Eq.11 at w (D11)."""
    w = _f64(w).reshape(-1)
    out = [np.empty_like(w) for _ in range(3)]
    _load().oracle_newton_jacobian(_ptr(w), w.size, float(L), float(nu), float(dt), float(theta), int(bc),
                                   int(adv is not None), float(adv or 0.0), *[_ptr(o) for o in out])
    return tuple(out)


def newton_btcs(u0, L, nu, dt, n_steps, bc, tol=1e-6, max_iter=50, adv=None, threads=None,
                return_iters=False, theta=1.0):
    """Implicit central-convection theta-scheme by Newton-Raphson (D11; theta = 1: the paper's BTCS
    Eq.11, theta = 1/2: Crank-Nicolson); returns a new array (and the per-trajectory iteration
    totals when return_iters)."""
    u = _f64(u0).copy()
    shape = u.shape
    u = u.reshape(-1, shape[-1])
    B, N = u.shape
    nu_a, dt_a = _per_traj(nu, B), _per_traj(dt, B)
    iters = np.zeros(B, dtype=np.int64)
    rc = _load().oracle_newton_btcs(_ptr(u), B, N, float(L), _ptr(nu_a), _ptr(dt_a), float(theta), int(n_steps),
                                    int(bc), float(tol), int(max_iter), int(adv is not None),
                                    float(adv or 0.0), ctypes.c_void_p(iters.ctypes.data),
                                    int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_newton_btcs: bad arguments")
    return (u.reshape(shape), iters) if return_iters else u.reshape(shape)


def explicit_trajectory(u0, L, nu, dt, n_steps, bc, scheme, snap_every, threads=None):
    """Snapshots of explicit time stepping after every snap_every-th step: [n_steps // snap_every][B][N]
    plus the final state.  Plain composition of `explicit` calls (p then q steps == p+q steps, bitwise:
    pinned by tests/test_oracle_pins.py::test_steps_compose_bitwise)."""
    u = _f64(u0).copy()
    snaps = []
    done = 0
    while done + snap_every <= n_steps:
        u = explicit(u, L, nu, dt, snap_every, bc, scheme, threads=threads)
        snaps.append(u.copy())
        done += snap_every
    if done < n_steps:
        u = explicit(u, L, nu, dt, n_steps - done, bc, scheme, threads=threads)
    return u, (np.stack(snaps) if snaps else np.empty((0,) + u.shape))


def btcs_gs(u0, L, nu, dt, n_steps, bc, tol=1e-6, max_iter=1000, adv=None, threads=None, return_iters=False):
    """BTCS (D4) with the linear system solved by lexicographic Gauss-Seidel sweeps to max residual
    < tol (D12); returns a new array (and the per-trajectory sweep totals)."""
    u = _f64(u0).copy()
    shape = u.shape
    u = u.reshape(-1, shape[-1])
    B, N = u.shape
    nu_a, dt_a = _per_traj(nu, B), _per_traj(dt, B)
    iters = np.zeros(B, dtype=np.int64)
    rc = _load().oracle_btcs_gs(_ptr(u), B, N, float(L), _ptr(nu_a), _ptr(dt_a), int(n_steps), int(bc),
                                float(tol), int(max_iter), int(adv is not None), float(adv or 0.0),
                                ctypes.c_void_p(iters.ctypes.data), int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_btcs_gs: bad arguments")
    return (u.reshape(shape), iters) if return_iters else u.reshape(shape)


def explicit_adaptive(u0, L, nu, C, n_outer, m_steps, bc, scheme, dtype=np.float64, threads=None):
    """n_outer times { dt = dt_from_cfl(u) rounded to `dtype`; m_steps explicit steps with it }: plain
    composition of the pinned `dt_from_cfl` and `explicit`.  Returns (u, t) with t = sum m_steps*dt."""
    u = _f64(u0).copy()
    u2 = u.reshape(-1, u.shape[-1])
    t = np.zeros(u2.shape[0])
    for _ in range(n_outer):
        dt = dt_from_cfl(u2.astype(dtype).astype(np.float64) if dtype != np.float64 else u2, L, nu, C, bc)
        dt = dt.astype(dtype).astype(np.float64)
        u2 = explicit(u2, L, nu, dt, m_steps, bc, scheme, threads=threads)
        t += m_steps * dt
    return u2.reshape(u.shape), t


def btcs_adjoint(u0, lam_T, L, nu, dt, n_steps, bc, adv=None, threads=None) -> np.ndarray:
    """Discrete adjoint of n_steps lagged-upwind BTCS steps (D15): dJ/du^0 from lam_T = dJ/du^N."""
    u = _f64(u0)
    shape = u.shape
    u = np.ascontiguousarray(u.reshape(-1, shape[-1]))
    lam = np.ascontiguousarray(_f64(lam_T).reshape(u.shape).copy())
    B, N = u.shape
    nu_a, dt_a = _per_traj(nu, B), _per_traj(dt, B)
    rc = _load().oracle_btcs_adjoint(_ptr(u), _ptr(lam), B, N, float(L), _ptr(nu_a), _ptr(dt_a), int(n_steps),
                                     int(bc), int(adv is not None), float(adv or 0.0), int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_btcs_adjoint: bad arguments")
    return lam.reshape(shape)


def newton_adjoint(u0, lam_T, L, nu, dt, n_steps, bc, tol=1e-13, max_iter=50, adv=None, threads=None,
                   theta=1.0) -> np.ndarray:
    """Reverse mode of n_steps Newton / theta-scheme steps (D16; implicit-function theorem at the converged
    states): dJ/du^0 from lam_T = dJ/du^N."""
    u = _f64(u0)
    shape = u.shape
    u = np.ascontiguousarray(u.reshape(-1, shape[-1]))
    lam = np.ascontiguousarray(_f64(lam_T).reshape(u.shape).copy())
    B, N = u.shape
    nu_a, dt_a = _per_traj(nu, B), _per_traj(dt, B)
    rc = _load().oracle_newton_adjoint(_ptr(u), _ptr(lam), B, N, float(L), _ptr(nu_a), _ptr(dt_a), float(theta),
                                       int(n_steps), int(bc), float(tol), int(max_iter), int(adv is not None),
                                       float(adv or 0.0), int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_newton_adjoint: bad arguments")
    return lam.reshape(shape)


def explicit_adjoint(u0, lam_T, L, nu, dt, n_steps, bc, adv=None, threads=None, scheme=EULER) -> np.ndarray:
    """Discrete adjoint of n_steps forward-Euler (D13) or classical RK4 (D14) steps: dJ/du^0 from
    lam_T = dJ/du^N."""
    u = _f64(u0)
    shape = u.shape
    u = np.ascontiguousarray(u.reshape(-1, shape[-1]))
    lam = np.ascontiguousarray(_f64(lam_T).reshape(u.shape).copy())
    B, N = u.shape
    nu_a, dt_a = _per_traj(nu, B), _per_traj(dt, B)
    fn = _load().oracle_explicit_adjoint if scheme == EULER else _load().oracle_rk4_adjoint
    rc = fn(_ptr(u), _ptr(lam), B, N, float(L), _ptr(nu_a), _ptr(dt_a), int(n_steps),
            int(bc), int(adv is not None), float(adv or 0.0), int(threads or default_threads()))
    if rc != 0:
        raise ValueError("oracle_explicit_adjoint: bad arguments")
    return lam.reshape(shape)
