"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (AUTO plan,
dt from the library's own dt_from_cfl, one call for all n_steps).

The oracle cannot run the full configs in seconds, so it checks SAMPLED outputs it can compute one
by one, exactly:
  - batched configs (C2, C3, C5): trajectories are independent, so the oracle runs a seeded sample
    of whole trajectories (all steps) and every point of those is compared;
  - single long grids (C4a, C4b): the oracle runs WINDOWS of the grid.  Explicit Euler has a
    numerical domain of dependence of exactly one cell per step, so the central part of a window
    with a margin of n_steps cells is exact whatever is done at the window ends.  BTCS couples all
    points, but the influence of a point decays per cell like lam = ((1+2r) - sqrt(1+4r)) / (2r)
    per step (Green's function of the diffusion part; convection only strengthens the diagonal):
    at r = 5, lam = 0.642, i.e. < 1e-12 beyond 63 cells per step, so a margin of 64*n_steps cells
    makes the window's centre exact to far below the 1e-10 tolerance;
the rows of SURVEY 8(f) that bench.py times (Newton / Crank-Nicolson and Gauss-Seidel on C3's inputs, C2 with
trajectory output, the checkpointed adjoint of the whole C2 run) are checked the same way at the end of the file;
plus properties that hold at any size, checked on ALL outputs: finiteness, the discrete maximum
principle (D4 / D9), frozen Dirichlet ends, and for BTCS the defining residual
A(u^n) u^{n+1} = u^n of the last step evaluated in fp64 numpy over the whole grid.
"""
import math

import numpy as np
import pytest

import oracle
from parity import TOL, rel_err, to_dev
from paper_2601_12204_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


def _gpu_pass(B, w, scheme):
    """One bench.py pass: dt_from_cfl then the time-stepping call (AUTO plan).  Returns (u, dt)."""
    u, nu = to_dev(w.u0.copy()), to_dev(w.nu)
    dt = B.dt_from_cfl(u, w.L, nu, w.cfl, w.bc)
    if scheme is None:
        B.burgers_btcs(u, w.L, nu, dt, w.n_steps, w.bc)
    else:
        B.burgers_explicit(u, w.L, nu, dt, w.n_steps, w.bc, scheme)
    return u.cpu().numpy(), dt.cpu().numpy()


def _check_dt(w, dt):
    ref = oracle.dt_from_cfl(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), w.cfl, w.bc).astype(w.dtype)
    assert np.all(np.abs(dt - ref) <= 2 * np.spacing(np.abs(ref)))


def _max_principle(got, u0, slack):
    assert np.all(np.isfinite(got))
    hi, lo = u0.max(axis=1).astype(np.float64), u0.min(axis=1).astype(np.float64)
    s = slack * np.abs(u0).max(axis=1).astype(np.float64)
    assert np.all(got.max(axis=1) <= hi + s) and np.all(got.min(axis=1) >= lo - s)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_c2_full(B, dtype):
    w = W.c2_dirichlet_batch(dtype=dtype)                          # B=1024, N=4096, 10 000 steps
    assert B.plan_query(B.OP_EXPLICIT, dtype == np.float64, w.B, w.N, w.bc, 0) == B.PLAN_RESIDENT
    got, dt = _gpu_pass(B, w, B.SCHEME_EULER)
    _check_dt(w, dt)
    rows = np.sort(np.random.default_rng(2).choice(w.B, 24, replace=False))
    rows[0], rows[-1] = 0, w.B - 1
    ref = oracle.explicit(w.u0[rows].astype(np.float64), w.L, w.nu[rows].astype(np.float64),
                          dt[rows].astype(np.float64), w.n_steps, w.bc, oracle.EULER)
    assert rel_err(got[rows], ref, w.u0[rows]) <= TOL[np.dtype(dtype)]
    np.testing.assert_array_equal(got[:, 0], w.u0[:, 0])
    np.testing.assert_array_equal(got[:, -1], w.u0[:, -1])
    _max_principle(got, w.u0, 1e-5 if dtype == np.float32 else 1e-12)   # |c| + 2r <= 0.8: monotone


def test_c3_full(B):
    w = W.c3_periodic_btcs()                                       # B=4096, N=2048, 1 000 steps
    assert B.plan_query(B.OP_BTCS, True, w.B, w.N, w.bc) == B.PLAN_HYBRID
    got, dt = _gpu_pass(B, w, None)
    _check_dt(w, dt)
    rows = np.sort(np.random.default_rng(3).choice(w.B, 24, replace=False))
    rows[0], rows[-1] = 0, w.B - 1
    ref = oracle.btcs(w.u0[rows], w.L, w.nu[rows], dt[rows], w.n_steps, w.bc)
    assert rel_err(got[rows], ref, w.u0[rows]) <= 1e-10
    _max_principle(got, w.u0, 1e-12)                               # M-matrix: any dt


def test_c5_full(B):
    w = W.c5_rk4_ensemble()                                        # B=65536, N=1024, 5 000 RK4 steps
    assert B.plan_query(B.OP_EXPLICIT, False, w.B, w.N, w.bc, 1) == B.PLAN_RESIDENT
    got, dt = _gpu_pass(B, w, B.SCHEME_RK4)
    _check_dt(w, dt)
    rows = np.arange(0, w.B, 4096)                                 # 16 trajectories
    rows[-1] = w.B - 1
    ref = oracle.explicit(w.u0[rows].astype(np.float64), w.L, w.nu[rows].astype(np.float64),
                          dt[rows].astype(np.float64), w.n_steps, w.bc, oracle.RK4)
    assert rel_err(got[rows], ref, w.u0[rows]) <= 1e-4
    assert np.all(np.isfinite(got))
    # RK4 is not monotone, but these pulses only decay: bounded by the initial range (+ rounding)
    _max_principle(got, w.u0, 1e-3)


def _window(u0_row, start, width):
    idx = (start + np.arange(width)) % u0_row.shape[0]
    return idx, u0_row[idx]


def test_c4a_full_windows(B):
    w = W.c4a_long_explicit()                                      # N=2^24, 2 000 Euler steps, fp32
    assert B.plan_query(B.OP_EXPLICIT, False, 1, w.N, w.bc, 0) == B.PLAN_TILED
    got, dt = _gpu_pass(B, w, B.SCHEME_EULER)
    _check_dt(w, dt)
    n, N = w.n_steps, w.N
    margin, width = n + 8, 1 << 16
    # the grid wrap, both smoothed steps, a tile boundary region and a flat part
    for start in (N - width // 2, N // 4 - width // 2, 3 * N // 4 - width // 2, 5 * 4064 * 100 - 77, N // 2):
        idx, win = _window(w.u0[0], start, width)
        # same dx as the full grid: Dirichlet window of `width` nodes has dx = Lw/(width-1)
        Lw = (w.L / N) * (width - 1)
        ref = oracle.explicit(win[None, :].astype(np.float64), Lw, w.nu.astype(np.float64),
                              dt.astype(np.float64), n, oracle.DIRICHLET, oracle.EULER)[0]
        c = slice(margin, width - margin)
        err = np.abs(got[0, idx[c]].astype(np.float64) - ref[c]).max() / np.abs(w.u0).max()
        assert err <= 1e-4, (start, err)
    _max_principle(got, w.u0, 1e-5)


def test_c4b_full_windows_and_residual(B):
    w = W.c4b_long_btcs()                                          # N=2^22, 200 BTCS steps, fp64
    assert B.plan_query(B.OP_BTCS, True, 1, w.N, w.bc) == B.PLAN_LONG
    u, nu = to_dev(w.u0.copy()), to_dev(w.nu)
    dt_d = B.dt_from_cfl(u, w.L, nu, w.cfl, w.bc)
    B.burgers_btcs(u, w.L, nu, dt_d, w.n_steps - 1, w.bc)
    prev = u.cpu().numpy()[0].copy()
    B.burgers_btcs(u, w.L, nu, dt_d, 1, w.bc)
    got = u.cpu().numpy()
    dt = dt_d.cpu().numpy()
    _check_dt(w, dt)
    # in one call too (the bench configuration): p then q steps == p+q steps, bitwise
    one, _ = _gpu_pass(B, w, None)
    np.testing.assert_array_equal(one, got)
    # residual of the last step over the whole grid, fp64 numpy (D4 written out)
    N = w.N
    dx = w.L / N
    c = prev * dt[0] / dx
    r = w.nu[0] * dt[0] / dx ** 2
    x = got[0]
    res = (-r - np.maximum(c, 0)) * np.roll(x, 1) + (1 + 2 * r + np.abs(c)) * x + (-r + np.minimum(c, 0)) * np.roll(x, -1) - prev
    assert np.abs(res).max() <= 1e-13 * (1 + 4 * r), np.abs(res).max()
    # windows against the oracle (margin: 64 cells per step, see the module docstring)
    lam = ((1 + 2 * r) - math.sqrt(1 + 4 * r)) / (2 * r)
    assert lam ** 64 < 1e-12
    n = w.n_steps
    margin, width = 64 * n, 1 << 16
    for start in (N - width // 2, N // 4 - width // 2, 3 * N // 4 - width // 2):
        idx, win = _window(w.u0[0], start, width)
        Lw = dx * (width - 1)
        ref = oracle.btcs(win[None, :], Lw, w.nu, dt, n, oracle.DIRICHLET)[0]
        cc = slice(margin, width - margin)
        err = np.abs(got[0, idx[cc]] - ref[cc]).max() / np.abs(w.u0).max()
        assert err <= 1e-10, (start, err)
    _max_principle(got, w.u0, 1e-12)


def test_c2_full_adjoint_checkpointed(B):
    """Reverse-mode derivative of the whole C2 fp32 run (1024 trajectories, 10 000 Euler steps): 168 GB of
    forward states, so the call checkpoints (100 segments of 100 steps, 3.3 GB).  Sampled trajectories
    against the oracle's adjoint, which stores every state."""
    w = W.c2_dirichlet_batch(dtype=np.float32)
    u0, nu = to_dev(w.u0), to_dev(w.nu)
    dt = B.dt_from_cfl(u0, w.L, nu, w.cfl, w.bc)
    rng = np.random.default_rng(77)
    lam_T = rng.standard_normal(w.u0.shape).astype(np.float32)
    lam = to_dev(lam_T.copy())
    need = B.raw().burgers_adjoint_workspace_bytes(0, w.B, w.N, w.bc, w.n_steps)
    assert need < 6 << 30                                   # checkpointed: far below the 168 GB of all states
    B.burgers_explicit_adjoint(u0, lam, w.L, nu, dt, w.n_steps, w.bc)
    got = lam.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(got))
    np.testing.assert_array_equal(u0.cpu().numpy(), w.u0)
    rows = np.array([0, 313, 700, w.B - 1])
    dth = dt.cpu().numpy().astype(np.float64)
    ref = oracle.explicit_adjoint(w.u0[rows].astype(np.float64), lam_T[rows].astype(np.float64), w.L,
                                  w.nu[rows].astype(np.float64), dth[rows], w.n_steps, w.bc)
    scale = np.abs(ref).max(axis=1, keepdims=True)
    assert (np.abs(got[rows] - ref) / scale).max() <= 1e-4


# ---- the §8(f) rows at the sizes and settings bench.py times (`schemes`: c3_newton, c3_cn, c3_gs, c2_traj) ----

def _c3_inputs(B, cfl):
    import torch
    w = W.c3_periodic_btcs()                                       # B=4096, N=2048
    u, nu = to_dev(w.u0.copy()), to_dev(w.nu)
    dt = B.dt_from_cfl(u, w.L, nu, cfl, w.bc)
    it = torch.zeros(w.B, dtype=torch.int64, device="cuda")
    rows = np.sort(np.random.default_rng(5).choice(w.B, 12, replace=False))
    rows[0], rows[-1] = 0, w.B - 1
    return w, u, nu, dt, it, rows


@pytest.mark.parametrize("theta", [1.0, 0.5])
def test_c3_full_newton_and_crank_nicolson(B, theta):
    """bench.py's c3_newton / c3_cn: 1 000 steps, tol 1e-6.  Newton converges quadratically, so an iterate
    accepted at residual < 1e-6 is the converged one to ~1e-12 and a stopping decision taken differently at a
    tie cannot move the result above the bar; the iteration totals may differ by such ties only."""
    w, u, nu, dt, it, rows = _c3_inputs(B, W.c3_periodic_btcs().cfl)
    B.burgers_newton(u, w.L, nu, dt, w.n_steps, w.bc, tol=1e-6, max_iter=50, iters_out=it, theta=theta)
    got, dth, itg = u.cpu().numpy(), dt.cpu().numpy(), it.cpu().numpy()
    ref, it_ref = oracle.newton_btcs(w.u0[rows], w.L, w.nu[rows], dth[rows], w.n_steps, w.bc, tol=1e-6, max_iter=50,
                                     return_iters=True, theta=theta)
    assert rel_err(got[rows], ref, w.u0[rows]) <= 1e-9
    assert np.all(np.abs(itg[rows] - it_ref) <= 0.01 * it_ref)
    assert np.all(np.isfinite(got)) and itg.min() >= w.n_steps and itg.max() <= 4 * w.n_steps


def test_c3_full_gauss_seidel(B):
    """bench.py's c3_gs: C = 0.4, 100 steps, tol 1e-6 (the CTA-per-system plan at N = 2048)."""
    w, u, nu, dt, it, rows = _c3_inputs(B, 0.4)
    n = 100
    B.burgers_btcs_gs(u, w.L, nu, dt, n, w.bc, tol=1e-6, max_iter=1000, iters_out=it)
    got, dth, itg = u.cpu().numpy(), dt.cpu().numpy(), it.cpu().numpy()
    ref, it_ref = oracle.btcs_gs(w.u0[rows], w.L, w.nu[rows], dth[rows], n, w.bc, tol=1e-6, max_iter=1000,
                                 return_iters=True)
    np.testing.assert_array_equal(itg[rows], it_ref)              # same sweeps: iterates agree to rounding
    assert rel_err(got[rows], ref, w.u0[rows]) <= 1e-10
    direct = oracle.btcs(w.u0[rows], w.L, w.nu[rows], dth[rows], n, w.bc)
    assert rel_err(got[rows], direct, w.u0[rows]) <= 10 * n * 1e-6
    _max_principle(got, w.u0, 1e-12)                               # every sweep is a convex combination (M-matrix)
    assert 3.0 <= itg.mean() / n <= 8.0


def test_c2_full_trajectory_snapshots(B):
    """bench.py's c2_traj: C2 fp32, a snapshot of all 1024 trajectories every 50 steps (200 snapshots, 3.4 GB)."""
    import torch
    w = W.c2_dirichlet_batch(dtype=np.float32)
    u, nu = to_dev(w.u0.copy()), to_dev(w.nu)
    dt = B.dt_from_cfl(u, w.L, nu, w.cfl, w.bc)
    _, snaps = B.burgers_explicit_traj(u, w.L, nu, dt, w.n_steps, w.bc, B.SCHEME_EULER, 50)
    assert tuple(snaps.shape) == (200, w.B, w.N)
    rows = np.array([0, 411, w.B - 1])
    dth = dt.cpu().numpy().astype(np.float64)
    ref_u, ref_snaps = oracle.explicit_trajectory(w.u0[rows].astype(np.float64), w.L, w.nu[rows].astype(np.float64),
                                                  dth[rows], w.n_steps, w.bc, oracle.EULER, 50)
    got = snaps[:, torch.as_tensor(rows, device="cuda"), :].cpu().numpy()
    assert got.shape == ref_snaps.shape
    scale = np.abs(w.u0[rows]).max()
    assert np.abs(got - ref_snaps).max() / scale <= 1e-4
    assert rel_err(u.cpu().numpy()[rows], ref_u, w.u0[rows]) <= 1e-4
    # the last snapshot is the final state up to the rounding of the unscaling (snapshots: reciprocal + one
    # correction, final state: exact quotient; burgers.h); the frozen Dirichlet ends are in every snapshot, bit-exact
    assert (snaps[-1] - u).abs().max().item() <= 2.4e-7 * float(scale)
    assert torch.equal(snaps[:, :, 0], to_dev(w.u0[:, 0]).expand(200, -1))
    assert torch.equal(snaps[:, :, -1], to_dev(w.u0[:, -1]).expand(200, -1))
