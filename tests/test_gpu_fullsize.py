"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (AUTO plan,
dt from the library's own dt_from_cfl, one call for all n_steps), against the oracle on the WHOLE output
("C5 parity uses the deterministic subset b = 0 (mod 16); all other configs run full size"):

  - C2 (fp32 and fp64) and C3: the oracle runs every trajectory, every point is compared;
  - C5: the oracle runs the 4096 trajectories b = 0 (mod 16), every point of those is compared;
  - C4a: the oracle (oracle.explicit_long) runs the whole 2^24-point grid for all 2 000 steps;
  - C4b: (i) the oracle (oracle.btcs, B = 1: Thomas + Sherman-Morrison on the whole 2^22-point cyclic system)
    runs the whole grid for the first 16 steps; (ii) for all 200 steps every output point is compared with
    the oracle run on 40 overlapping WINDOWS that together cover the grid: BTCS couples all points, but the
    influence of a point decays per cell like lam = ((1+2r) - sqrt(1+4r)) / (2r) per step (Green's function
    of the diffusion part; convection only strengthens the diagonal): at r = 5, lam = 0.642, i.e. < 1e-12
    beyond 63 cells per step, so a margin of 64*n_steps cells makes a window's centre exact to far below the
    1e-10 tolerance whatever is done at the window ends.  (The whole-grid oracle for all 200 steps would take
    several minutes on one host core: its second Sherman-Morrison solve decays into the subnormal range and
    stays there.)  (iii) the defining residual A(u^n) u^{n+1} = u^n of the last step in fp64 numpy over the
    whole grid;

the rows of SURVEY 8(f) that bench.py times (Newton / Crank-Nicolson and Gauss-Seidel on C3's inputs, C2 with
trajectory output, the checkpointed adjoint of the whole C2 run), whose oracles are slow, stay on seeded
samples of whole trajectories at the end of the file; plus properties that hold at any size, checked on ALL
outputs: finiteness, the discrete maximum principle (D4 / D9), frozen Dirichlet ends.

The worst error of each config is appended to gpurun_out/fullsize_parity.json (when that folder exists) so
that DESIGN.md can quote it.
"""
import json
import math
import os

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


def _record(name, err, tol):
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "fullsize_parity.json"), "a") as f:
            f.write(json.dumps({"case": name, "worst_rel_err": err, "tol": tol}) + "\n")


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
    ref = oracle.explicit(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64),
                          dt.astype(np.float64), w.n_steps, w.bc, oracle.EULER)      # all 1024 trajectories
    e = rel_err(got, ref, w.u0)
    _record(f"c2_{np.dtype(dtype).name}", e, TOL[np.dtype(dtype)])
    assert e <= TOL[np.dtype(dtype)]
    np.testing.assert_array_equal(got[:, 0], w.u0[:, 0])
    np.testing.assert_array_equal(got[:, -1], w.u0[:, -1])
    _max_principle(got, w.u0, 1e-5 if dtype == np.float32 else 1e-12)   # |c| + 2r <= 0.8: monotone


def test_c3_full(B):
    w = W.c3_periodic_btcs()                                       # B=4096, N=2048, 1 000 steps
    assert B.plan_query(B.OP_BTCS, True, w.B, w.N, w.bc) == B.PLAN_HYBRID
    got, dt = _gpu_pass(B, w, None)
    _check_dt(w, dt)
    ref = oracle.btcs(w.u0, w.L, w.nu, dt, w.n_steps, w.bc)           # all 4096 trajectories
    e = rel_err(got, ref, w.u0)
    _record("c3", e, 1e-10)
    assert e <= 1e-10
    _max_principle(got, w.u0, 1e-12)                               # M-matrix: any dt


def test_c5_full(B):
    w = W.c5_rk4_ensemble()                                        # B=65536, N=1024, 5 000 RK4 steps
    assert B.plan_query(B.OP_EXPLICIT, False, w.B, w.N, w.bc, 1) == B.PLAN_RESIDENT
    got, dt = _gpu_pass(B, w, B.SCHEME_RK4)
    _check_dt(w, dt)
    rows = np.arange(0, w.B, 16)                                   # b = 0 (mod 16), 4096 trajectories
    ref = oracle.explicit(w.u0[rows].astype(np.float64), w.L, w.nu[rows].astype(np.float64),
                          dt[rows].astype(np.float64), w.n_steps, w.bc, oracle.RK4)
    e = rel_err(got[rows], ref, w.u0[rows])
    _record("c5_mod16", e, 1e-4)
    assert e <= 1e-4
    assert np.all(np.isfinite(got))
    # RK4 is not monotone, but these pulses only decay: bounded by the initial range (+ rounding)
    _max_principle(got, w.u0, 1e-3)


def test_c4a_full_grid(B):
    w = W.c4a_long_explicit()                                      # N=2^24, 2 000 Euler steps, fp32
    assert B.plan_query(B.OP_EXPLICIT, False, 1, w.N, w.bc, 0) == B.PLAN_TILED
    got, dt = _gpu_pass(B, w, B.SCHEME_EULER)
    _check_dt(w, dt)
    ref = oracle.explicit_long(w.u0[0].astype(np.float64), w.L, float(w.nu[0]), float(dt[0]), w.n_steps, w.bc)
    e = rel_err(got, ref[None, :], w.u0)                           # every one of the 2^24 points
    _record("c4a", e, 1e-4)
    assert e <= 1e-4
    _max_principle(got, w.u0, 1e-5)


def test_c4b_full_grid(B):
    w = W.c4b_long_btcs()                                          # N=2^22, 200 BTCS steps, fp64
    assert B.plan_query(B.OP_BTCS, True, 1, w.N, w.bc) == B.PLAN_LONG
    u, nu = to_dev(w.u0.copy()), to_dev(w.nu)
    dt_d = B.dt_from_cfl(u, w.L, nu, w.cfl, w.bc)
    dt = dt_d.cpu().numpy()
    _check_dt(w, dt)
    # (i) the whole grid against the whole-grid oracle (B = 1) after 16 steps
    n1 = 16
    B.burgers_btcs(u, w.L, nu, dt_d, n1, w.bc)
    got16 = u.cpu().numpy()
    ref16 = oracle.btcs(w.u0, w.L, w.nu, dt, n1, w.bc)
    e = rel_err(got16, ref16, w.u0)
    _record("c4b_16steps_whole_grid", e, 1e-10)
    assert e <= 1e-10
    B.burgers_btcs(u, w.L, nu, dt_d, w.n_steps - n1 - 1, w.bc)
    prev = u.cpu().numpy()[0].copy()
    B.burgers_btcs(u, w.L, nu, dt_d, 1, w.bc)
    got = u.cpu().numpy()
    # in one call too (the bench configuration): 16 + 183 + 1 steps == 200 steps, bitwise
    one, _ = _gpu_pass(B, w, None)
    np.testing.assert_array_equal(one, got)
    # (iii) residual of the last step over the whole grid, fp64 numpy (D4 written out)
    N = w.N
    dx = w.L / N
    c = prev * dt[0] / dx
    r = w.nu[0] * dt[0] / dx ** 2
    x = got[0]
    res = (-r - np.maximum(c, 0)) * np.roll(x, 1) + (1 + 2 * r + np.abs(c)) * x + (-r + np.minimum(c, 0)) * np.roll(x, -1) - prev
    assert np.abs(res).max() <= 1e-13 * (1 + 4 * r), np.abs(res).max()
    # (ii) all 200 steps, every point, against the oracle on overlapping windows (margin: 64 cells per
    # step, see the module docstring)
    lam = ((1 + 2 * r) - math.sqrt(1 + 4 * r)) / (2 * r)
    assert lam ** 64 < 1e-12
    n = w.n_steps
    margin, width = 64 * n, 1 << 17
    core = width - 2 * margin
    starts = np.arange(0, N, core) - margin                        # window k is exact on [k*core, (k+1)*core)
    idx = (starts[:, None] + np.arange(width)[None, :]) % N
    wins = w.u0[0][idx]
    Lw = dx * (width - 1)                                          # same dx: a Dirichlet window of `width` nodes
    ref = oracle.btcs(wins, Lw, np.full(len(starts), w.nu[0]), np.full(len(starts), dt[0]), n, oracle.DIRICHLET)
    cover = np.zeros(N, dtype=bool)
    worst = 0.0
    for k in range(len(starts)):
        cc = slice(margin, margin + core)
        gi = idx[k, cc]
        worst = max(worst, float(np.abs(got[0, gi] - ref[k, cc]).max()))
        cover[gi] = True
    assert cover.all()                                             # every one of the 2^22 points was compared
    e = worst / np.abs(w.u0).max()
    _record("c4b_200steps_window_cover", e, 1e-10)
    assert e <= 1e-10
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


@pytest.mark.parametrize("theta", [1.0, 0.5])
def test_c3_full_newton_converged_meets_the_fp64_bar(B, theta):
    """The same full-size run iterated to tol = 1e-12, where the stopping decision cannot move the result: the
    north_star's fp64 bar of 1e-10 holds (the tol = 1e-6 run above is the bench setting)."""
    w, u, nu, dt, it, rows = _c3_inputs(B, W.c3_periodic_btcs().cfl)
    n = 200
    B.burgers_newton(u, w.L, nu, dt, n, w.bc, tol=1e-12, max_iter=50, iters_out=it, theta=theta)
    got, dth = u.cpu().numpy(), dt.cpu().numpy()
    ref = oracle.newton_btcs(w.u0[rows], w.L, w.nu[rows], dth[rows], n, w.bc, tol=1e-12, max_iter=50, theta=theta)
    e = rel_err(got[rows], ref, w.u0[rows])
    _record(f"c3_newton_theta{theta}_tol1e-12", e, 1e-10)
    assert e <= 1e-10
    assert np.all(np.isfinite(got))


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
