"""Trajectory output of the explicit schemes (SURVEY 8(f) NEXT-4b: snapshots for data generation,
PAPER.md:22, :409): burgers_explicit_traj_* against the oracle stepped snapshot by snapshot."""
import numpy as np
import pytest

import oracle
from parity import TOL, oracle_dt, rel_err, to_dev
from paper_2601_12204_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


def check(B, w, n, scheme, every, cfl=None):
    dt = oracle_dt(w.u0, w.L, w.nu, cfl or w.cfl, w.bc, w.dtype)
    ref_u, ref_s = oracle.explicit_trajectory(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64),
                                              dt.astype(np.float64), n, w.bc, scheme, every)
    u = to_dev(w.u0.copy())
    _, snaps = B.burgers_explicit_traj(u, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, scheme, every)
    got_u, got_s = u.cpu().numpy(), snaps.cpu().numpy()
    assert got_s.shape == ref_s.shape == (n // every,) + w.u0.shape
    assert rel_err(got_u, ref_u, w.u0) <= TOL[w.dtype]
    for k in range(n // every):
        assert rel_err(got_s[k], ref_s[k], w.u0) <= TOL[w.dtype], k
    return got_u, got_s, dt


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_resident_euler_and_rk4(B, dtype):
    w = W.c2_dirichlet_batch(B=6, N=2048, dtype=dtype)
    got_u, got_s, dt = check(B, w, 230, B.SCHEME_EULER, 50)        # ragged tail of 30 steps
    np.testing.assert_array_equal(got_s[:, :, 0], np.broadcast_to(w.u0[:, 0], got_s[:, :, 0].shape))
    check(B, w, 40, B.SCHEME_RK4, 8, cfl=0.8)
    check(B, w, 12, B.SCHEME_EULER, 1)                              # every step
    w5 = W.c5_rk4_ensemble(rows=np.arange(0, 65536, 8192), dtype=dtype)
    check(B, w5, 90, B.SCHEME_RK4, 30)
    if dtype == np.float64:     # fp64 steps compose bitwise: a snapshot equals a separate call of that length
        u = to_dev(w.u0.copy())
        B.burgers_explicit(u, w.L, to_dev(w.nu), to_dev(dt), 100, w.bc, B.SCHEME_EULER)
        np.testing.assert_array_equal(u.cpu().numpy(), got_s[1])


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_tiled_plan_chunks(B, dtype):
    w = W.c4a_long_explicit(N=(1 << 15) + 24, n_steps=0, dtype=dtype)
    assert B.plan_query(B.OP_EXPLICIT, dtype == np.float64, 1, w.N, w.bc, 0) == B.PLAN_TILED
    check(B, w, 150, B.SCHEME_EULER, 70)
    check(B, w, 30, B.SCHEME_RK4, 10, cfl=0.5)     # at this N the two limits coincide: c + 2r = 2C must stay < 1.39 (D9)


def test_semantics(B):
    w = W.c2_dirichlet_batch(B=2, N=256, dtype=np.float64)
    dt = oracle_dt(w.u0, w.L, w.nu, 0.4, w.bc, w.dtype)
    u = to_dev(w.u0.copy())
    _, snaps = B.burgers_explicit_traj(u, w.L, to_dev(w.nu), to_dev(dt), 5, w.bc, 0, 10)   # no snapshot due
    assert snaps.shape[0] == 0
    ref = oracle.explicit(w.u0, w.L, w.nu, dt, 5, w.bc, 0)
    assert rel_err(u.cpu().numpy(), ref, w.u0) <= 1e-12
    with pytest.raises(B.BurgersError):
        B.burgers_explicit_traj(u, w.L, to_dev(w.nu), to_dev(dt), 5, w.bc, 0, 0)


def test_btcs_trajectory(B):
    for w, n, every in ((W.c3_periodic_btcs(B=6, N=512, n_steps=0), 23, 5),
                        (W.c2_dirichlet_batch(B=3, N=1000, dtype=np.float64), 12, 4),       # THOMAS plan
                        (W.c4b_long_btcs(N=1 << 14, n_steps=0), 9, 3)):                     # LONG plan
        dt = oracle_dt(w.u0, w.L, w.nu, 10.0, w.bc, w.dtype)
        u = to_dev(w.u0.copy())
        _, snaps = B.burgers_btcs_traj(u, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, every)
        assert snaps.shape[0] == n // every
        ref = w.u0.astype(np.float64)
        for k in range(n // every):
            ref = oracle.btcs(ref, w.L, w.nu, dt, every, w.bc)
            assert rel_err(snaps[k].cpu().numpy(), ref, w.u0) <= 1e-10, (w.name, k)
        ref = oracle.btcs(ref, w.L, w.nu, dt, n - (n // every) * every, w.bc)
        assert rel_err(u.cpu().numpy(), ref, w.u0) <= 1e-10


@pytest.mark.parametrize("theta", [1.0, 0.5])
def test_newton_trajectory_snapshots(B, theta):
    """burgers_newton_traj_*: snapshots of the Newton / Crank-Nicolson scheme every m steps equal the oracle's states
    after m, 2m, ... steps (the oracle called interval by interval: the same composition), the iteration totals are
    those of the single call, resident ragged (N = 201) and exact (N = 512) plans, Dirichlet and periodic."""
    import torch
    for w in (W.c3_periodic_btcs(B=5, N=512, n_steps=0), W.c2_dirichlet_batch(B=4, N=201, dtype=np.float64)):
        nu = np.full(w.B, 0.1)                                     # cell Peclet number below 2 (D11)
        dt = oracle.dt_from_cfl(w.u0, w.L, nu, 2.0, w.bc)
        n, m = 23, 5
        u = to_dev(w.u0.copy()); it = torch.zeros(w.B, dtype=torch.int64, device="cuda")
        _, snaps = B.burgers_newton_traj(u, w.L, to_dev(nu), to_dev(dt), n, w.bc, m, tol=1e-12, iters_out=it, theta=theta)
        assert tuple(snaps.shape) == (4, w.B, w.N)
        ref = w.u0.copy(); tot = np.zeros(w.B, dtype=np.int64)
        for k in range(4):
            ref, itr = oracle.newton_btcs(ref, w.L, nu, dt, m, w.bc, tol=1e-12, theta=theta, return_iters=True)
            tot += itr
            assert rel_err(snaps[k].cpu().numpy(), ref, w.u0) <= 1e-10, (w.name, k)
        ref, itr = oracle.newton_btcs(ref, w.L, nu, dt, n - 4 * m, w.bc, tol=1e-12, theta=theta, return_iters=True)
        tot += itr
        assert rel_err(u.cpu().numpy(), ref, w.u0) <= 1e-10
        u1 = to_dev(w.u0.copy()); it1 = torch.zeros(w.B, dtype=torch.int64, device="cuda")
        B.burgers_newton(u1, w.L, to_dev(nu), to_dev(dt), n, w.bc, tol=1e-12, iters_out=it1, theta=theta)
        assert torch.equal(u1, u) and torch.equal(it1, it)          # the composition is bitwise the single call
        assert np.all(np.abs(it.cpu().numpy() - tot) <= 2)
