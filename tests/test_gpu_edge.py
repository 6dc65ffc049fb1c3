"""Edge cases of the CUDA path: NaN / Inf stay inside their trajectory, many tiny trajectories, the
largest resident sizes, dt = 0, and step counts that are not multiples of any blocking factor."""
import math

import numpy as np
import pytest

import oracle
from parity import rel_err, to_dev
from paper_2601_12204_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_nan_stays_in_its_trajectory(B, dtype):
    w = W.c3_periodic_btcs(B=4, N=512, n_steps=0, dtype=dtype)
    u0 = w.u0.copy(); u0[2, 100] = np.nan
    dt = oracle.dt_from_cfl(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), 0.4, w.bc).astype(dtype)
    clean = [0, 1, 3]
    tol = 1e-4 if dtype == np.float32 else 1e-10
    for name, run, ref in (
        ("euler", lambda u: B.burgers_explicit(u, w.L, to_dev(w.nu), to_dev(dt), 30, w.bc, 0),
         lambda a: oracle.explicit(a, w.L, w.nu.astype(np.float64)[clean], dt.astype(np.float64)[clean], 30, w.bc, 0)),
        ("rk4", lambda u: B.burgers_explicit(u, w.L, to_dev(w.nu), to_dev(dt), 10, w.bc, 1),
         lambda a: oracle.explicit(a, w.L, w.nu.astype(np.float64)[clean], dt.astype(np.float64)[clean], 10, w.bc, 1)),
        ("btcs", lambda u: B.burgers_btcs(u, w.L, to_dev(w.nu), to_dev(dt), 6, w.bc),
         lambda a: oracle.btcs(a, w.L, w.nu.astype(np.float64)[clean], dt.astype(np.float64)[clean], 6, w.bc)),
        ("newton", lambda u: B.burgers_newton(u, w.L, to_dev(w.nu), to_dev(dt), 4, w.bc, tol=1e-5 if dtype == np.float32 else 1e-12,
                                              max_iter=8),
         lambda a: oracle.newton_btcs(a, w.L, w.nu.astype(np.float64)[clean], dt.astype(np.float64)[clean], 4, w.bc, tol=1e-12)),
    ):
        u = to_dev(u0.copy())
        run(u)
        got = u.cpu().numpy()
        assert np.isnan(got[2]).any(), name
        assert np.isfinite(got[clean]).all(), name
        want = ref(w.u0.astype(np.float64)[clean])
        assert rel_err(got[clean], want, w.u0[clean]) <= tol, name


def test_many_tiny_and_largest_resident(B):
    rng = np.random.default_rng(4)
    # 70 000 trajectories of 8 points: grid dimension beyond 65 535, one warp or less per trajectory
    u0 = rng.uniform(-1, 1, (70000, 8)); nu = rng.uniform(0.05, 0.2, 70000)
    dt = oracle.dt_from_cfl(u0, 1.0, nu, 0.4, 0)
    got = B.dt_from_cfl(to_dev(u0), 1.0, to_dev(nu), 0.4, 0).cpu().numpy()
    assert np.all(np.abs(got - dt) <= 2 * np.spacing(dt))
    sel = rng.choice(70000, 64, replace=False)
    for scheme, n in ((0, 11), (1, 5)):
        u = to_dev(u0.copy()); B.burgers_explicit(u, 1.0, to_dev(nu), to_dev(dt), n, 0, scheme)
        ref = oracle.explicit(u0[sel], 1.0, nu[sel], dt[sel], n, 0, scheme)
        assert rel_err(u.cpu().numpy()[sel], ref, u0[sel]) <= 1e-12
    u = to_dev(u0.copy()); B.burgers_btcs(u, 1.0, to_dev(nu), to_dev(dt * 10), 4, 0)
    assert rel_err(u.cpu().numpy()[sel], oracle.btcs(u0[sel], 1.0, nu[sel], dt[sel] * 10, 4, 0), u0[sel]) <= 1e-12
    # the largest sizes the resident plans take (fp32 Euler: 32 points x 256 threads; fp64: 32 x 512), found
    # through burgers_plan_query so that the test cannot silently run nothing
    for dtype, expect in ((np.float32, 8192), (np.float64, 16384)):
        is64 = dtype == np.float64
        N = 64
        while B.plan_query(B.OP_EXPLICIT, is64, 2, 2 * N, 0, 0) == B.PLAN_RESIDENT:
            N *= 2
        assert N == expect, (dtype, N)
        assert B.plan_query(B.OP_EXPLICIT, is64, 2, N, 0, 0) == B.PLAN_RESIDENT
        assert B.plan_query(B.OP_EXPLICIT, is64, 2, 2 * N, 0, 0) == B.PLAN_TILED
        x = np.arange(N) / N
        v0 = np.stack([np.sin(2 * math.pi * x), 0.3 + np.cos(6 * math.pi * x)]).astype(dtype)
        nv = np.array([0.01, 0.02], dtype=dtype)
        dv = oracle.dt_from_cfl(v0.astype(np.float64), 1.0, nv.astype(np.float64), 0.4, 0).astype(dtype)
        u = to_dev(v0.copy()); B.burgers_explicit(u, 1.0, to_dev(nv), to_dev(dv), 77, 0, 0)
        ref = oracle.explicit(v0.astype(np.float64), 1.0, nv.astype(np.float64), dv.astype(np.float64), 77, 0, 0)
        assert rel_err(u.cpu().numpy(), ref, v0) <= (1e-4 if dtype == np.float32 else 1e-10)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_zero_time_step_changes_nothing(B, dtype):
    w = W.c2_dirichlet_batch(B=3, N=1024, dtype=dtype)
    dt = np.zeros(3, dtype=dtype)
    for plan in (B.PLAN_RESIDENT, B.PLAN_TILED):
        for scheme in (0, 1):
            u = to_dev(w.u0.copy())
            B.burgers_explicit(u, w.L, to_dev(w.nu), to_dev(dt), 9, w.bc, scheme, plan=plan)
            np.testing.assert_array_equal(u.cpu().numpy(), w.u0)
    u = to_dev(w.u0.copy()); B.burgers_btcs(u, w.L, to_dev(w.nu), to_dev(dt), 3, w.bc)
    np.testing.assert_array_equal(u.cpu().numpy(), w.u0)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_step_function_at_five_times_the_convective_limit(B, dtype):
    """PAPER.md:193 (Eq.20) with Dirichlet ends on the paper's grid N = 201 at dt = 5 dx/u_max:
    parity with the oracle, max principle, monotone front, frozen ends -- batched (every plan that takes
    N = 201) and one trajectory."""
    w = W.step_dirichlet(dtype=dtype)
    tol = 1e-4 if dtype == np.float32 else 1e-10
    for Bn in (1, 300):
        u0 = np.repeat(w.u0, Bn, axis=0)
        nu = np.repeat(w.nu, Bn)
        dt = np.full(Bn, w.meta["dt"], dtype=dtype)
        ref = oracle.btcs(u0.astype(np.float64), w.L, nu.astype(np.float64), dt.astype(np.float64), w.n_steps, w.bc)
        for plan in (B.PLAN_AUTO, B.PLAN_THOMAS):
            u = to_dev(u0.copy())
            B.burgers_btcs(u, w.L, to_dev(nu), to_dev(dt), w.n_steps, w.bc, plan=plan)
            got = u.cpu().numpy()
            assert rel_err(got, ref, u0) <= tol, (Bn, plan)
            slack = 1e-5 if dtype == np.float32 else 1e-13
            assert got.min() >= -slack and got.max() <= 1 + slack
            assert np.all(np.diff(got.astype(np.float64), axis=1) <= slack)
            np.testing.assert_array_equal(got[:, 0], u0[:, 0]); np.testing.assert_array_equal(got[:, -1], u0[:, -1])
