"""Adaptive time step (SURVEY 8(f) NEXT-4a): burgers_explicit_adaptive_* against the oracle's composition
of dt_from_cfl and explicit stepping."""
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


@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 1e-4)])
def test_adaptive_matches_oracle_composition(B, dtype, tol):
    for w, scheme, C, n_outer, m in ((W.c5_rk4_ensemble(rows=np.arange(0, 65536, 8192), dtype=dtype), 1, 0.8, 6, 25),
                                     (W.c2_dirichlet_batch(B=5, N=1024, dtype=dtype), 0, 0.4, 5, 40),
                                     (W.c4a_long_explicit(N=(1 << 15) + 8, n_steps=0, dtype=dtype), 0, 0.4, 3, 70)):
        ref_u, ref_t = oracle.explicit_adaptive(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), C, n_outer, m,
                                                w.bc, scheme, dtype=dtype)
        u = to_dev(w.u0.copy())
        _, t, dt = B.burgers_explicit_adaptive(u, w.L, to_dev(w.nu), C, n_outer, m, w.bc, scheme)
        assert rel_err(u.cpu().numpy(), ref_u, w.u0) <= tol, w.name
        np.testing.assert_allclose(t.cpu().numpy(), ref_t, rtol=1e-5 if dtype == np.float32 else 1e-12)
        # the solution decays, so the convective bound can only relax: dt never shrinks
        dt0 = oracle.dt_from_cfl(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), C, w.bc)
        assert np.all(dt.cpu().numpy() >= dt0 * (1 - 1e-6))


def test_zero_outer_iterations(B):
    w = W.c2_dirichlet_batch(B=2, N=256, dtype=np.float64)
    u = to_dev(w.u0.copy())
    _, t, _ = B.burgers_explicit_adaptive(u, w.L, to_dev(w.nu), 0.4, 0, 10, w.bc, 0)
    np.testing.assert_array_equal(u.cpu().numpy(), w.u0)
    assert np.all(t.cpu().numpy() == 0)


@pytest.mark.parametrize("scheme", [0, 1])
@pytest.mark.parametrize("bc_dirichlet", [False, True])
def test_fused_resident_path_equals_separate_calls_bitwise_in_fp64(B, scheme, bc_dirichlet):
    """RESIDENT shapes run ONE kernel with the CFL evaluation inside the time loop.  In fp64 (unscaled state,
    same max, same dt formula, p then q steps == p+q steps) it must give the bits of the composition
    dt_from_cfl -> m explicit steps -> ... made of separate library calls, including t and the last dt."""
    import torch
    w = (W.c2_dirichlet_batch(B=7, N=2048, dtype=np.float64) if bc_dirichlet
         else W.c5_rk4_ensemble(rows=np.arange(0, 65536, 9000), dtype=np.float64))
    assert B.plan_query(B.OP_EXPLICIT, True, w.B, w.N, w.bc, scheme) == B.PLAN_RESIDENT
    C, n_outer, m = (0.4 if scheme == 0 else 0.7), 9, 13
    nu = to_dev(w.nu)
    u1 = to_dev(w.u0.copy())
    _, t1, dt1 = B.burgers_explicit_adaptive(u1, w.L, nu, C, n_outer, m, w.bc, scheme)
    u2 = to_dev(w.u0.copy())
    t2 = torch.zeros(w.B, dtype=torch.float64, device="cuda")
    for _ in range(n_outer):
        dt2 = B.dt_from_cfl(u2, w.L, nu, C, w.bc)
        B.burgers_explicit(u2, w.L, nu, dt2, m, w.bc, scheme)
        t2 += m * dt2
    assert torch.equal(u1, u2)
    assert torch.equal(dt1, dt2)
    assert torch.allclose(t1, t2, rtol=1e-14, atol=0.0)           # (the kernel accumulates m*dt with an FMA)


def test_fused_fp32_rescaling_is_accurate_over_many_evaluations(B):
    """fp32 carries the state scaled by dt/dx, so every new dt rescales it (two-term ratio, explicit_impl.cuh):
    600 evaluations must not cost accuracy against the oracle's composition."""
    w = W.c2_dirichlet_batch(B=4, N=1024, dtype=np.float32)
    n_outer, m = 600, 5
    ref_u, ref_t = oracle.explicit_adaptive(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), 0.4, n_outer, m,
                                            w.bc, 0, dtype=np.float32)
    u = to_dev(w.u0.copy())
    _, t, _ = B.burgers_explicit_adaptive(u, w.L, to_dev(w.nu), 0.4, n_outer, m, w.bc, 0)
    got = u.cpu().numpy()
    assert rel_err(got, ref_u, w.u0) <= 1e-4
    np.testing.assert_array_equal(got[:, 0], w.u0[:, 0])          # frozen Dirichlet ends keep their bits
    np.testing.assert_array_equal(got[:, -1], w.u0[:, -1])
    np.testing.assert_allclose(t.cpu().numpy(), ref_t, rtol=1e-5)


def test_zero_state_and_single_warp_shapes(B):
    """u == 0: dt is the diffusive bound, the state stays 0.  N = 64 (one warp per trajectory: the shuffle
    exchange variant of the kernel) against the oracle."""
    for dtype, tol in ((np.float64, 1e-10), (np.float32, 1e-4)):
        z = np.zeros((3, 512), dtype=dtype)
        nu = np.full(3, 0.02, dtype=dtype)
        u = to_dev(z.copy())
        _, t, dt = B.burgers_explicit_adaptive(u, 1.0, to_dev(nu), 0.4, 4, 6, 0, 0)
        assert np.all(u.cpu().numpy() == 0)
        ref_dt = oracle.dt_from_cfl(z.astype(np.float64), 1.0, nu.astype(np.float64), 0.4, 0)
        np.testing.assert_allclose(dt.cpu().numpy(), ref_dt, rtol=1e-6)
        np.testing.assert_allclose(t.cpu().numpy(), 24 * ref_dt, rtol=1e-6)
        w = W.c3_periodic_btcs(B=6, N=64, n_steps=0, dtype=dtype)
        for scheme in (0, 1):
            ref_u, ref_t = oracle.explicit_adaptive(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), 0.4, 7, 9,
                                                    w.bc, scheme, dtype=dtype)
            u = to_dev(w.u0.copy())
            _, t, _ = B.burgers_explicit_adaptive(u, w.L, to_dev(w.nu), 0.4, 7, 9, w.bc, scheme)
            assert rel_err(u.cpu().numpy(), ref_u, w.u0) <= tol
            np.testing.assert_allclose(t.cpu().numpy(), ref_t, rtol=1e-5 if dtype == np.float32 else 1e-12)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("scheme,m", [(0, 300), (0, 70), (1, 90)])
def test_fused_tiled_path_equals_separate_calls_bitwise(B, dtype, scheme, m):
    """TILED grids: the CFL reduction rides on the launches of the time stepping (the last launch of a segment leaves
    max |u| of what it stores in a slot, the next segment's launches evaluate dt from it).  Same maximum, same dt
    formula, same launches otherwise: the bits of dt_from_cfl -> m explicit steps -> ... made of separate library
    calls, in fp32 too (the state is unscaled in HBM at every segment boundary in both).  m = 300 / 90: two launches
    per segment (256 Euler / 64 RK4 steps per launch); batches of two long rows, periodic and Dirichlet."""
    import torch
    n_outer = 4
    for bc in (0, 1):
        N = 40000
        x = np.arange(N) / N
        u0 = np.stack([np.sin(2 * np.pi * x) + 0.3, 0.8 * np.cos(6 * np.pi * x) - 0.2]).astype(dtype)
        nu_h = np.array([2e-4, 5e-4], dtype=dtype)
        L = 1.0
        C = 0.4 if scheme == 0 else 0.7
        assert B.plan_query(B.OP_EXPLICIT, dtype == np.float64, 2, N, bc, scheme) == B.PLAN_TILED
        nu = to_dev(nu_h)
        u1 = to_dev(u0.copy())
        _, t1, dt1 = B.burgers_explicit_adaptive(u1, L, nu, C, n_outer, m, bc, scheme)
        u2 = to_dev(u0.copy())
        t2 = torch.zeros(2, dtype=torch.float64, device="cuda")
        for _ in range(n_outer):
            dt2 = B.dt_from_cfl(u2, L, nu, C, bc)
            B.burgers_explicit(u2, L, nu, dt2, m, bc, scheme)
            t2 += m * dt2.double()
        assert torch.equal(u1, u2), (bc, "state")
        assert torch.equal(dt1, dt2) and torch.equal(t1, t2), (bc, "dt / t")
        ref_u, ref_t = oracle.explicit_adaptive(u0.astype(np.float64), L, nu_h.astype(np.float64), C, n_outer, m, bc, scheme,
                                                dtype=dtype)
        assert rel_err(u1.cpu().numpy(), ref_u, u0) <= (1e-4 if dtype == np.float32 else 1e-10)
