"""GPU parity of the discrete adjoint of forward Euler (SURVEY 8(f) NEXT-4c; D13) against the
oracle's adjoint, plus the dot-product identity checked against the GPU forward path itself."""
import numpy as np
import pytest

import oracle
from parity import oracle_dt, to_dev
from paper_2601_12204_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 1e-4)])
def test_adjoint_matches_oracle(B, dtype, tol):
    rng = np.random.default_rng(6)
    for w, n in ((W.c3_periodic_btcs(B=5, N=512, n_steps=0, dtype=dtype), 60),        # mixed signs, periodic
                 (W.c2_dirichlet_batch(B=4, N=1000, dtype=dtype), 35),                # Dirichlet, ragged N
                 (W.c4a_long_explicit(N=(1 << 15) + 8, n_steps=0, dtype=dtype), 20)): # TILED forward pass
        dt = oracle_dt(w.u0, w.L, w.nu, 0.4, w.bc, dtype)
        lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
        ref = oracle.explicit_adjoint(w.u0.astype(np.float64), lam_T.astype(np.float64), w.L, w.nu.astype(np.float64),
                                      dt.astype(np.float64), n, w.bc)
        u0 = to_dev(w.u0.copy()); lam = to_dev(lam_T.copy())
        B.burgers_explicit_adjoint(u0, lam, w.L, to_dev(w.nu), to_dev(dt), n, w.bc)
        got = lam.cpu().numpy().astype(np.float64)
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert (np.abs(got - ref) / scale).max() <= tol, w.name
        np.testing.assert_array_equal(u0.cpu().numpy(), w.u0)          # u0 untouched


def test_gradient_against_gpu_finite_differences(B):
    # J(u0) = <lam_T, u^N(u0)> with the GPU forward path; its directional derivative along v must equal
    # <adjoint(lam_T), v>
    rng = np.random.default_rng(9)
    N, L, n = 256, 1.0, 80
    x = np.arange(N) / N
    u0 = (0.9 + 0.5 * np.sin(2 * np.pi * x) + 0.2 * np.cos(6 * np.pi * x))[None, :]
    nu = np.array([0.02]); dt = oracle.dt_from_cfl(u0, L, nu, 0.4, 0)
    lam_T = rng.standard_normal((1, N)); v = rng.standard_normal((1, N))

    def J(u):
        d = to_dev(u.copy()); B.burgers_explicit(d, L, to_dev(nu), to_dev(dt), n, 0, 0)
        return float((lam_T * d.cpu().numpy()).sum())

    eps = 1e-6
    fd = (J(u0 + eps * v) - J(u0 - eps * v)) / (2 * eps)
    lam = to_dev(lam_T.copy())
    B.burgers_explicit_adjoint(to_dev(u0), lam, L, to_dev(nu), to_dev(dt), n, 0)
    ad = float((lam.cpu().numpy() * v).sum())
    assert abs(fd - ad) <= 1e-6 * (abs(ad) + 1), (fd, ad)


def test_zero_and_one_step(B):
    w = W.c2_dirichlet_batch(B=2, N=64, dtype=np.float64)
    dt = oracle_dt(w.u0, w.L, w.nu, 0.4, w.bc, w.dtype)
    lam_T = np.random.default_rng(1).standard_normal(w.u0.shape)
    lam = to_dev(lam_T.copy()); B.burgers_explicit_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), 0, w.bc)
    np.testing.assert_array_equal(lam.cpu().numpy(), lam_T)
    lam = to_dev(lam_T.copy()); B.burgers_explicit_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), 1, w.bc)
    ref = oracle.explicit_adjoint(w.u0, lam_T, w.L, w.nu, dt, 1, w.bc)
    np.testing.assert_allclose(lam.cpu().numpy(), ref, atol=1e-14)


@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 1e-4)])
def test_checkpointed_adjoint(B, dtype, tol):
    """Segments of 1, 7, 16 and 100 steps (ragged last segment, single-step segments, one segment) give the
    gradient of the un-checkpointed run: bitwise in fp64 (the recomputed states are the same numbers)."""
    rng = np.random.default_rng(10)
    w = W.c3_periodic_btcs(B=4, N=256, n_steps=0, dtype=dtype)
    n = 45
    dt = oracle_dt(w.u0, w.L, w.nu, 0.4, w.bc, dtype)
    lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
    ref = oracle.explicit_adjoint(w.u0.astype(np.float64), lam_T.astype(np.float64), w.L, w.nu.astype(np.float64),
                                  dt.astype(np.float64), n, w.bc)
    scale = np.abs(ref).max(axis=1, keepdims=True)
    full = None
    for segment in (0, 1, 7, 16, 100):
        lam = to_dev(lam_T.copy())
        B.burgers_explicit_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, segment=segment)
        got = lam.cpu().numpy()
        assert (np.abs(got.astype(np.float64) - ref) / scale).max() <= tol, segment
        if full is None:
            full = got
        elif dtype == np.float64:
            np.testing.assert_array_equal(got, full)


# ---------------------------------------------------------------- adjoint of classical RK4 (D14)
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 1e-4)])
def test_rk4_adjoint_matches_oracle(B, dtype, tol):
    """PAPER.md:224-229 (Eq.22), :231: reverse-mode derivative of RK4 steps, against the oracle's adjoint (pinned by the
    dot-product identity, R(dt A)^T and finite differences).  Shapes: mixed signs periodic, Dirichlet with a ragged N,
    a grid whose forward pass is TILED, a checkpointed run (segments of 7 steps), C5's pulses."""
    rng = np.random.default_rng(16)
    for w, n, seg in ((W.c3_periodic_btcs(B=5, N=512, n_steps=0, dtype=dtype), 40, 0),
                      (W.c2_dirichlet_batch(B=4, N=1000, dtype=dtype), 25, 0),
                      (W.c4a_long_explicit(N=(1 << 15) + 8, n_steps=0, dtype=dtype), 12, 0),
                      (W.c3_periodic_btcs(B=3, N=256, n_steps=0, dtype=dtype), 30, 7),
                      (W.c5_rk4_ensemble(B=6, N=1024, dtype=dtype), 30, 0)):
        dt = oracle_dt(w.u0, w.L, w.nu, 0.8, w.bc, dtype)
        lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
        ref = oracle.explicit_adjoint(w.u0.astype(np.float64), lam_T.astype(np.float64), w.L, w.nu.astype(np.float64),
                                      dt.astype(np.float64), n, w.bc, scheme=oracle.RK4)
        u0 = to_dev(w.u0.copy()); lam = to_dev(lam_T.copy())
        B.burgers_explicit_adjoint(u0, lam, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, segment=seg, scheme=B.SCHEME_RK4)
        got = lam.cpu().numpy().astype(np.float64)
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert (np.abs(got - ref) / scale).max() <= tol, (w.name, seg)
        np.testing.assert_array_equal(u0.cpu().numpy(), w.u0)          # u0 untouched


def test_rk4_adjoint_dot_product_identity_with_the_gpu_forward_path(B):
    """J(u0) = <lam_T, u^N(u0)> with the GPU's own RK4 forward path: its directional derivative along v (central
    differences) equals <adjoint(lam_T), v>; zero steps leave lam alone; bad scheme -> error."""
    rng = np.random.default_rng(19)
    w = W.c3_periodic_btcs(B=2, N=256, n_steps=0)
    dt = oracle_dt(w.u0, w.L, w.nu, 0.8, w.bc, np.float64)
    n = 30
    lam_T = rng.standard_normal(w.u0.shape); v = rng.standard_normal(w.u0.shape)
    lam = to_dev(lam_T.copy())
    B.burgers_explicit_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, scheme=B.SCHEME_RK4)
    g = lam.cpu().numpy()
    eps = 1e-6

    def J(u0):
        u = to_dev(u0.copy()); B.burgers_explicit(u, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, B.SCHEME_RK4)
        return (lam_T * u.cpu().numpy()).sum(axis=1)
    fd = (J(w.u0 + eps * v) - J(w.u0 - eps * v)) / (2 * eps)
    an = (g * v).sum(axis=1)
    assert np.all(np.abs(fd - an) <= 1e-6 * (1 + np.abs(an)))
    lam = to_dev(lam_T.copy())
    B.burgers_explicit_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), 0, w.bc, scheme=B.SCHEME_RK4)
    np.testing.assert_array_equal(lam.cpu().numpy(), lam_T)
    with pytest.raises(B.BurgersError):
        B.burgers_explicit_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), 3, w.bc, scheme=7)


# ---------------------------------------------------------------- adjoint of the lagged upwind BTCS scheme (D15)
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 1e-4)])
def test_btcs_adjoint_matches_oracle(B, dtype, tol):
    """PAPER.md:231 "gradients of the numerical solution" for the implicit scheme of the hot path: against the oracle's
    adjoint (pinned by the transpose identity, the dense (I - D) A^{-T} formula and finite differences).  Shapes:
    C3-like periodic with mixed signs (resident, exact partitions), the paper's N = 201 and N = 1000 Dirichlet
    (ragged partitions), a long grid (thread-per-system fallback), at the hot path's C = 10."""
    rng = np.random.default_rng(26)
    for w, n in ((W.c3_periodic_btcs(B=5, N=2048, n_steps=0, dtype=dtype), 12),
                 (W.c3_periodic_btcs(B=6, N=201, n_steps=0, dtype=dtype), 15),
                 (W.c2_dirichlet_batch(B=4, N=1000, dtype=dtype), 10),
                 (W.c4b_long_btcs(N=20000, n_steps=0, dtype=dtype), 4)):
        u0 = w.u0.copy()
        if w.bc == 1:
            u0[:, 0] = dtype(0.3); u0[:, -1] = dtype(-0.2)
        dt = oracle_dt(u0, w.L, w.nu, 10.0, w.bc, dtype)
        lam_T = rng.standard_normal(u0.shape).astype(dtype)
        ref = oracle.btcs_adjoint(u0.astype(np.float64), lam_T.astype(np.float64), w.L, w.nu.astype(np.float64),
                                  dt.astype(np.float64), n, w.bc)
        d_u0 = to_dev(u0.copy()); lam = to_dev(lam_T.copy())
        B.burgers_btcs_adjoint(d_u0, lam, w.L, to_dev(w.nu), to_dev(dt), n, w.bc)
        got = lam.cpu().numpy().astype(np.float64)
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert (np.abs(got - ref) / scale).max() <= tol, w.name
        np.testing.assert_array_equal(d_u0.cpu().numpy(), u0)          # u0 untouched


def test_btcs_adjoint_against_finite_differences_of_the_gpu_forward_path(B):
    rng = np.random.default_rng(29)
    w = W.c3_periodic_btcs(B=2, N=256, n_steps=0)
    dt = oracle_dt(w.u0, w.L, w.nu, 10.0, w.bc, np.float64)
    n = 8
    lam_T = rng.standard_normal(w.u0.shape); v = rng.standard_normal(w.u0.shape)
    lam = to_dev(lam_T.copy())
    B.burgers_btcs_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), n, w.bc)
    g = lam.cpu().numpy()
    eps = 1e-6

    def J(u0):
        u = to_dev(u0.copy()); B.burgers_btcs(u, w.L, to_dev(w.nu), to_dev(dt), n, w.bc)
        return (lam_T * u.cpu().numpy()).sum(axis=1)
    fd = (J(w.u0 + eps * v) - J(w.u0 - eps * v)) / (2 * eps)
    an = (g * v).sum(axis=1)
    assert np.all(np.abs(fd - an) <= 1e-6 * (1 + np.abs(an)))
    lam = to_dev(lam_T.copy())
    B.burgers_btcs_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), 0, w.bc)
    np.testing.assert_array_equal(lam.cpu().numpy(), lam_T)


# ---------------------------------------------------------------- D16: reverse mode of the Newton / theta-scheme
def _newton_adjoint_cases(dtype):
    """(workload, u0, nu, n_steps): cell Peclet number |u| dx / nu < 2 everywhere (the Jacobian needs no pivoting)."""
    out = []
    w = W.c3_periodic_btcs(B=5, N=2048, n_steps=0, dtype=dtype)          # resident, exact partitions, mixed signs
    out.append((w, w.u0.copy(), w.nu.copy(), 10))
    w = W.c3_periodic_btcs(B=6, N=201, n_steps=0, dtype=dtype)           # the paper's grid: ragged partitions
    out.append((w, w.u0.copy(), np.full(6, 0.1, dtype), 12))
    w = W.c2_dirichlet_batch(B=4, N=1000, dtype=dtype)                   # Dirichlet, ragged
    u0 = w.u0.copy(); u0[:, 0] = dtype(0.3); u0[:, -1] = dtype(-0.2)
    out.append((w, u0, np.maximum(w.nu, dtype(5e-3)), 8))
    w = W.c4b_long_btcs(N=20000, n_steps=0, dtype=dtype)                 # a long grid: thread-per-system fallback
    out.append((w, w.u0.copy(), np.full(1, 1e-3, dtype), 4))
    return out


@pytest.mark.parametrize("theta", [1.0, 0.5])
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 1e-4)])
def test_newton_adjoint_matches_oracle(B, dtype, tol, theta):
    """Reverse mode of the paper's fully implicit scheme (Eq.10-15) and of Crank-Nicolson against the oracle's (D16:
    pinned by the exact transpose of the linear case, the dense one-step formula and finite differences)."""
    rng = np.random.default_rng(31)
    newton_tol = 1e-13 if dtype == np.float64 else 2e-6
    for w, u0, nu, n in _newton_adjoint_cases(dtype):
        dt = oracle_dt(u0, w.L, nu, 4.0, w.bc, dtype)
        lam_T = rng.standard_normal(u0.shape).astype(dtype)
        ref = oracle.newton_adjoint(u0.astype(np.float64), lam_T.astype(np.float64), w.L, nu.astype(np.float64),
                                    dt.astype(np.float64), n, w.bc, tol=1e-13, theta=theta)
        d_u0 = to_dev(u0.copy()); lam = to_dev(lam_T.copy())
        B.burgers_newton_adjoint(d_u0, lam, w.L, to_dev(nu), to_dev(dt), n, w.bc, theta=theta, tol=newton_tol)
        got = lam.cpu().numpy().astype(np.float64)
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert np.isfinite(got).all(), w.name
        assert (np.abs(got - ref) / scale).max() <= tol, (w.name, theta)
        np.testing.assert_array_equal(d_u0.cpu().numpy(), u0)          # u0 untouched


def test_newton_adjoint_against_finite_differences_of_the_gpu_forward_path(B):
    rng = np.random.default_rng(37)
    w = W.c3_periodic_btcs(B=2, N=256, n_steps=0)
    nu = np.full(2, 0.05)
    dt = oracle_dt(w.u0, w.L, nu, 4.0, w.bc, np.float64)
    n = 6
    lam_T = rng.standard_normal(w.u0.shape); v = rng.standard_normal(w.u0.shape)
    for theta in (1.0, 0.5):
        lam = to_dev(lam_T.copy())
        B.burgers_newton_adjoint(to_dev(w.u0), lam, w.L, to_dev(nu), to_dev(dt), n, w.bc, theta=theta)
        g = lam.cpu().numpy()
        eps = 1e-6

        def J(u0):
            u = to_dev(u0.copy()); B.burgers_newton(u, w.L, to_dev(nu), to_dev(dt), n, w.bc, tol=1e-13, theta=theta)
            return (lam_T * u.cpu().numpy()).sum(axis=1)
        fd = (J(w.u0 + eps * v) - J(w.u0 - eps * v)) / (2 * eps)
        an = (g * v).sum(axis=1)
        assert np.all(np.abs(fd - an) <= 1e-6 * (1 + np.abs(an))), theta
    lam = to_dev(lam_T.copy())
    B.burgers_newton_adjoint(to_dev(w.u0), lam, w.L, to_dev(nu), to_dev(dt), 0, w.bc)
    np.testing.assert_array_equal(lam.cpu().numpy(), lam_T)


@pytest.mark.parametrize("scheme", ["btcs", "newton"])
def test_implicit_adjoints_checkpointed(B, scheme):
    """Checkpoint segments of the implicit adjoints (burgers_*_adjoint_ckpt_*): any segment length gives the bits of
    the one-segment sweep (the recomputed states are those of the first sweep: p then q steps == p + q steps), the
    workspace shrinks as n/m + m, and a long grid (thread-per-system backward sweep) goes the same way."""
    rng = np.random.default_rng(41)
    for w, nu, n in ((W.c3_periodic_btcs(B=3, N=512, n_steps=0), np.full(3, 0.05), 17),
                     (W.c4b_long_btcs(N=12000, n_steps=0), np.full(1, 1e-3), 7)):
        dt = oracle_dt(w.u0, w.L, nu, 4.0, w.bc, np.float64)
        lam_T = rng.standard_normal(w.u0.shape)
        is_btcs = scheme == "btcs"
        fn = B.burgers_btcs_adjoint if is_btcs else B.burgers_newton_adjoint
        ref = (oracle.btcs_adjoint if is_btcs else oracle.newton_adjoint)(w.u0, lam_T, w.L, nu, dt, n, w.bc)
        want = None
        sizes = []
        for seg in (n, 1, 3, 5, n + 7, 0):
            lam = to_dev(lam_T.copy())
            fn(to_dev(w.u0), lam, w.L, to_dev(nu), to_dev(dt), n, w.bc, segment=seg)
            got = lam.cpu().numpy()
            if want is None:
                want = got
                assert (np.abs(got - ref) / np.abs(ref).max(axis=1, keepdims=True)).max() <= 1e-10, (w.name, seg)
            np.testing.assert_array_equal(got, want, err_msg=f"{w.name} segment {seg}")
            sizes.append(int(B.raw().burgers_implicit_adjoint_ckpt_workspace_bytes(
                B.OP_BTCS if is_btcs else B.OP_NEWTON, 1, w.u0.shape[0], w.u0.shape[1], w.bc, n, seg)))
        assert sizes[3] < sizes[0] and sizes[4] == sizes[0] and sizes[5] == sizes[0]     # 5-step segments < one segment
    # error paths
    one = to_dev(np.ones((1, 64)))
    with pytest.raises(B.BurgersError) as e:
        (B.burgers_btcs_adjoint if scheme == "btcs" else B.burgers_newton_adjoint)(
            one, one.clone(), 1.0, to_dev(np.array([0.1])), to_dev(np.array([1e-3])), 4, 0, segment=-1)
    assert e.value.status in (B.ERR_SHAPE, B.ERR_WORKSPACE)
