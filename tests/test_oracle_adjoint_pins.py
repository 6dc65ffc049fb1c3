"""Pins of the oracle's discrete adjoints of forward Euler (D13) and of classical RK4 (D14)
 against the (already pinned) forward oracle: the dot-product identity in the linear case, and central
finite differences of the forward map in the nonlinear case."""
import numpy as np
import pytest

import oracle

P, D = oracle.PERIODIC, oracle.DIRICHLET


SCHEMES = [oracle.EULER, oracle.RK4]


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("bc", [P, D])
@pytest.mark.parametrize("adv", [0.9, -0.6])
def test_linear_case_is_the_exact_transpose(bc, adv, scheme):
    # constant advection speed: u^N = M u^0 with a fixed matrix M, and the adjoint must be M^T:
    # <lam, M v> == <M^T lam, v> for arbitrary v, lam
    rng = np.random.default_rng(1)
    N, L, nu, dt, n = 37, 1.0, 0.02, 0.004, 25
    v, lam = rng.standard_normal(N), rng.standard_normal(N)
    Mv = oracle.explicit(v, L, nu, dt, n, bc, scheme, adv=adv)
    Mt_lam = oracle.explicit_adjoint(v, lam, L, nu, dt, n, bc, adv=adv, scheme=scheme)
    assert abs(lam @ Mv - Mt_lam @ v) <= 1e-13 * (np.abs(lam) @ np.abs(Mv) + 1)


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("bc", [P, D])
def test_nonlinear_gradient_matches_finite_differences(bc, scheme):
    rng = np.random.default_rng(7)
    N, L, nu, n = 24, 1.0, 0.03, 40
    x = np.arange(N) / N
    u0 = 0.8 + 0.5 * np.sin(2 * np.pi * x) - 1.6 * (x > 0.6)       # both signs, away from zero at the nodes
    assert np.abs(u0).min() > 0.05
    dt = oracle.dt_from_cfl(u0, L, nu, 0.4 if scheme == oracle.EULER else 0.8, bc)[0]
    lam = rng.standard_normal(N)
    grad = oracle.explicit_adjoint(u0, lam, L, nu, dt, n, bc, scheme=scheme)
    # (the map is continuous but has kinks where a node value crosses zero; a +-1e-6 perturbation
    # straddles one only if some node is within ~1e-6 of zero at some step)
    eps = 1e-6
    for j in range(N):
        e = np.zeros(N); e[j] = eps
        Jp = lam @ oracle.explicit(u0 + e, L, nu, dt, n, bc, scheme)
        Jm = lam @ oracle.explicit(u0 - e, L, nu, dt, n, bc, scheme)
        fd = (Jp - Jm) / (2 * eps)
        assert abs(fd - grad[j]) <= 2e-7 * (1 + np.abs(grad).max()), (j, fd, grad[j])


@pytest.mark.parametrize("scheme", SCHEMES)
def test_zero_steps_and_batches(scheme):
    rng = np.random.default_rng(2)
    u0 = rng.uniform(0.2, 1.0, (3, 16)); lam = rng.standard_normal((3, 16))
    np.testing.assert_array_equal(oracle.explicit_adjoint(u0, lam, 1.0, 0.1, 0.001, 0, P, scheme=scheme), lam)
    nu = np.array([0.05, 0.1, 0.2]); dt = np.array([1e-3, 2e-3, 5e-4])
    g = oracle.explicit_adjoint(u0, lam, 1.0, nu, dt, 9, P, scheme=scheme)
    for b in range(3):
        np.testing.assert_array_equal(g[b], oracle.explicit_adjoint(u0[b], lam[b], 1.0, nu[b], dt[b], 9, P, scheme=scheme))


def test_rk4_adjoint_of_one_step_is_the_transposed_step_matrix():
    """One RK4 step with a constant advection speed is u' = R(dt A) u with R(z) = 1 + z + z^2/2 + z^3/6 + z^4/24
    and A the (circulant) matrix of the D2 operator: the adjoint of one step must equal R(dt A)^T lam, built here
    from A assembled column by column with the pinned oracle.rhs -- no oracle adjoint code involved."""
    rng = np.random.default_rng(11)
    N, L, nu, dt, adv = 19, 1.0, 0.02, 0.004, 0.7
    A = np.stack([oracle.rhs(np.eye(N)[j], L, nu, P, adv=adv) for j in range(N)], axis=1)      # A[:, j] = F(e_j)
    Z = dt * A
    R = np.eye(N) + Z + Z @ Z / 2 + Z @ Z @ Z / 6 + Z @ Z @ Z @ Z / 24
    lam = rng.standard_normal(N)
    got = oracle.explicit_adjoint(rng.standard_normal(N), lam, L, nu, dt, 1, P, adv=adv, scheme=oracle.RK4)
    np.testing.assert_allclose(got, R.T @ lam, rtol=0, atol=1e-14)
    got3 = oracle.explicit_adjoint(rng.standard_normal(N), lam, L, nu, dt, 3, P, adv=adv, scheme=oracle.RK4)
    np.testing.assert_allclose(got3, np.linalg.matrix_power(R.T, 3) @ lam, rtol=0, atol=1e-14)


# ---------------------------------------------------------------- D15: adjoint of the lagged upwind BTCS scheme
@pytest.mark.parametrize("bc", [P, D])
@pytest.mark.parametrize("adv", [0.9, -0.6])
def test_btcs_adjoint_linear_case_is_the_exact_transpose(bc, adv):
    # constant advection speed: u^N = M u^0 with M = (A^{-1})^n; the adjoint must be M^T
    rng = np.random.default_rng(3)
    N, L, nu, dt, n = 33, 1.0, 0.02, 0.03, 9          # dt far above the explicit limit (r = nu dt/dx^2 ~ 0.65, c ~ 0.9)
    v, lam = rng.standard_normal(N), rng.standard_normal(N)
    Mv = oracle.btcs(v, L, nu, dt, n, bc, adv=adv)
    Mt_lam = oracle.btcs_adjoint(v, lam, L, nu, dt, n, bc, adv=adv)
    assert abs(lam @ Mv - Mt_lam @ v) <= 1e-13 * (np.abs(lam) @ np.abs(Mv) + 1)


@pytest.mark.parametrize("bc", [P, D])
def test_btcs_adjoint_of_one_step_against_the_dense_formula(bc):
    """One step: du' = A^{-1} (I - D) du with A from the pinned oracle.btcs_rows and D written out here in numpy (dense
    matrices, numpy.linalg): the adjoint must be (I - D) A^{-T} lam."""
    rng = np.random.default_rng(5)
    N, L, nu, dt = 12, 1.0, 0.05, 0.04
    u = rng.uniform(-1.0, 1.5, N)
    u[np.abs(u) < 0.1] += 0.3
    lam = rng.standard_normal(N)
    sub, diag, sup, _ = oracle.btcs_rows(u, L, nu, dt, bc)
    dx = L / N if bc == P else L / (N - 1)
    A = np.diag(diag) + np.diag(sub[1:], -1) + np.diag(sup[:-1], 1)
    if bc == P:
        A[0, N - 1] = sub[0]; A[N - 1, 0] = sup[N - 1]
    else:
        A[0, :] = 0; A[0, 0] = 1; A[N - 1, :] = 0; A[N - 1, N - 1] = 1
    up = oracle.btcs(u, L, nu, dt, 1, bc)
    np.testing.assert_allclose(A @ up, u, atol=1e-13)                 # (the step itself, for the record)
    Dv = np.where(u > 0, up - np.roll(up, 1), np.roll(up, -1) - up) * dt / dx
    if bc == D:
        Dv[0] = Dv[-1] = 0.0
    want = (1.0 - Dv) * np.linalg.solve(A.T, lam)
    got = oracle.btcs_adjoint(u, lam, L, nu, dt, 1, bc)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)


@pytest.mark.parametrize("bc", [P, D])
def test_btcs_adjoint_matches_finite_differences(bc):
    rng = np.random.default_rng(8)
    N, L, nu, n = 24, 1.0, 0.03, 12
    x = np.arange(N) / N
    u0 = 0.8 + 0.5 * np.sin(2 * np.pi * x) - 1.6 * (x > 0.6)       # both signs, away from zero at the nodes
    dt = 10 * oracle.dt_from_cfl(u0, L, nu, 0.4, bc)[0]            # the hot path's "10x the explicit limit"
    lam = rng.standard_normal(N)
    grad = oracle.btcs_adjoint(u0, lam, L, nu, dt, n, bc)
    eps = 1e-6
    for j in range(N):
        e = np.zeros(N); e[j] = eps
        Jp = lam @ oracle.btcs(u0 + e, L, nu, dt, n, bc)
        Jm = lam @ oracle.btcs(u0 - e, L, nu, dt, n, bc)
        fd = (Jp - Jm) / (2 * eps)
        assert abs(fd - grad[j]) <= 2e-7 * (1 + np.abs(grad).max()), (j, fd, grad[j])


def test_btcs_adjoint_zero_steps_and_batches():
    rng = np.random.default_rng(2)
    u0 = rng.uniform(0.2, 1.0, (3, 16)); lam = rng.standard_normal((3, 16))
    np.testing.assert_array_equal(oracle.btcs_adjoint(u0, lam, 1.0, 0.1, 0.01, 0, P), lam)
    nu = np.array([0.05, 0.1, 0.2]); dt = np.array([1e-2, 2e-2, 5e-3])
    g = oracle.btcs_adjoint(u0, lam, 1.0, nu, dt, 5, P)
    for b in range(3):
        np.testing.assert_array_equal(g[b], oracle.btcs_adjoint(u0[b], lam[b], 1.0, nu[b], dt[b], 5, P))


# ---------------------------------------------------------------- D16: reverse mode of the Newton / theta-scheme
THETAS = [1.0, 0.5, 0.3]


def _dense_G_prime(v, h, r, bc, adv=None):
    """d G / d v written out densely (numpy): G_i(v) = h a_i (v_{i+1} - v_{i-1}) - r (v_{i+1} - 2 v_i + v_{i-1}),
    a_i = v_i (or the constant adv), cyclic neighbours; rows of Dirichlet end nodes are zero (M G')."""
    N = len(v)
    Gp = np.zeros((N, N))
    for i in range(N):
        if bc == D and i in (0, N - 1):
            continue
        im, ip = (i - 1) % N, (i + 1) % N
        a = v[i] if adv is None else adv
        Gp[i, im] += -h * a - r
        Gp[i, ip] += h * a - r
        Gp[i, i] += 2 * r + (h * (v[ip] - v[im]) if adv is None else 0.0)
    return Gp


@pytest.mark.parametrize("theta", THETAS)
@pytest.mark.parametrize("bc", [P, D])
@pytest.mark.parametrize("adv", [0.9, -0.6])
def test_newton_adjoint_linear_case_is_the_exact_transpose(bc, adv, theta):
    # constant multiplier: u^N = S^n u^0 with S = (I + theta G')^{-1} (I - (1 - theta) G'); the adjoint must be S^T
    rng = np.random.default_rng(13)
    N, L, nu, dt, n = 21, 1.0, 0.02, 0.01, 7
    v, lam = rng.standard_normal(N), rng.standard_normal(N)
    Sv = oracle.newton_btcs(v, L, nu, dt, n, bc, tol=1e-14, adv=adv, theta=theta)
    St_lam = oracle.newton_adjoint(v, lam, L, nu, dt, n, bc, tol=1e-14, adv=adv, theta=theta)
    assert abs(lam @ Sv - St_lam @ v) <= 1e-12 * (np.abs(lam) @ np.abs(Sv) + 1)
    dx = L / N if bc == P else L / (N - 1)
    Gp = _dense_G_prime(v, dt / (2 * dx), nu * dt / dx**2, bc, adv)
    S = np.linalg.solve(np.eye(N) + theta * Gp, np.eye(N) - (1 - theta) * Gp)
    np.testing.assert_allclose(St_lam, np.linalg.matrix_power(S.T, n) @ lam, rtol=0, atol=1e-12)


@pytest.mark.parametrize("theta", THETAS)
@pytest.mark.parametrize("bc", [P, D])
def test_newton_adjoint_of_one_step_against_the_dense_formula(bc, theta):
    """One step from u to the root w (pinned forward oracle): dw/du = (I + theta M G'(w))^{-1} (I - (1 - theta) M G'(u))
    with G' written out densely here; the adjoint must be the transpose applied to lam (numpy.linalg)."""
    rng = np.random.default_rng(17)
    N, L, nu, dt = 14, 1.0, 0.05, 0.004
    u = rng.uniform(-1.0, 1.5, N)
    lam = rng.standard_normal(N)
    dx = L / N if bc == P else L / (N - 1)
    h, r = dt / (2 * dx), nu * dt / dx**2
    w = oracle.newton_btcs(u, L, nu, dt, 1, bc, tol=1e-14, theta=theta)
    Jw = np.eye(N) + theta * _dense_G_prime(w, h, r, bc)
    Ku = np.eye(N) - (1 - theta) * _dense_G_prime(u, h, r, bc)
    want = Ku.T @ np.linalg.solve(Jw.T, lam)
    got = oracle.newton_adjoint(u, lam, L, nu, dt, 1, bc, tol=1e-14, theta=theta)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-12)


@pytest.mark.parametrize("theta", [1.0, 0.5])
@pytest.mark.parametrize("bc", [P, D])
def test_newton_adjoint_matches_finite_differences(bc, theta):
    rng = np.random.default_rng(19)
    N, L, nu, n = 24, 1.0, 0.03, 10
    x = np.arange(N) / N
    u0 = 0.8 + 0.5 * np.sin(2 * np.pi * x) - 1.6 * (x > 0.6)       # both signs, a jump
    dt = 4 * oracle.dt_from_cfl(u0, L, nu, 0.4, bc)[0]             # implicit step, cell Peclet number < 2
    lam = rng.standard_normal(N)
    grad = oracle.newton_adjoint(u0, lam, L, nu, dt, n, bc, tol=1e-14, theta=theta)
    eps = 1e-6
    for j in range(N):
        e = np.zeros(N); e[j] = eps
        Jp = lam @ oracle.newton_btcs(u0 + e, L, nu, dt, n, bc, tol=1e-14, theta=theta)
        Jm = lam @ oracle.newton_btcs(u0 - e, L, nu, dt, n, bc, tol=1e-14, theta=theta)
        fd = (Jp - Jm) / (2 * eps)
        assert abs(fd - grad[j]) <= 2e-7 * (1 + np.abs(grad).max()), (j, fd, grad[j])


def test_newton_adjoint_theta_zero_is_the_explicit_central_transpose_and_batches():
    rng = np.random.default_rng(23)
    u0 = rng.uniform(0.2, 1.0, (3, 16)); lam = rng.standard_normal((3, 16))
    np.testing.assert_array_equal(oracle.newton_adjoint(u0, lam, 1.0, 0.1, 0.01, 0, P), lam)
    # theta = 0: w = u - G(u) explicitly, J = I, so one step's adjoint is (I - G'(u))^T lam
    N, L, nu, dt = 16, 1.0, 0.1, 1e-3
    dx = L / N
    Gp = _dense_G_prime(u0[0], dt / (2 * dx), nu * dt / dx**2, P)
    np.testing.assert_allclose(oracle.newton_adjoint(u0[0], lam[0], L, nu, dt, 1, P, theta=0.0),
                               (np.eye(N) - Gp).T @ lam[0], rtol=0, atol=1e-14)
    nu = np.array([0.05, 0.1, 0.2]); dt = np.array([1e-3, 2e-3, 5e-4])
    g = oracle.newton_adjoint(u0, lam, 1.0, nu, dt, 5, P, theta=0.5)
    for b in range(3):
        np.testing.assert_array_equal(g[b], oracle.newton_adjoint(u0[b], lam[b], 1.0, nu[b], dt[b], 5, P, theta=0.5))
