"""Pins of the oracle's Newton-Raphson fully-implicit BTCS (D11; Eq.10-15),
against things other than itself: the 4-node example iterated in exact rational arithmetic, a
finite-difference Jacobian, the exact Fourier amplification factor of the linearised scheme, the
Cole-Hopf solution (second-order convergence -- central convection -- where the upwind schemes of the
hot path give first order), and invariants."""
import math

import numpy as np
import pytest

import oracle
from refs import amplification, colehopf_sin, read_golden

P, D = oracle.PERIODIC, oracle.DIRICHLET
U4 = np.array([1.0, 2.0, -1.0, 0.0])


def test_worked_example_residual_jacobian_and_iterates():
    G = read_golden("newton_4node.txt")
    np.testing.assert_allclose(oracle.newton_residual(U4, U4, 4.0, 0.1, 0.1, P), G["F0_periodic"], atol=1e-15)
    sub, diag, sup = oracle.newton_jacobian(U4, 4.0, 0.1, 0.1, P)
    np.testing.assert_allclose(sub, G["J0_sub_periodic"], atol=1e-15)
    np.testing.assert_allclose(diag, G["J0_diag_periodic"], atol=1e-15)
    np.testing.assert_allclose(sup, G["J0_sup_periodic"], atol=1e-15)
    for k in (1, 2, 3):     # tol = 0: exactly k iterations
        w = oracle.newton_btcs(U4, 4.0, 0.1, 0.1, 1, P, tol=0.0, max_iter=k)
        np.testing.assert_allclose(w, G[f"newton{k}_periodic"], atol=2e-15)
        w = oracle.newton_btcs(U4, 3.0, 0.1, 0.1, 1, D, tol=0.0, max_iter=k)
        np.testing.assert_allclose(w, G[f"newton{k}_dirichlet"], atol=2e-15)


@pytest.mark.parametrize("bc", [P, D])
def test_jacobian_is_the_derivative_of_the_residual(bc):
    rng = np.random.default_rng(5)
    N, L, nu, dt = 9, 2.0, 0.07, 0.03
    w, un = rng.uniform(-2, 2, N), rng.uniform(-2, 2, N)
    sub, diag, sup = oracle.newton_jacobian(w, L, nu, dt, bc)
    J = np.zeros((N, N))
    for i in range(N):
        J[i, (i - 1) % N] += sub[i]; J[i, i] += diag[i]; J[i, (i + 1) % N] += sup[i]
    eps = 1e-6
    for j in range(N):
        if bc == D and j in (0, N - 1):
            continue                      # frozen nodes are not unknowns
        e = np.zeros(N); e[j] = eps
        col = (oracle.newton_residual(w + e, un, L, nu, dt, bc) - oracle.newton_residual(w - e, un, L, nu, dt, bc)) / (2 * eps)
        rows = range(N) if bc == P else range(1, N - 1)
        for i in rows:
            assert abs(col[i] - J[i, j]) < 1e-8, (i, j)


@pytest.mark.parametrize("adv", [0.8, -1.7])
def test_linearised_scheme_has_the_central_btcs_amplification_factor(adv):
    # constant advection speed: F is linear, ONE Newton iteration per step is exact, and a Fourier
    # mode is multiplied by G = 1 / (1 + i c sin(theta) + 4 r sin^2(theta/2)), c = adv dt/dx
    N, L, nu, k, n = 32, 2 * math.pi, 0.03, 3, 7
    dx = L / N
    dt = 0.9 * dx
    theta = 2 * math.pi * k / N
    c, r = adv * dt / dx, nu * dt / dx ** 2
    Gf = 1.0 / (1.0 + 1j * c * math.sin(theta) + 4 * r * math.sin(theta / 2) ** 2)
    i = np.arange(N)
    u0 = np.cos(theta * i + 0.4)
    got, iters = oracle.newton_btcs(u0, L, nu, dt, n, P, tol=1e-12, max_iter=10, adv=adv, return_iters=True)
    want = np.real(Gf ** n * np.exp(1j * (theta * i + 0.4)))
    np.testing.assert_allclose(got, want, atol=1e-13)
    assert iters[0] == n
    # the upwind factor of refs.amplification("btcs") is a different number: the pin can tell them apart
    assert abs(Gf - amplification("btcs", theta, abs(c), r, math.copysign(1.0, adv))) > 1e-3


def _c1_newton(N, tol=1e-12):
    L, nu = 2 * math.pi, 0.05
    x = np.arange(N) * (L / N)
    u0 = np.sin(2 * math.pi * np.arange(N) / N)
    dtc = oracle.dt_from_cfl(u0, L, nu, 4.0, P)[0]
    n = int(math.ceil(1.0 / dtc - 1e-12))
    u, it = oracle.newton_btcs(u0, L, nu, 1.0 / n, n, P, tol=tol, return_iters=True)
    err = u - colehopf_sin(x, 1.0, nu)
    return n, int(it[0]), math.sqrt(np.mean(err ** 2))


def test_colehopf_second_order_and_iteration_counts():
    res = {N: _c1_newton(N) for N in (128, 256, 512)}
    e = [res[N][2] for N in (128, 256, 512)]
    # dt ~ dx^2: O(dt) + O(dx^2) = second order, 1.82 -> 1.96 -> 1.99 (the upwind BTCS of the hot path is
    # first order: 1.80e-2 at N=256 against 4.2e-3 here)
    o1, o2 = math.log2(e[0] / e[1]), math.log2(e[1] / e[2])
    assert 1.7 < o1 < 2.05 and 1.9 < o2 < 2.05 and o2 > o1, e
    assert 3.5e-3 < e[1] < 5e-3
    n, it, _ = _c1_newton(256, tol=1e-6)          # the paper's criterion
    assert n == 42 and 2 * n <= it <= 4 * n       # quadratic convergence: 2-3 iterations per step


def test_converged_state_satisfies_eq11():
    rng = np.random.default_rng(8)
    N, L = 64, 1.0
    u0 = rng.uniform(-1, 1, (3, N))
    nu = np.array([0.05, 0.1, 0.2])
    dt = oracle.dt_from_cfl(u0, L, nu, 4.0, P)
    u1 = oracle.newton_btcs(u0, L, nu, dt, 1, P, tol=1e-13)
    for b in range(3):
        F = oracle.newton_residual(u1[b], u0[b], L, nu[b], dt[b], P)
        assert np.abs(F).max() < 1e-13
        # written out independently (numpy), Eq.11
        dx = L / N
        w = u1[b]
        F2 = w - u0[b] + dt[b] * (w * (np.roll(w, -1) - np.roll(w, 1)) / (2 * dx)
                                  - nu[b] * (np.roll(w, -1) - 2 * w + np.roll(w, 1)) / dx ** 2)
        assert np.abs(F2).max() < 1e-12


def test_invariants_and_threads():
    N, L = 40, 2.0
    const = np.full((1, N), 0.7)
    u, it = oracle.newton_btcs(const, L, 0.1, 0.05, 5, P, return_iters=True)
    np.testing.assert_array_equal(u, const)
    assert it[0] == 0                                            # residual is exactly zero
    i = np.arange(N)
    odd = np.sin(2 * math.pi * i / N); odd[0] = 0.0; odd[N // 2] = 0.0
    odd[N // 2 + 1:] = -odd[1:N // 2][::-1]
    u = oracle.newton_btcs(odd, L, 0.05, 0.02, 6, P, tol=1e-13)
    np.testing.assert_allclose(u[1:], -u[1:][::-1], atol=1e-14)
    ud = np.linspace(1.0, -0.5, N) + 0.1 * np.sin(7 * i)
    got = oracle.newton_btcs(ud, L, 0.05, 0.02, 6, D, tol=1e-13)
    assert got[0] == ud[0] and got[-1] == ud[-1]
    rng = np.random.default_rng(3)
    ub = rng.uniform(-1, 1, (6, N))
    a = oracle.newton_btcs(ub, L, 0.1, 0.01, 4, P, threads=1)
    b = oracle.newton_btcs(ub, L, 0.1, 0.01, 4, P, threads=4)
    np.testing.assert_array_equal(a, b)


# ---------------------------------------------------------------- theta-scheme
def test_theta_half_worked_example():
    G = read_golden("newton_4node.txt")
    for k in (1, 2, 3):
        w = oracle.newton_btcs(U4, 4.0, 0.1, 0.1, 1, P, tol=0.0, max_iter=k, theta=0.5)
        np.testing.assert_allclose(w, G[f"cn{k}_periodic"], atol=2e-15)
        w = oracle.newton_btcs(U4, 3.0, 0.1, 0.1, 1, D, tol=0.0, max_iter=k, theta=0.5)
        np.testing.assert_allclose(w, G[f"cn{k}_dirichlet"], atol=2e-15)


@pytest.mark.parametrize("theta", [0.5, 0.25, 1.0])
def test_theta_scheme_amplification_factor(theta):
    # linearised: G = (1 - (1-theta) zeta) / (1 + theta zeta), zeta = i c sin(th) + 4 r sin^2(th/2)
    N, L, nu, k, n, adv = 32, 2 * math.pi, 0.03, 5, 9, 1.3
    dx = L / N
    dt = 0.7 * dx
    th = 2 * math.pi * k / N
    zeta = 1j * (adv * dt / dx) * math.sin(th) + 4 * (nu * dt / dx ** 2) * math.sin(th / 2) ** 2
    Gf = (1 - (1 - theta) * zeta) / (1 + theta * zeta)
    i = np.arange(N)
    u0 = np.cos(th * i - 0.3)
    got = oracle.newton_btcs(u0, L, nu, dt, n, P, tol=1e-13, adv=adv, theta=theta)
    np.testing.assert_allclose(got, np.real(Gf ** n * np.exp(1j * (th * i - 0.3))), atol=1e-13)


def test_theta_zero_is_forward_euler_with_central_convection():
    rng = np.random.default_rng(2)
    N, L, nu, dt = 24, 3.0, 0.1, 0.004
    u0 = rng.uniform(-1, 1, N)
    dx = L / N
    want = u0 - dt * (u0 * (np.roll(u0, -1) - np.roll(u0, 1)) / (2 * dx)
                      - nu * (np.roll(u0, -1) - 2 * u0 + np.roll(u0, 1)) / dx ** 2)
    got, it = oracle.newton_btcs(u0, L, nu, dt, 1, P, tol=1e-14, theta=0.0, return_iters=True)
    np.testing.assert_allclose(got, want, atol=1e-15)
    assert it[0] == 1        # J = I: one (trivial) iteration


def test_crank_nicolson_is_second_order_with_dt_proportional_to_dx():
    # dt = dx/4 (NOT dx^2): Crank-Nicolson O(dt^2 + dx^2) keeps order 2, BTCS (theta = 1) drops to order 1
    L, nu = 2 * math.pi, 0.05

    def err(N, theta):
        x = np.arange(N) * (L / N)
        n = int(round(1.0 / (0.25 * L / N)))
        u = oracle.newton_btcs(np.sin(x), L, nu, 1.0 / n, n, P, tol=1e-13, theta=theta)
        return math.sqrt(np.mean((u - colehopf_sin(x, 1.0, nu)) ** 2))

    e_cn = [err(N, 0.5) for N in (128, 256, 512)]
    e_be = [err(N, 1.0) for N in (128, 256, 512)]
    o_cn = [math.log2(e_cn[i] / e_cn[i + 1]) for i in range(2)]
    o_be = [math.log2(e_be[i] / e_be[i + 1]) for i in range(2)]
    assert all(1.9 < o < 2.1 for o in o_cn), (e_cn, o_cn)
    assert all(0.85 < o < 1.35 for o in o_be), (e_be, o_be)
    assert e_cn[2] < 0.2 * e_be[2]
