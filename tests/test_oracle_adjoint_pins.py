"""Pins of the oracle's discrete adjoint of forward Euler (D13)
against the (already pinned) forward oracle: the dot-product identity in the linear case, and central
finite differences of the forward map in the nonlinear case."""
import numpy as np
import pytest

import oracle

P, D = oracle.PERIODIC, oracle.DIRICHLET


@pytest.mark.parametrize("bc", [P, D])
@pytest.mark.parametrize("adv", [0.9, -0.6])
def test_linear_case_is_the_exact_transpose(bc, adv):
    # constant advection speed: u^N = M u^0 with a fixed matrix M, and the adjoint must be M^T:
    # <lam, M v> == <M^T lam, v> for arbitrary v, lam
    rng = np.random.default_rng(1)
    N, L, nu, dt, n = 37, 1.0, 0.02, 0.004, 25
    v, lam = rng.standard_normal(N), rng.standard_normal(N)
    Mv = oracle.explicit(v, L, nu, dt, n, bc, oracle.EULER, adv=adv)
    Mt_lam = oracle.explicit_adjoint(v, lam, L, nu, dt, n, bc, adv=adv)
    assert abs(lam @ Mv - Mt_lam @ v) <= 1e-13 * (np.abs(lam) @ np.abs(Mv) + 1)


@pytest.mark.parametrize("bc", [P, D])
def test_nonlinear_gradient_matches_finite_differences(bc):
    rng = np.random.default_rng(7)
    N, L, nu, n = 24, 1.0, 0.03, 40
    x = np.arange(N) / N
    u0 = 0.8 + 0.5 * np.sin(2 * np.pi * x) - 1.6 * (x > 0.6)       # both signs, away from zero at the nodes
    assert np.abs(u0).min() > 0.05
    dt = oracle.dt_from_cfl(u0, L, nu, 0.4, bc)[0]
    lam = rng.standard_normal(N)
    grad = oracle.explicit_adjoint(u0, lam, L, nu, dt, n, bc)
    # (the map is continuous but has kinks where a node value crosses zero; a +-1e-6 perturbation
    # straddles one only if some node is within ~1e-6 of zero at some step)
    eps = 1e-6
    for j in range(N):
        e = np.zeros(N); e[j] = eps
        Jp = lam @ oracle.explicit(u0 + e, L, nu, dt, n, bc, oracle.EULER)
        Jm = lam @ oracle.explicit(u0 - e, L, nu, dt, n, bc, oracle.EULER)
        fd = (Jp - Jm) / (2 * eps)
        assert abs(fd - grad[j]) <= 2e-7 * (1 + np.abs(grad).max()), (j, fd, grad[j])


def test_zero_steps_and_batches():
    rng = np.random.default_rng(2)
    u0 = rng.uniform(0.2, 1.0, (3, 16)); lam = rng.standard_normal((3, 16))
    np.testing.assert_array_equal(oracle.explicit_adjoint(u0, lam, 1.0, 0.1, 0.001, 0, P), lam)
    nu = np.array([0.05, 0.1, 0.2]); dt = np.array([1e-3, 2e-3, 5e-4])
    g = oracle.explicit_adjoint(u0, lam, 1.0, nu, dt, 9, P)
    for b in range(3):
        np.testing.assert_array_equal(g[b], oracle.explicit_adjoint(u0[b], lam[b], 1.0, nu[b], dt[b], 9, P))
