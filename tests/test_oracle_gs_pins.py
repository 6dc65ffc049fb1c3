"""Pins of the oracle's Gauss-Seidel BTCS (D12): exact-rational
sweeps of the 4-node example, convergence to the DIRECT solution of the same system (itself pinned by
dense Gaussian elimination) within the bound the M-matrix gives, and the sweep counts the paper reports."""
import math

import numpy as np
import pytest

import oracle
from refs import read_golden

P, D = oracle.PERIODIC, oracle.DIRICHLET
U4 = np.array([1.0, 2.0, -1.0, 0.0])


def test_worked_example_sweeps():
    G = read_golden("newton_4node.txt")
    for k in (1, 2, 3):     # tol = 0: exactly k sweeps
        x, it = oracle.btcs_gs(U4, 4.0, 0.1, 0.1, 1, P, tol=0.0, max_iter=k, return_iters=True)
        np.testing.assert_allclose(x, G[f"gs{k}_periodic"], atol=2e-15)
        assert it[0] == k
        x = oracle.btcs_gs(U4, 3.0, 0.1, 0.1, 1, D, tol=0.0, max_iter=k)
        np.testing.assert_allclose(x, G[f"gs{k}_dirichlet"], atol=2e-15)


@pytest.mark.parametrize("bc", [P, D])
def test_converges_to_the_direct_solution_within_the_residual_bound(bc):
    rng = np.random.default_rng(12)
    N, L = 50, 1.0
    u0 = rng.uniform(-2, 2, (4, N))
    nu = rng.uniform(0.01, 0.1, 4)
    dt = oracle.dt_from_cfl(u0, L, nu, 3.0, bc)
    direct = oracle.btcs(u0, L, nu, dt, 1, bc)
    for tol in (1e-3, 1e-6, 1e-13):
        x = oracle.btcs_gs(u0, L, nu, dt, 1, bc, tol=tol, max_iter=100000)
        # A is an M-matrix with row sums 1 (D4): ||A^-1||_inf <= 1, so |x - x*| <= max residual < tol
        assert np.abs(x - direct).max() <= tol + 1e-14, tol


def test_sweep_counts_match_the_paper():
    # the paper's setting: N = 201, nu = 0.01, CFL-sized dt, max residual < 1e-6 -> "5-7 iterations"
    N, L, nu = 201, 2.0, 0.01
    x = np.arange(N) * (L / N)
    u0 = np.sin(math.pi * x)
    for C, lo, hi in ((0.2, 4.0, 6.0), (0.4, 5.5, 7.5), (0.8, 9.0, 12.0)):      # measured: 4.9, 6.6, 10.4
        dt = oracle.dt_from_cfl(u0, L, nu, C, P)[0]
        _, it = oracle.btcs_gs(u0, L, nu, dt, 100, P, tol=1e-6, return_iters=True)
        assert lo <= it[0] / 100 <= hi, (C, it[0] / 100)
    # ten times the explicit limit (r = 5): Gauss-Seidel contracts like (2r/(1+2r))^2 = 0.83 per sweep
    dt = oracle.dt_from_cfl(u0, L, nu, 10.0, P)[0]
    _, it = oracle.btcs_gs(u0, L, nu, dt, 10, P, tol=1e-6, return_iters=True)
    assert it[0] / 10 > 30


def test_invariants():
    const = np.full((1, 16), -0.3)
    x, it = oracle.btcs_gs(const, 1.0, 0.1, 0.01, 3, P, return_iters=True)
    np.testing.assert_allclose(x, const, atol=1e-16)
    assert it[0] == 0
    ud = np.linspace(1.0, -0.5, 30) + 0.05 * np.sin(np.arange(30))
    got = oracle.btcs_gs(ud, 1.0, 0.05, 0.01, 4, D, tol=1e-12)
    assert got[0] == ud[0] and got[-1] == ud[-1]
    assert got.max() <= ud.max() + 1e-12 and got.min() >= ud.min() - 1e-12
    rng = np.random.default_rng(3)
    ub = rng.uniform(-1, 1, (5, 33))
    np.testing.assert_array_equal(oracle.btcs_gs(ub, 1.0, 0.1, 0.01, 3, P, threads=1),
                                  oracle.btcs_gs(ub, 1.0, 0.1, 0.01, 3, P, threads=4))
