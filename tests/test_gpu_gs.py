"""GPU parity of the Gauss-Seidel BTCS (D12): same sweep order as the
oracle, so iterates agree to rounding and the sweep counts agree except at tolerance ties."""
import math

import numpy as np
import pytest

import oracle
from parity import rel_err, to_dev
from refs import read_golden
from paper_2601_12204_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


def run(B, u0, L, nu, dt, n, bc, tol, max_iter=1000):
    import torch
    u = to_dev(np.ascontiguousarray(u0).copy())
    it = torch.zeros(u.shape[0], dtype=torch.int64, device="cuda")
    B.burgers_btcs_gs(u, L, to_dev(nu), to_dev(dt), n, bc, tol=tol, max_iter=max_iter, iters_out=it)
    return u.cpu().numpy(), it.cpu().numpy()


def test_worked_example_sweeps_on_gpu(B):
    G = read_golden("newton_4node.txt")
    u4 = np.array([[1.0, 2.0, -1.0, 0.0]]); nu = np.array([0.1]); dt = np.array([0.1])
    for k in (1, 2, 3):
        got, it = run(B, u4, 4.0, nu, dt, 1, B.BC_PERIODIC, tol=0.0, max_iter=k)
        np.testing.assert_allclose(got[0], G[f"gs{k}_periodic"], atol=1e-14)
        assert it[0] == k
        got, _ = run(B, u4, 3.0, nu, dt, 1, B.BC_DIRICHLET, tol=0.0, max_iter=k)
        np.testing.assert_allclose(got[0], G[f"gs{k}_dirichlet"], atol=1e-14)


@pytest.mark.parametrize("dtype,tol,bar", [(np.float64, 1e-6, 1e-10), (np.float64, 1e-12, 1e-10), (np.float32, 1e-5, 1e-4)])
def test_parity_and_sweep_counts(B, dtype, tol, bar):
    for w, C, n in ((W.c3_periodic_btcs(B=9, N=201, n_steps=0, dtype=dtype), 0.4, 30),
                    (W.c2_dirichlet_batch(B=5, N=333, dtype=dtype), 2.0, 12)):
        dt = oracle.dt_from_cfl(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), C, w.bc).astype(dtype)
        ref, it_ref = oracle.btcs_gs(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), dt.astype(np.float64), n,
                                     w.bc, tol=tol, return_iters=True)
        got, it = run(B, w.u0, w.L, w.nu, dt, n, w.bc, tol=tol)
        # same sweeps in the same order: iterates agree to rounding unless a residual sits exactly at tol
        assert rel_err(got, ref, w.u0) <= max(bar, 3 * tol), w.name
        if dtype == np.float64:
            assert np.all(np.abs(it - it_ref) <= n), (it, it_ref)
        direct = oracle.btcs(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), dt.astype(np.float64), n, w.bc)
        assert rel_err(got, direct, w.u0) <= 10 * n * tol + bar      # converges to the direct solution


def test_paper_setting_sweeps_per_step(B):
    N, L, nu = 201, 2.0, 0.01
    x = np.arange(N) * (L / N)
    u0 = np.sin(math.pi * x)[None, :]
    dt = oracle.dt_from_cfl(u0, L, np.array([nu]), 0.4, 0)
    _, it = run(B, u0, L, np.array([nu]), dt, 100, 0, tol=1e-6)
    assert 5.5 <= it[0] / 100 <= 7.5          # "5-7 iterations per step"


@pytest.mark.parametrize("N,bc_name", [(64, "p"), (1000, "p"), (1024, "d"), (1025, "p"), (2048, "p"), (2047, "d"),
                                       (2049, "d"), (4096, "p"), (4095, "d"), (63, "p"), (4097, "p")])
def test_cta_plan_shapes(B, N, bc_name):
    """Every branch of the plan choice (CTA per system with 4 or 8 rows per thread and 1..16 warps, ragged
    last threads, and the thread-per-system plan on both sides of its range) against the oracle."""
    if bc_name == "p":
        w = W.c3_periodic_btcs(B=3, N=N, n_steps=0)
    else:
        w = W.c2_dirichlet_batch(B=3, N=N, dtype=np.float64)
    n = 6
    dt = oracle.dt_from_cfl(w.u0, w.L, w.nu, 0.4, w.bc)
    ref, it_ref = oracle.btcs_gs(w.u0, w.L, w.nu, dt, n, w.bc, tol=1e-9, return_iters=True)
    got, it = run(B, w.u0, w.L, w.nu, dt, n, w.bc, tol=1e-9)
    assert rel_err(got, ref, w.u0) <= 1e-10, (N, bc_name)
    assert np.all(np.abs(it - it_ref) <= n), (it, it_ref)
    assert it.min() >= n                                   # at least one sweep per step at this tolerance
    # max_iter caps the sweeps of every step
    got2, it2 = run(B, w.u0, w.L, w.nu, dt, n, w.bc, tol=0.0, max_iter=3)
    ref2 = oracle.btcs_gs(w.u0, w.L, w.nu, dt, n, w.bc, tol=0.0, max_iter=3)
    assert np.all(it2 == 3 * n)
    assert rel_err(got2, ref2, w.u0) <= 1e-10
