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
