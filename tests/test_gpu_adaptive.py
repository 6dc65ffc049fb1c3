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
