"""Differential test on RANDOM shapes: for seeded random (B, N, boundary type, dtype, CFL number) the AUTO plan of
every hot-path call agrees with the oracle -- grid lengths that are prime, odd, just above / below the plan
boundaries (resident / tiled, one CTA / many CTAs, vector-aligned or not).  SURVEY.md 8(b): "any N >= 3 must work"."""
import math

import numpy as np
import pytest

import oracle
from parity import TOL, oracle_dt, rel_err, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


def _data(rng, Bn, N, dtype):
    x = np.arange(N) / N
    k = rng.integers(1, 5, (Bn, 1))
    u0 = (rng.uniform(0.3, 2.0, (Bn, 1)) * np.sin(2 * math.pi * k * x + rng.uniform(0, 6, (Bn, 1))) + rng.uniform(-0.8, 0.8, (Bn, 1))
          + 0.02 * rng.standard_normal((Bn, N))).astype(dtype)
    nu = rng.uniform(0.01, 0.1, Bn).astype(dtype)
    return u0, nu


def _shapes(seed, n, Nmax):
    rng = np.random.default_rng(seed)
    special = [3, 4, 5, 6, 7, 31, 33, 63, 65, 127, 129, 201, 4095, 4097, 5119, 5120, 5121, 8191, 8193]
    out = []
    for i in range(n):
        N = int(special[i]) if i < len(special) and special[i] <= Nmax else int(rng.integers(3, Nmax))
        Bn = int(rng.choice([1, 2, 3, 7, 33]))
        out.append((Bn, N, int(rng.integers(0, 2)), np.float32 if rng.integers(0, 2) else np.float64))
    return out


@pytest.mark.parametrize("case", _shapes(11, 40, 12000), ids=lambda c: f"B{c[0]}-N{c[1]}-bc{c[2]}-{np.dtype(c[3]).name}")
def test_btcs_random_shapes(B, case):
    Bn, N, bc, dtype = case
    rng = np.random.default_rng(N * 7 + Bn)
    u0, nu = _data(rng, Bn, N, dtype)
    L = 2 * math.pi if bc == 0 else 1.0
    for C in (0.5, 10.0, 300.0):
        dt = oracle_dt(u0, L, nu, C, bc, dtype)
        ref = oracle.btcs(u0.astype(np.float64), L, nu.astype(np.float64), dt.astype(np.float64), 4, bc)
        u = to_dev(u0.copy())
        B.burgers_btcs(u, L, to_dev(nu), to_dev(dt), 4, bc)
        assert rel_err(u.cpu().numpy(), ref, u0) <= TOL[np.dtype(dtype)], (case, C)


@pytest.mark.parametrize("case", _shapes(12, 30, 40000), ids=lambda c: f"B{c[0]}-N{c[1]}-bc{c[2]}-{np.dtype(c[3]).name}")
def test_explicit_and_cfl_random_shapes(B, case):
    Bn, N, bc, dtype = case
    rng = np.random.default_rng(N * 5 + Bn)
    u0, nu = _data(rng, Bn, N, dtype)
    L = 2 * math.pi if bc == 0 else 1.0
    ref_dt = oracle.dt_from_cfl(u0.astype(np.float64), L, nu.astype(np.float64), 0.4, bc).astype(dtype)
    got_dt = B.dt_from_cfl(to_dev(u0), L, to_dev(nu), 0.4, bc).cpu().numpy()
    assert np.all(np.abs(got_dt - ref_dt) <= 2 * np.spacing(np.abs(ref_dt)))
    for scheme, C, n in ((0, 0.4, 37), (1, 0.8, 11)):
        dt = oracle_dt(u0, L, nu, C, bc, dtype)
        ref = oracle.explicit(u0.astype(np.float64), L, nu.astype(np.float64), dt.astype(np.float64), n, bc, scheme)
        u = to_dev(u0.copy())
        B.burgers_explicit(u, L, to_dev(nu), to_dev(dt), n, bc, scheme)
        assert rel_err(u.cpu().numpy(), ref, u0) <= TOL[np.dtype(dtype)], (case, scheme)


@pytest.mark.parametrize("case", _shapes(13, 20, 6000), ids=lambda c: f"B{c[0]}-N{c[1]}-bc{c[2]}-{np.dtype(c[3]).name}")
def test_newton_random_shapes(B, case):
    Bn, N, bc, dtype = case
    rng = np.random.default_rng(N * 3 + Bn)
    u0, _ = _data(rng, Bn, N, dtype)
    L = 2 * math.pi if bc == 0 else 1.0
    dx = L / N if bc == 0 else L / (N - 1)
    nu = np.maximum(0.05, 0.75 * np.abs(u0).max(axis=1) * dx).astype(dtype)       # cell Peclet number < 2 (D11)
    dt = oracle_dt(u0, L, nu, 2.0, bc, dtype)
    for theta in (1.0, 0.5):
        ref = oracle.newton_btcs(u0.astype(np.float64), L, nu.astype(np.float64), dt.astype(np.float64), 3, bc, tol=1e-13,
                                 theta=theta)
        u = to_dev(u0.copy())
        B.burgers_newton(u, L, to_dev(nu), to_dev(dt), 3, bc, tol=2e-6 if dtype == np.float32 else 1e-13, max_iter=30, theta=theta)
        assert rel_err(u.cpu().numpy(), ref, u0) <= TOL[np.dtype(dtype)], (case, theta)


@pytest.mark.parametrize("case", _shapes(14, 24, 7000), ids=lambda c: f"B{c[0]}-N{c[1]}-bc{c[2]}-{np.dtype(c[3]).name}")
def test_implicit_adjoints_random_shapes(B, case):
    """Reverse mode of the two implicit schemes (D15, D16) on random shapes: every register-slot count of the
    resident backward kernels (P = 4 .. 16, exact and ragged), the thread-per-system fallback beyond one CTA,
    both boundary types and dtypes, with a checkpoint segment that does not divide the step count."""
    Bn, N, bc, dtype = case
    rng = np.random.default_rng(N * 11 + Bn)
    u0, _ = _data(rng, Bn, N, dtype)
    L = 2 * math.pi if bc == 0 else 1.0
    dx = L / N if bc == 0 else L / (N - 1)
    nu = np.maximum(0.05, 0.75 * np.abs(u0).max(axis=1) * dx).astype(dtype)       # cell Peclet number < 2 (D11)
    lam_T = rng.standard_normal(u0.shape).astype(dtype)
    n = 5
    tol = TOL[np.dtype(dtype)]

    def check(got, ref, what):
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert np.isfinite(got).all(), (case, what)
        assert (np.abs(got.astype(np.float64) - ref) / scale).max() <= tol, (case, what)

    f64 = lambda a: a.astype(np.float64)
    dt = oracle_dt(u0, L, nu, 10.0, bc, dtype)
    ref = oracle.btcs_adjoint(f64(u0), f64(lam_T), L, f64(nu), f64(dt), n, bc)
    for seg in (0, 2):
        lam = to_dev(lam_T.copy())
        B.burgers_btcs_adjoint(to_dev(u0), lam, L, to_dev(nu), to_dev(dt), n, bc, segment=seg)
        check(lam.cpu().numpy(), ref, ("btcs", seg))
    dt = oracle_dt(u0, L, nu, 2.0, bc, dtype)
    for theta in (1.0, 0.5):
        ref = oracle.newton_adjoint(f64(u0), f64(lam_T), L, f64(nu), f64(dt), n, bc, tol=1e-13, theta=theta)
        lam = to_dev(lam_T.copy())
        B.burgers_newton_adjoint(to_dev(u0), lam, L, to_dev(nu), to_dev(dt), n, bc, theta=theta,
                                 tol=2e-6 if dtype == np.float32 else 1e-13, max_iter=30, segment=2)
        check(lam.cpu().numpy(), ref, ("newton", theta))
