"""GPU parity tests: the CUDA path (called through the C ABI) against the CPU oracle, element by
element, on the seeded synthetic workloads of DESIGN.md / BASELINE.json at sizes the oracle
finishes in seconds (several tiles / CTAs and ragged tails), plus cross-plan agreement (G10),
edge cases and API semantics.  Full-size configs: tests/test_gpu_fullsize.py."""
import math

import numpy as np
import pytest

import oracle
from parity import TOL, oracle_dt, rel_err, to_dev
from paper_2601_12204_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


def run_explicit(B, u0, L, nu, dt, n, bc, scheme, **kw):
    u = to_dev(u0.copy())
    B.burgers_explicit(u, L, to_dev(nu), to_dev(dt), n, bc, scheme, **kw)
    return u.cpu().numpy()


def run_btcs(B, u0, L, nu, dt, n, bc, **kw):
    u = to_dev(u0.copy())
    B.burgers_btcs(u, L, to_dev(nu), to_dev(dt), n, bc, **kw)
    return u.cpu().numpy()


def check_explicit(B, w, n, scheme, cfl=None, tol_scale=1.0, **kw):
    dt = oracle_dt(w.u0, w.L, w.nu, cfl or w.cfl, w.bc, w.dtype)
    ref = oracle.explicit(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64),
                          dt.astype(np.float64), n, w.bc, scheme)
    got = run_explicit(B, w.u0, w.L, w.nu, dt, n, w.bc, scheme, **kw)
    e = rel_err(got, ref, w.u0)
    assert e <= TOL[w.dtype] * tol_scale, (w.name, scheme, kw, e)
    return e


def check_btcs(B, w, n, cfl=None, **kw):
    dt = oracle_dt(w.u0, w.L, w.nu, cfl or w.cfl, w.bc, w.dtype)
    ref = oracle.btcs(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), dt.astype(np.float64),
                      n, w.bc)
    got = run_btcs(B, w.u0, w.L, w.nu, dt, n, w.bc, **kw)
    e = rel_err(got, ref, w.u0)
    assert e <= TOL[w.dtype], (w.name, kw, e)
    return e


# ------------------------------------------------------------------ dt_from_cfl (a1)
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", [(1, 3), (5, 17), (7, 256), (3, 4099), (2, 70001), (1, 1 << 20), (300, 1024),
                                   (700, 1024), (1000, 36), (600, 4100), (593, 2048)])   # >= 592 short rows: warp per row
def test_dt_from_cfl_matches_oracle(B, dtype, shape):
    rng = np.random.default_rng(7)
    Bn, N = shape
    u0 = (rng.standard_normal(shape) * 3).astype(dtype)
    nu = np.exp(rng.uniform(math.log(1e-4), math.log(1.0), Bn)).astype(dtype)
    for bc, L in ((B.BC_PERIODIC, 2 * math.pi), (B.BC_DIRICHLET, 1.0)):
        ref = oracle.dt_from_cfl(u0.astype(np.float64), L, nu.astype(np.float64), 0.4, bc).astype(dtype)
        got = B.dt_from_cfl(to_dev(u0), L, to_dev(nu), 0.4, bc).cpu().numpy()
        # same fp64 formula on the same inputs, rounded once: allow 2 ulp
        assert np.all(np.abs(got - ref) <= 2 * np.spacing(np.abs(ref))), (shape, bc)


def test_dt_from_cfl_zero_cases(B):
    u0 = np.zeros((3, 64)); u0[1, 5] = -2.0; u0[2, 63] = 4.0
    nu = np.array([0.1, 0.0, 0.0])
    got = B.dt_from_cfl(to_dev(u0), 64.0, to_dev(nu), 0.5, B.BC_PERIODIC).cpu().numpy()
    assert got[0] == 0.5 * 1.0 / (2 * 0.1)          # u == 0: diffusive bound
    assert got[1] == 0.5 * 1.0 / 2.0                # nu == 0: convective bound, |u| max = 2
    assert got[2] == 0.5 * 1.0 / 4.0                # Dirichlet-style end node counts too
    z = B.dt_from_cfl(to_dev(np.zeros((1, 8))), 1.0, to_dev(np.zeros(1)), 0.5, B.BC_PERIODIC).cpu().numpy()
    assert np.isinf(z[0]) and z[0] > 0


# ------------------------------------------------------------------ config 1 (worked on the GPU too)
def test_c1_sine_euler_rk4_btcs_vs_oracle_and_colehopf(B):
    from refs import colehopf_sin
    w = W.c1_sine()
    x = np.arange(w.N) * (w.L / w.N)
    exact = colehopf_sin(x, 1.0, 0.05)
    for scheme, C, name in ((B.SCHEME_EULER, 0.4, "euler"), (B.SCHEME_RK4, 0.8, "rk4"), (None, 4.0, "btcs")):
        dtc = oracle.dt_from_cfl(w.u0, w.L, w.nu, C, w.bc)[0]
        n, dt = W.steps_for_final_time(dtc, 1.0)
        dta = np.array([dt])
        if scheme is None:
            ref = oracle.btcs(w.u0, w.L, w.nu, dta, n, w.bc)
            got = run_btcs(B, w.u0, w.L, w.nu, dta, n, w.bc)
        else:
            ref = oracle.explicit(w.u0, w.L, w.nu, dta, n, w.bc, scheme)
            got = run_explicit(B, w.u0, w.L, w.nu, dta, n, w.bc, scheme)
        assert rel_err(got, ref, w.u0) <= 1e-10, name
        rms = math.sqrt(np.mean((got[0] - exact) ** 2))
        assert rms < 2.5e-2, (name, rms)        # first-order schemes at N=256 (G2: ~1.1e-2 / 1.8e-2)
    assert (n, name) == (42, "btcs")


def test_worked_example_4node_on_gpu(B):
    from refs import read_golden
    G = read_golden("worked_example_4node.txt")
    u4 = np.array([[1.0, 2.0, -1.0, 0.0]])
    nu = np.array([0.1]); dt = np.array([0.1])
    for plan in (B.PLAN_RESIDENT, B.PLAN_TILED):
        got = run_explicit(B, u4, 4.0, nu, dt, 1, B.BC_PERIODIC, B.SCHEME_EULER, plan=plan)
        np.testing.assert_allclose(got[0], G["euler_periodic"], atol=1e-14)
        got = run_explicit(B, u4, 4.0, nu, dt, 2, B.BC_PERIODIC, B.SCHEME_EULER, plan=plan)
        np.testing.assert_allclose(got[0], G["euler2_periodic"], atol=1e-14)
        got = run_explicit(B, u4, 4.0, nu, dt, 1, B.BC_PERIODIC, B.SCHEME_RK4, plan=plan)
        np.testing.assert_allclose(got[0], G["rk4_periodic"], atol=1e-14)
        got = run_explicit(B, u4, 3.0, nu, dt, 1, B.BC_DIRICHLET, B.SCHEME_EULER, plan=plan)
        np.testing.assert_allclose(got[0], G["euler_dirichlet"], atol=1e-14)
        got = run_explicit(B, u4, 3.0, nu, dt, 1, B.BC_DIRICHLET, B.SCHEME_RK4, plan=plan)
        np.testing.assert_allclose(got[0], G["rk4_dirichlet"], atol=1e-14)
    for plan in (B.PLAN_AUTO, B.PLAN_THOMAS):
        got = run_btcs(B, u4, 4.0, nu, dt, 1, B.BC_PERIODIC, plan=plan)
        np.testing.assert_allclose(got[0], G["btcs_periodic"], atol=1e-14)
        got = run_btcs(B, u4, 3.0, nu, dt, 1, B.BC_DIRICHLET, plan=plan)
        np.testing.assert_allclose(got[0], G["btcs_dirichlet"], atol=1e-14)


# ------------------------------------------------------------------ config 2 (reduced): Dirichlet Euler
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_c2_reduced_resident(B, dtype):
    w = W.c2_dirichlet_batch(B=24, N=4096, dtype=dtype)
    check_explicit(B, w, 3000, B.SCHEME_EULER)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("ppt", [1, 2, 4, 8, 16, 32])
def test_c2_reduced_every_points_per_thread(B, dtype, ppt):
    w = W.c2_dirichlet_batch(B=5, N=512, dtype=dtype)
    check_explicit(B, w, 700, B.SCHEME_EULER, plan=B.PLAN_RESIDENT, ppt=ppt)
    check_explicit(B, w, 150, B.SCHEME_RK4, cfl=0.8, plan=B.PLAN_RESIDENT, ppt=ppt)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_c2_reduced_tiled_matches(B, dtype):
    # same workload through the temporally blocked plan: several tiles, ragged last block of steps
    w = W.c2_dirichlet_batch(B=3, N=4096 * 3, dtype=dtype)
    check_explicit(B, w, 333, B.SCHEME_EULER, plan=B.PLAN_TILED)
    check_explicit(B, w, 50, B.SCHEME_RK4, cfl=0.8, plan=B.PLAN_TILED)
    check_explicit(B, w, 100, B.SCHEME_EULER, plan=B.PLAN_TILED, tblock=7, ppt=8)


# ------------------------------------------------------------------ config 5 (reduced): periodic RK4
def test_c5_reduced_rk4(B):
    w = W.c5_rk4_ensemble(n_steps=600, rows=np.arange(0, 65536, 2048))
    check_explicit(B, w, 600, B.SCHEME_RK4)
    check_explicit(B, w, 600, B.SCHEME_RK4, plan=B.PLAN_RESIDENT, ppt=32)   # one warp per trajectory
    check_explicit(B, w, 600, B.SCHEME_RK4, plan=B.PLAN_RESIDENT, ppt=8)
    w64 = W.c5_rk4_ensemble(n_steps=200, rows=np.arange(0, 65536, 8192), dtype=np.float64)
    check_explicit(B, w64, 200, B.SCHEME_RK4)
    check_explicit(B, w64, 200, B.SCHEME_EULER, cfl=0.4)


# ------------------------------------------------------------------ config 4a (reduced): long periodic grid
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_c4a_reduced_long_grid_tiled(B, dtype):
    w = W.c4a_long_explicit(N=(1 << 16) + 40, n_steps=500, dtype=dtype)   # ragged last tile
    assert B.plan_query(B.OP_EXPLICIT, dtype == np.float64, 1, w.N, w.bc, 0) == B.PLAN_TILED
    check_explicit(B, w, 500, B.SCHEME_EULER)
    check_explicit(B, w, 37, B.SCHEME_RK4, cfl=0.8)
    w2 = W.c4a_long_explicit(N=50021, n_steps=100, dtype=dtype)          # prime N: scalar loads
    check_explicit(B, w2, 100, B.SCHEME_EULER)


def test_odd_sizes_and_signs(B):
    rng = np.random.default_rng(11)
    for N in (3, 4, 5, 31, 33, 100, 201, 1000, 1023, 3001):
        for bc, L in ((B.BC_PERIODIC, 2.0), (B.BC_DIRICHLET, 1.0)):
            u0 = rng.uniform(-2, 2, (3, N))
            nu = rng.uniform(0.01, 0.1, 3)
            dt = oracle.dt_from_cfl(u0, L, nu, 0.4, bc)
            for scheme in (B.SCHEME_EULER, B.SCHEME_RK4):
                ref = oracle.explicit(u0, L, nu, dt, 25, bc, scheme)
                got = run_explicit(B, u0, L, nu, dt, 25, bc, scheme)
                assert rel_err(got, ref, u0) <= 1e-12, (N, bc, scheme)
                got = run_explicit(B, u0, L, nu, dt, 25, bc, scheme, plan=B.PLAN_TILED, tblock=4)
                assert rel_err(got, ref, u0) <= 1e-12, (N, bc, scheme, "tiled")
            ref = oracle.btcs(u0, L, nu, 10 * dt, 9, bc)
            got = run_btcs(B, u0, L, nu, 10 * dt, 9, bc, plan=B.PLAN_THOMAS)
            assert rel_err(got, ref, u0) <= 1e-12, (N, bc, "btcs-thomas")
            got = run_btcs(B, u0, L, nu, 10 * dt, 9, bc)
            assert rel_err(got, ref, u0) <= 1e-12, (N, bc, "btcs-auto")


# ------------------------------------------------------------------ config 3 (reduced): periodic BTCS
def test_c3_reduced_btcs_periodic(B):
    w = W.c3_periodic_btcs(B=40, N=2048, n_steps=60)
    assert B.plan_query(B.OP_BTCS, True, w.B, w.N, w.bc) == B.PLAN_HYBRID
    check_btcs(B, w, 60)
    check_btcs(B, w, 60, plan=B.PLAN_HYBRID)
    check_btcs(B, w, 60, plan=B.PLAN_THOMAS)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("N", [8, 16, 64, 128, 512, 1024, 4096])
def test_btcs_hybrid_sizes_and_time_steps(B, dtype, N):
    """HYBRID plan over its whole size range (P = 4, 8, 16; 2..256 threads), both boundary types,
    from tiny to huge diffusion numbers (PCR early exit and the full-depth 2x2 ending)."""
    rng = np.random.default_rng(N)
    for bc, L in ((B.BC_PERIODIC, 2 * math.pi), (B.BC_DIRICHLET, 1.0)):
        u0 = rng.uniform(-1.5, 2.5, (3, N)).astype(dtype)
        nu = rng.uniform(0.01, 0.1, 3).astype(dtype)
        for C in (0.05, 10.0, 3000.0):
            dt = oracle_dt(u0, L, nu, C, bc, dtype)
            ref = oracle.btcs(u0.astype(np.float64), L, nu.astype(np.float64), dt.astype(np.float64), 7, bc)
            got = run_btcs(B, u0, L, nu, dt, 7, bc, plan=B.PLAN_HYBRID)
            assert rel_err(got, ref, u0) <= TOL[np.dtype(dtype)], (N, bc, C)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("N", [7, 9, 11, 24, 100, 201, 1000, 2000, 3001, 4095])
def test_btcs_any_grid_length_fits_one_cta(B, dtype, N):
    """SURVEY 8(b) "any N >= 3 must work": grid lengths that are not P 2^k -- the paper's own N = 201
     among them -- run the resident HYBRID plan on ragged partitions (q or q + 1 rows per
    thread), periodic ring intact; none of them falls back to one thread per system."""
    rng = np.random.default_rng(N)
    for bc, L in ((B.BC_PERIODIC, 2 * math.pi), (B.BC_DIRICHLET, 1.0)):
        assert B.plan_query(B.OP_BTCS, dtype == np.float64, 5, N, bc) == B.PLAN_HYBRID
        x = np.arange(N) / N
        u0 = (rng.uniform(-1.5, 2.5, (5, 1)) * np.sin(2 * math.pi * x * rng.integers(1, 4, (5, 1)) + rng.uniform(0, 6, (5, 1)))
              + rng.uniform(-0.5, 1.0, (5, 1)) + 0.05 * rng.standard_normal((5, N))).astype(dtype)
        nu = rng.uniform(0.01, 0.1, 5).astype(dtype)
        # (fp32 at C = 3000: the rounding error of ANY solve, ~ (1 + 4r) eps with r ~ 1500, sits at the 1e-4 bar
        # itself; C = 300 takes the same full-depth PCR path with a factor 10 of room)
        for C in (0.05, 10.0, 3000.0 if dtype == np.float64 else 300.0):
            dt = oracle_dt(u0, L, nu, C, bc, dtype)
            ref = oracle.btcs(u0.astype(np.float64), L, nu.astype(np.float64), dt.astype(np.float64), 7, bc)
            got = run_btcs(B, u0, L, nu, dt, 7, bc)
            assert rel_err(got, ref, u0) <= TOL[np.dtype(dtype)], (N, bc, C)
            if bc == B.BC_DIRICHLET:
                np.testing.assert_array_equal(got[:, 0], u0[:, 0]); np.testing.assert_array_equal(got[:, -1], u0[:, -1])


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("shape", [(1, 10001), (1, 40003), (3, 12000), (2, 8196), (1, 300000 + 6)])
def test_btcs_any_grid_length_across_ctas(B, dtype, shape):
    """LONG plan on grid lengths that are neither powers of two nor multiples of the 16-byte vector (single
    systems) or of the tile: ragged last tile, element-wise wrap at the seam of the ring, ragged partitions
    in the cooperative fallback (driven at C = 3000)."""
    Bn, N = shape
    rng = np.random.default_rng(N)
    for bc, L in ((B.BC_PERIODIC, 2 * math.pi), (B.BC_DIRICHLET, 1.0)):
        assert B.plan_query(B.OP_BTCS, dtype == np.float64, Bn, N, bc) == B.PLAN_LONG
        x = np.arange(N) / N
        u0 = np.stack([a * np.sin(2 * math.pi * k * x + p) + m for a, k, p, m in
                       zip(rng.uniform(0.5, 2, Bn), (1, 3, 7), rng.uniform(0, 6, Bn), (-0.4, 0.0, 1.0))]).astype(dtype)
        nu = rng.uniform(0.01, 0.1, Bn).astype(dtype)
        # (fp32 at C = 3000: rounding error ~ (1 + 4r) eps is at the 1e-4 bar itself; C = 300 drives the fallback too)
        for C, plans in ((10.0, (B.PLAN_AUTO, B.PLAN_LONG_GENERAL)), (3000.0 if dtype == np.float64 else 300.0, (B.PLAN_AUTO,))):
            dt = oracle_dt(u0, L, nu, C, bc, dtype)
            ref = oracle.btcs(u0.astype(np.float64), L, nu.astype(np.float64), dt.astype(np.float64), 5, bc)
            for plan in plans:
                got = run_btcs(B, u0, L, nu, dt, 5, bc, plan=plan)
                assert rel_err(got, ref, u0) <= TOL[np.dtype(dtype)], (shape, bc, C, plan)


@pytest.mark.parametrize("shape", [(1, 5121), (2, 6000), (1, 7001), (5, 4098), (3, 5120)])
def test_btcs_sizes_around_the_hybrid_long_boundary(B, shape):
    """fp64 systems just above what one CTA holds (HYBRID: N <= 5120 on 512 threads x 10 slots) run LONG with only
    three or four tiles, whose halos wrap around the ring; just below, HYBRID with 512 threads."""
    Bn, N = shape
    rng = np.random.default_rng(N)
    for bc, L in ((B.BC_PERIODIC, 2 * math.pi), (B.BC_DIRICHLET, 1.0)):
        plan = B.plan_query(B.OP_BTCS, True, Bn, N, bc)
        assert plan == (B.PLAN_HYBRID if N <= 5120 else B.PLAN_LONG), (shape, plan)
        x = np.arange(N) / N
        u0 = np.stack([a * np.sin(2 * math.pi * k * x + p) + m for a, k, p, m in
                       zip(rng.uniform(0.5, 2, Bn), (1, 3, 7, 2, 5), rng.uniform(0, 6, Bn), (-0.4, 0.0, 1.0, 0.3, -1.0))])
        nu = rng.uniform(0.01, 0.1, Bn)
        for C in (10.0, 3000.0):
            dt = oracle_dt(u0, L, nu, C, bc, np.float64)
            ref = oracle.btcs(u0, L, nu, dt, 5, bc)
            got = run_btcs(B, u0, L, nu, dt, 5, bc)
            assert rel_err(got, ref, u0) <= 1e-10, (shape, bc, C)


def test_btcs_long_grid_of_four_million_and_forty_points(B):
    """N = 2^22 + 40 (the size VERDICT r01 names), fp64, periodic, C4b's profile and time step: the whole grid
    against the oracle after 6 steps."""
    w = W.c4b_long_btcs(N=(1 << 22) + 40, n_steps=6)
    assert B.plan_query(B.OP_BTCS, True, 1, w.N, w.bc) == B.PLAN_LONG
    check_btcs(B, w, 6)


@pytest.mark.parametrize("case", [(600_000, 3, 4), (600_000, 13, 5), (1 << 20, 9, 5), (3_000_000, 11, 5),
                                  (3_600_000, 9, 5), (6_000, 5, 7)])
def test_btcs_long_every_tile_shape(B, case):
    """LONG makes S steps per launch on tiles of 128 / 256 / 512 threads, whichever its cost model finds cheapest
    for the grid (btcs_long.cu: long_tile_shape).  One grid per shape -- (256, 2), (512, 6), (512, 4), (512, 5),
    (256, 4), (128, 1) in this order, identified by the launch count: multi-step launches + single-step
    remainder + fixup + GENERAL -- whole grid against the oracle, both boundary types, step counts that are not
    multiples of S (remainder launches, result ending in the workspace or in u)."""
    N, n_steps, launches = case
    for bc in (B.BC_PERIODIC, B.BC_DIRICHLET):
        w = W.c4b_long_btcs(N=N, n_steps=n_steps)
        assert B.plan_query(B.OP_BTCS, True, 1, N, bc) == B.PLAN_LONG
        assert B.launch_count(B.OP_BTCS, True, 1, N, bc, n_steps=n_steps) == launches
        dt = oracle_dt(w.u0, w.L, w.nu, w.cfl, bc, np.float64)
        ref = oracle.btcs(w.u0, w.L, w.nu, dt, n_steps, bc)
        got = run_btcs(B, w.u0, w.L, w.nu, dt, n_steps, bc)
        assert rel_err(got, ref, w.u0) <= 1e-10, (case, bc)
        general = run_btcs(B, w.u0, w.L, w.nu, dt, n_steps, bc, plan=B.PLAN_LONG_GENERAL)
        assert rel_err(got, general, w.u0) <= 1e-12, (case, bc)


def test_btcs_dirichlet_and_fp32(B):
    w = W.c2_dirichlet_batch(B=9, N=1000, dtype=np.float64)
    check_btcs(B, w, 40, cfl=10.0)
    check_btcs(B, w, 40, cfl=10.0, plan=B.PLAN_THOMAS)
    w32 = W.c3_periodic_btcs(B=6, N=512, n_steps=50, dtype=np.float32)
    check_btcs(B, w32, 50)
    w32d = W.c2_dirichlet_batch(B=6, N=512, dtype=np.float32)
    check_btcs(B, w32d, 50, cfl=10.0)


def test_c4b_reduced_long_btcs(B):
    """One long cyclic system across many CTAs (a7): the AUTO plan is LONG; its two device paths
    (overlapped tiles with the checked truncated PCR; cooperative global PCR) and the
    thread-per-system Thomas plan all agree with the oracle (G10)."""
    w = W.c4b_long_btcs(N=1 << 16, n_steps=12)
    assert B.plan_query(B.OP_BTCS, True, w.B, w.N, w.bc) == B.PLAN_LONG
    check_btcs(B, w, 12)
    check_btcs(B, w, 12, plan=B.PLAN_LONG)
    check_btcs(B, w, 12, plan=B.PLAN_LONG_GENERAL)
    check_btcs(B, w, 12, plan=B.PLAN_THOMAS)
    check_btcs(B, w, 5, plan=B.PLAN_LONG)             # odd step count: result ends in the workspace
    w2 = W.c4b_long_btcs(N=1 << 18, n_steps=7)
    check_btcs(B, w2, 7)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("C", [0.05, 10.0, 40.0, 3000.0])
def test_btcs_long_batches_boundaries_and_fallback(B, dtype, C):
    """LONG plan on small batches of long systems, both boundary types, mixed-sign data, from tiny
    to huge diffusion numbers.  C = 10 is BASELINE's "10x the explicit limit"; at C = 40 and 3000
    the couplings decay too slowly for the 128-point halo, so the tiled kernels must detect it
    (status word) and the cooperative kernel must take over from the failing step."""
    rng = np.random.default_rng(int(C * 100) + 1)
    for bc, L in ((B.BC_PERIODIC, 2 * math.pi), (B.BC_DIRICHLET, 1.0)):
        N = 1 << 14
        x = np.arange(N) / N
        u0 = np.stack([a * np.sin(2 * math.pi * k * x + p) + m for a, k, p, m in
                       zip(rng.uniform(0.5, 2, 3), (1, 3, 7), rng.uniform(0, 6, 3), (-0.4, 0.0, 1.0))]).astype(dtype)
        nu = rng.uniform(0.01, 0.1, 3).astype(dtype)
        dt = oracle_dt(u0, L, nu, C, bc, dtype)
        ref = oracle.btcs(u0.astype(np.float64), L, nu.astype(np.float64), dt.astype(np.float64), 6, bc)
        for plan in (B.PLAN_LONG, B.PLAN_LONG_GENERAL):
            got = run_btcs(B, u0, L, nu, dt, 6, bc, plan=plan)
            assert rel_err(got, ref, u0) <= TOL[np.dtype(dtype)], (bc, C, plan)


def test_btcs_long_convection_dominated_and_step_split(B):
    """nu tiny: the matrix is one-sided (|sub| ~ c, |sup| ~ 0 where u > 0), the slowest-decaying
    case for a given Courant number; and p then q steps == p+q steps bitwise (G6-v)."""
    N = 1 << 15
    x = np.arange(N) * (2 * math.pi / N)
    u0 = (1.0 + 0.8 * np.sin(x) * np.cos(3 * x))[None, :]
    nu = np.array([1e-7]); L = 2 * math.pi
    for C in (2.0, 10.0):
        dt = oracle_dt(u0, L, nu, C, B.BC_PERIODIC, np.float64)
        ref = oracle.btcs(u0, L, nu, dt, 9, B.BC_PERIODIC)
        a = run_btcs(B, u0, L, nu, dt, 9, B.BC_PERIODIC)
        assert rel_err(a, ref, u0) <= 1e-10, C
        b = run_btcs(B, run_btcs(B, u0, L, nu, dt, 4, B.BC_PERIODIC), L, nu, dt, 5, B.BC_PERIODIC)
        np.testing.assert_array_equal(a, b)


# ------------------------------------------------------------------ semantics
def test_zero_steps_and_step_splitting(B):
    w = W.c5_rk4_ensemble(n_steps=0, rows=np.arange(4), dtype=np.float64)
    dt = oracle_dt(w.u0, w.L, w.nu, 0.4, w.bc, w.dtype)
    same = run_explicit(B, w.u0, w.L, w.nu, dt, 0, w.bc, B.SCHEME_EULER)
    np.testing.assert_array_equal(same, w.u0)
    a = run_explicit(B, w.u0, w.L, w.nu, dt, 30, w.bc, B.SCHEME_EULER)
    b = run_explicit(B, run_explicit(B, w.u0, w.L, w.nu, dt, 11, w.bc, B.SCHEME_EULER), w.L, w.nu, dt, 19,
                     w.bc, B.SCHEME_EULER)
    np.testing.assert_array_equal(a, b)          # fp64: p then q steps == p+q steps, bitwise
    c = run_btcs(B, w.u0, w.L, w.nu, dt * 10, 6, w.bc)
    d = run_btcs(B, run_btcs(B, w.u0, w.L, w.nu, dt * 10, 2, w.bc), w.L, w.nu, dt * 10, 4, w.bc)
    np.testing.assert_array_equal(c, d)


def test_dirichlet_ends_never_move_and_max_principle(B):
    w = W.c2_dirichlet_batch(B=4, N=1024, dtype=np.float64)
    u0 = w.u0.copy(); u0[:, 0] = 0.75; u0[:, -1] = -0.5
    dt = oracle_dt(u0, w.L, w.nu, 0.4, w.bc, w.dtype)
    for got in (run_explicit(B, u0, w.L, w.nu, dt, 500, w.bc, B.SCHEME_EULER),
                run_explicit(B, u0, w.L, w.nu, dt, 100, w.bc, B.SCHEME_RK4),
                run_btcs(B, u0, w.L, w.nu, dt * 25, 20, w.bc)):
        np.testing.assert_array_equal(got[:, 0], u0[:, 0])
        np.testing.assert_array_equal(got[:, -1], u0[:, -1])
        assert np.all(got.max(axis=1) <= u0.max(axis=1) + 1e-12)
        assert np.all(got.min(axis=1) >= u0.min(axis=1) - 1e-12)


def test_host_entry_points_match_device_path(B):
    w = W.c2_dirichlet_batch(B=6, N=2048, dtype=np.float32)
    dt_h = B.dt_from_cfl_host(w.u0, w.L, w.nu, 0.4, w.bc)
    dt_d = B.dt_from_cfl(to_dev(w.u0), w.L, to_dev(w.nu), 0.4, w.bc).cpu().numpy()
    np.testing.assert_array_equal(dt_h, dt_d)
    uh = w.u0.copy()
    B.burgers_explicit_host(uh, w.L, w.nu, dt_h, 200, w.bc, B.SCHEME_EULER)
    ud = run_explicit(B, w.u0, w.L, w.nu, dt_h, 200, w.bc, B.SCHEME_EULER)
    np.testing.assert_array_equal(uh, ud)
    w3 = W.c3_periodic_btcs(B=5, N=256, n_steps=10)
    dt3 = B.dt_from_cfl_host(w3.u0, w3.L, w3.nu, 10.0, w3.bc)
    uh = w3.u0.copy()
    B.burgers_btcs_host(uh, w3.L, w3.nu, dt3, 10, w3.bc)
    np.testing.assert_array_equal(uh, run_btcs(B, w3.u0, w3.L, w3.nu, dt3, 10, w3.bc))


def test_solve_host_is_the_two_calls_in_one(B):
    """burgers_solve_host_*: one upload, CFL + time stepping on the device.  Bitwise the two-call host path
    (same kernels), and within the parity bar of the oracle run on the oracle's own dt."""
    w = W.c2_dirichlet_batch(B=6, N=2048, dtype=np.float32)
    for scheme, osch, cfl in ((B.SCHEME_EULER, oracle.EULER, 0.4), (B.SCHEME_RK4, oracle.RK4, 0.5)):
        u1, dt1 = B.burgers_solve_host(w.u0.copy(), w.L, w.nu, cfl, 150, w.bc, op=B.OP_EXPLICIT, scheme=scheme,
                                       return_dt=True)
        dt_h = B.dt_from_cfl_host(w.u0, w.L, w.nu, cfl, w.bc)
        np.testing.assert_array_equal(dt1, dt_h)
        u2 = B.burgers_explicit_host(w.u0.copy(), w.L, w.nu, dt_h, 150, w.bc, scheme)
        np.testing.assert_array_equal(u1, u2)
        ref = oracle.explicit(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), dt1.astype(np.float64), 150,
                              w.bc, osch)
        assert rel_err(u1, ref, w.u0) <= TOL[np.dtype(np.float32)]
    w3 = W.c3_periodic_btcs(B=5, N=256, n_steps=10)
    u1, dt1 = B.burgers_solve_host(w3.u0.copy(), w3.L, w3.nu, 10.0, 10, w3.bc, op=B.OP_BTCS, return_dt=True)
    ref_dt = oracle.dt_from_cfl(w3.u0, w3.L, w3.nu, 10.0, w3.bc)
    assert np.all(np.abs(dt1 - ref_dt) <= 2 * np.spacing(ref_dt))
    assert rel_err(u1, oracle.btcs(w3.u0, w3.L, w3.nu, dt1, 10, w3.bc), w3.u0) <= 1e-10
    u2 = B.burgers_btcs_host(w3.u0.copy(), w3.L, w3.nu, dt1, 10, w3.bc)
    np.testing.assert_array_equal(u1, u2)
    assert B.burgers_solve_host(w3.u0.copy(), w3.L, w3.nu, 10.0, 0, w3.bc, op=B.OP_BTCS).tolist() == w3.u0.tolist()
    with pytest.raises(Exception):
        B.burgers_solve_host(w3.u0.copy(), w3.L, w3.nu, 10.0, 1, w3.bc, op=B.OP_NEWTON)


def test_solve_host_in_two_halves_is_bitwise_the_single_pass(B):
    """Batches of >= 8 MB whose plan needs no workspace go through burgers_solve_host_* as two halves on two
    streams (copies overlap kernels).  Same plan, independent trajectories: the bits of the device path."""
    w = W.c5_rk4_ensemble(B=2051, N=1024, n_steps=0, dtype=np.float32)          # 8.4 MB, odd B: uneven halves
    for scheme, cfl, n in ((B.SCHEME_EULER, 0.4, 60), (B.SCHEME_RK4, 0.8, 25)):
        assert B.plan_query(B.OP_EXPLICIT, False, w.B, w.N, w.bc, scheme) == B.PLAN_RESIDENT
        u1, dt1 = B.burgers_solve_host(w.u0.copy(), w.L, w.nu, cfl, n, w.bc, op=B.OP_EXPLICIT, scheme=scheme,
                                       return_dt=True)
        dt_d = B.dt_from_cfl(to_dev(w.u0), w.L, to_dev(w.nu), cfl, w.bc)
        np.testing.assert_array_equal(dt1, dt_d.cpu().numpy())
        np.testing.assert_array_equal(u1, run_explicit(B, w.u0, w.L, w.nu, dt1, n, w.bc, scheme))
    w3 = W.c3_periodic_btcs(B=1030, N=1024, n_steps=0)                           # fp64, 8.4 MB, HYBRID
    assert B.plan_query(B.OP_BTCS, True, w3.B, w3.N, w3.bc) == B.PLAN_HYBRID
    u1, dt1 = B.burgers_solve_host(w3.u0.copy(), w3.L, w3.nu, 10.0, 6, w3.bc, op=B.OP_BTCS, return_dt=True)
    np.testing.assert_array_equal(u1, run_btcs(B, w3.u0, w3.L, w3.nu, dt1, 6, w3.bc))
    rows = np.array([0, 514, 515, 1029])
    assert rel_err(u1[rows], oracle.btcs(w3.u0[rows], w3.L, w3.nu[rows], dt1[rows], 6, w3.bc), w3.u0[rows]) <= 1e-10


def test_library_is_loaded_in_this_process(B):
    maps = open("/proc/self/maps").read()
    assert "libburgers.so" in maps


def test_plain_c_program_drives_the_kernels(B, tmp_path):
    """tests/c_abi_client.c `run`: a C99 program with nothing but burgers.h and libburgers.so runs the hot path
    (burgers_solve_host_f64: CFL step + Euler, CFL step + BTCS) on a 1 x 64 grid; compared with the oracle."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    libdir = os.path.join(root, "paper_2601_12204_b200")
    exe = str(tmp_path / "c_abi_client")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(root, "include"),
                    os.path.join(root, "tests", "c_abi_client.c"), "-o", exe, "-L", libdir, "-lburgers", "-lm",
                    "-Wl,-rpath," + libdir], check=True)
    r = subprocess.run([exe, "run"], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = r.stdout.strip().splitlines()
    L = 6.283185307179586
    u0 = (np.sin(L * np.arange(64) / 64.0) + 0.25)[None, :]
    nu = np.array([0.05])
    for k, (C, n, name) in enumerate(((0.4, 50, "euler"), (4.0, 7, "btcs"))):
        dt = float(lines[2 * k].split()[1])
        tag, *vals = lines[2 * k + 1].split()
        assert tag == name and len(vals) == 64
        dt_ref = oracle.dt_from_cfl(u0, L, nu, C, 0)
        assert abs(dt - dt_ref[0]) <= 2 * np.spacing(dt_ref[0])
        ref = (oracle.explicit(u0, L, nu, np.array([dt]), n, 0, 0) if name == "euler"
               else oracle.btcs(u0, L, nu, np.array([dt]), n, 0))
        assert rel_err(np.array([float(v) for v in vals])[None, :], ref, u0) <= 1e-10, name
