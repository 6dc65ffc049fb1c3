"""burgers_btcs_noalloc (include/burgers.h): BTCS time stepping with the library's built-in scratch array, for
callers that cannot allocate.  Its output against the stock path's (burgers_btcs_* with a caller-provided
workspace) on calls made back to back -- the array is shared by all calls and keeps the last call's contents --
and the rejection beyond the 32 MiB limit.  Collected last on purpose (the file name): the suite runs with
`pytest -x`, and a failure here must not hide the tests of the hot path."""
import ctypes
import math

import numpy as np
import pytest

from parity import TOL, oracle_dt, rel_err, to_dev
from paper_2601_12204_b200 import workloads as W


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


def _cases(B):
    """(name, u0, L, nu, dt, n_steps, bc): shapes whose AUTO plan needs scratch memory."""
    out = []
    # one long periodic fp64 grid, C4b's profile: LONG plan (ping-pong state + status words), odd step count
    w = W.c4b_long_btcs(N=1 << 18, n_steps=9)
    out.append(("long_f64", w.u0, w.L, w.nu, oracle_dt(w.u0, w.L, w.nu, w.cfl, w.bc, w.dtype), 9, w.bc))
    # a small batch of long Dirichlet fp32 systems, mixed signs
    rng = np.random.default_rng(1220499)
    N = 12000
    x = np.arange(N) / (N - 1)
    u0 = np.stack([a * np.sin(2 * math.pi * k * x + p) + m for a, k, p, m in
                   zip(rng.uniform(0.5, 2, 3), (1, 3, 7), rng.uniform(0, 6, 3), (-0.4, 0.0, 1.0))]).astype(np.float32)
    nu = rng.uniform(0.01, 0.1, 3).astype(np.float32)
    out.append(("batch_f32", u0, 1.0, nu, oracle_dt(u0, 1.0, nu, 10.0, B.BC_DIRICHLET, np.float32), 6, B.BC_DIRICHLET))
    # C = 40: the halo check of the tiled kernels fails and the cooperative kernel takes over (interface rows)
    N = 1 << 14
    x = np.arange(N) / N
    u0 = np.stack([np.sin(2 * math.pi * x) + 0.3, 1.5 * np.cos(6 * math.pi * x)]).astype(np.float64)
    nu = np.array([0.02, 0.05])
    L = 2 * math.pi
    out.append(("fallback_f64", u0, L, nu, oracle_dt(u0, L, nu, 40.0, B.BC_PERIODIC, np.float64), 5, B.BC_PERIODIC))
    return out


def _stock(B, u0, L, nu, dt, n, bc):
    u = to_dev(u0.copy())
    B.burgers_btcs(u, L, to_dev(nu), to_dev(dt), n, bc)          # workspace allocated by the binding (torch)
    return u.cpu().numpy()


def _noalloc(B, u0, L, nu, dt, n, bc):
    u = to_dev(u0.copy())
    B.burgers_btcs_noalloc(u, L, to_dev(nu), to_dev(dt), n, bc)
    return u.cpu().numpy()


@pytest.mark.gpu
def test_noalloc_matches_the_stock_path_on_calls_in_a_row(B):
    import torch
    cases = _cases(B)
    for name, u0, L, nu, dt, n, bc in cases:
        is64 = u0.dtype == np.float64
        assert B.plan_query(B.OP_BTCS, is64, u0.shape[0], u0.shape[1], bc) == B.PLAN_LONG, name
        need = B.workspace_bytes(B.OP_BTCS, is64, u0.shape[0], u0.shape[1], bc)
        assert 0 < need <= B.noalloc_scratch_bytes(), name
    want = [_stock(B, *c[1:]) for c in cases]
    # twice through all cases, back to back: every call finds the previous call's contents in the array
    for rnd in range(2):
        for (name, u0, L, nu, dt, n, bc), ref in zip(cases, want):
            got = _noalloc(B, u0, L, nu, dt, n, bc)
            assert np.isfinite(got).all(), (rnd, name)
            assert rel_err(got, ref, u0) <= TOL[np.dtype(u0.dtype)], (rnd, name)
    # the same call twice in a row on ONE stream, no host synchronisation in between
    name, u0, L, nu, dt, n, bc = cases[0]
    a, b = to_dev(u0.copy()), to_dev(u0.copy())
    dnu, ddt = to_dev(nu), to_dev(dt)
    B.burgers_btcs_noalloc(a, L, dnu, ddt, n, bc)
    B.burgers_btcs_noalloc(b, L, dnu, ddt, n, bc)
    torch.cuda.synchronize()
    assert rel_err(a.cpu().numpy(), want[0], u0) <= TOL[np.dtype(u0.dtype)]
    assert rel_err(b.cpu().numpy(), want[0], u0) <= TOL[np.dtype(u0.dtype)]


@pytest.mark.gpu
def test_noalloc_rejects_beyond_the_limit_and_leaves_u_alone(B):
    w = W.c4b_long_btcs(N=1 << 22, n_steps=2)                     # needs 80 MiB of scratch
    assert B.workspace_bytes(B.OP_BTCS, True, 1, w.N, w.bc) > B.noalloc_scratch_bytes()
    u = to_dev(w.u0.copy())
    dt = to_dev(oracle_dt(w.u0, w.L, w.nu, w.cfl, w.bc, w.dtype))
    with pytest.raises(B.BurgersError) as e:
        B.burgers_btcs_noalloc(u, w.L, to_dev(w.nu), dt, 2, w.bc)
    assert e.value.status == B.ERR_LIMIT
    np.testing.assert_array_equal(u.cpu().numpy(), w.u0)
    assert B.raw().burgers_noalloc_init() == B.OK                 # set-up alone, idempotent
    assert B.raw().burgers_noalloc_init() == B.OK


def test_noalloc_limit_and_argument_errors_need_no_gpu(B):
    """The size check comes before anything touches the device."""
    lib = B.raw()
    assert B.noalloc_scratch_bytes() == 32 << 20
    assert "scratch" in B.strerror(B.ERR_LIMIT)
    buf = (ctypes.c_double * 8)()
    one = ctypes.cast(buf, ctypes.c_void_p)
    f = lib.burgers_btcs_noalloc
    assert f(1, one, 1, 1 << 22, 1.0, one, one, 1, 0, None) == B.ERR_LIMIT
    assert f(0, one, 64, 1 << 20, 1.0, one, one, 1, 0, None) == B.ERR_LIMIT
    assert f(1, None, 1, 1 << 16, 1.0, one, one, 1, 0, None) == B.ERR_NULL
    assert f(1, one, 1, 1 << 16, 1.0, None, one, 1, 0, None) == B.ERR_NULL
    assert f(1, one, 0, 1 << 16, 1.0, one, one, 1, 0, None) == B.ERR_SHAPE
    assert f(1, one, 1, 1 << 16, 1.0, one, one, -1, 0, None) == B.ERR_SHAPE
    assert f(1, one, 1, 1 << 16, 1.0, one, one, 1, 7, None) == B.ERR_ENUM
    assert f(1, one, 1, 1 << 16, 0.0, one, one, 1, 0, None) == B.ERR_VALUE
