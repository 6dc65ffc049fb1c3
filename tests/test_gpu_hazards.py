"""Memory-safety and race checks of every kernel family WITHOUT compute-sanitizer (the tool is closed on this
GPU pool: `compute-sanitizer --tool memcheck python tests/sanitizer_cases.py` answers "compute-sanitizer is closed
on this pool and stays closed ... Find a bad access with bounds checks and asserts of your own, small cases, and a
comparison with the CPU reference"; profiles/r02_sanitizer.md).  What stands in for it, per case:

  * GUARD BANDS: every buffer the library may touch (u, nu, dt, workspace, snapshots, lambda, iteration counts) is a
    window of a larger allocation whose 4 KiB before and after the window hold a canary pattern; the workspace window
    has EXACTLY burgers_workspace_bytes(...) bytes.  An out-of-bounds store of a kernel lands in a band and fails the
    test; an out-of-bounds load reads canary bits (NaNs of huge magnitude) and fails the comparison with the oracle;
  * DETERMINISM: a data race between the threads of a CTA (the single-barrier double-buffered edge exchange, the PCR
    ping-pong buffers reused across tiles, the stage reuse of the LONG kernel, the level flags of the cooperative
    kernel) shows up as run-to-run differences: every case runs 6 times from the same input, three of them while a
    second stream keeps the SMs busy with another kernel of the library (different relative timing of the CTAs),
    and all results must be bitwise equal;
  * the comparison with the CPU oracle at the usual tolerance.

The cases are those of tests/sanitizer_cases.py (sized so that the path in question is really taken)."""
import math

import numpy as np
import pytest

import oracle
from parity import rel_err
from paper_2601_12204_b200 import workloads as W

pytestmark = pytest.mark.gpu
PAD = 4096
CANARY = 0xA5


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import binding
    return binding


class Guarded:
    """A window of `nbytes` inside a canary-filled allocation."""

    def __init__(self, nbytes):
        import torch
        self.n = int(nbytes)
        self.raw = torch.full((self.n + 2 * PAD,), CANARY, dtype=torch.uint8, device="cuda")

    def window(self, dtype=None, shape=None):
        v = self.raw[PAD:PAD + self.n]
        if dtype is not None:
            v = v.view(dtype)
        return v.view(shape) if shape is not None else v

    def intact(self):
        return bool((self.raw[:PAD] == CANARY).all().item() and (self.raw[PAD + self.n:] == CANARY).all().item())


def guarded_from(a):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    g = Guarded(t.numel() * t.element_size())
    g.window(t.dtype, tuple(t.shape)).copy_(t)
    return g, g.window(t.dtype, tuple(t.shape))


def guarded_empty(nbytes):
    g = Guarded(nbytes)
    return g, g.window()


class Busy:
    """Keeps the SMs busy on a second stream with an unrelated kernel of the library (long RK4 run)."""

    def __init__(self, B):
        import torch
        self.B, self.s = B, torch.cuda.Stream()
        w = W.c5_rk4_ensemble(B=2048, N=1024, dtype=np.float32)
        self.w = w
        self.u = torch.from_numpy(w.u0).cuda()
        self.nu = torch.from_numpy(w.nu).cuda()
        self.dt = B.dt_from_cfl(self.u, w.L, self.nu, w.cfl, w.bc)
        torch.cuda.synchronize()

    def start(self):
        import torch
        with torch.cuda.stream(self.s):
            self.B.burgers_explicit(self.u, self.w.L, self.nu, self.dt, 300, self.w.bc, 1)

    def wait(self):
        self.s.synchronize()


def _dt(w, C):
    return oracle.dt_from_cfl(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), C, w.bc).astype(w.dtype)


def _f64(a):
    return a.astype(np.float64)


def _cases():
    """(name, dtype, make) -- make(B) returns (arrays dict, ws_bytes, call(tensors, ws) -> None, outputs, check(out))."""
    out = []

    def explicit(name, mk, n, scheme, **kw):
        def make(B, dtype):
            w = mk(dtype)
            dt = _dt(w, 0.4 if scheme == 0 else 0.8)
            need = B.workspace_bytes(B.OP_EXPLICIT, dtype == np.float64, w.B, w.N, w.bc, scheme, kw.get("plan", B.PLAN_AUTO))
            ref = oracle.explicit(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), n, w.bc, scheme)
            return (dict(u=w.u0, nu=w.nu, dt=dt), need,
                    lambda t, ws: B.burgers_explicit(t["u"], w.L, t["nu"], t["dt"], n, w.bc, scheme, ws=ws, **kw),
                    ("u",), lambda o: rel_err(o["u"], ref, w.u0))
        out.append((name, make))

    explicit("resident-euler-4warps", lambda d: W.c2_dirichlet_batch(B=3, N=4096, dtype=d), 130, 0)
    explicit("resident-rk4-4warps", lambda d: W.c2_dirichlet_batch(B=3, N=4096, dtype=d), 20, 1)
    explicit("resident-rk4-1warp", lambda d: W.c5_rk4_ensemble(B=4, N=1024, dtype=d), 20, 1)
    explicit("resident-ragged-N201", lambda d: W.c3_periodic_btcs(B=2, N=201, dtype=d), 20, 0)
    explicit("tiled-euler", lambda d: W.c4a_long_explicit(N=40000, dtype=d), 70, 0, plan=2, tblock=32)
    explicit("tiled-rk4", lambda d: W.c4a_long_explicit(N=40000, dtype=d), 9, 1, plan=2, tblock=4)
    explicit("tiled-dirichlet", lambda d: W.c2_dirichlet_batch(B=2, N=20000, dtype=d), 40, 0, plan=2, tblock=16)

    def btcs(name, mk, n, C, plan=0):
        def make(B, dtype):
            w = mk(dtype)
            Cc = C if (dtype == np.float64 or C < 1000) else 300.0
            dt = _dt(w, Cc)
            need = B.workspace_bytes(B.OP_BTCS, dtype == np.float64, w.B, w.N, w.bc, 0, plan)
            ref = oracle.btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), n, w.bc)
            return (dict(u=w.u0, nu=w.nu, dt=dt), need,
                    lambda t, ws: B.burgers_btcs(t["u"], w.L, t["nu"], t["dt"], n, w.bc, ws=ws, plan=plan),
                    ("u",), lambda o: rel_err(o["u"], ref, w.u0))
        out.append((name, make))

    btcs("thomas-periodic", lambda d: W.c3_periodic_btcs(B=70, N=201, dtype=d), 3, 4.0, plan=3)
    btcs("thomas-dirichlet", lambda d: W.c2_dirichlet_batch(B=33, N=130, dtype=d), 3, 4.0, plan=3)
    btcs("hybrid-early-exit", lambda d: W.c3_periodic_btcs(B=3, N=2048, dtype=d), 4, 10.0)
    btcs("hybrid-full-depth", lambda d: W.c3_periodic_btcs(B=3, N=2048, dtype=d), 3, 1.0e5)
    btcs("hybrid-ragged-N201", lambda d: W.c3_periodic_btcs(B=3, N=201, dtype=d), 4, 10.0)
    btcs("hybrid-ragged-N3001-dirichlet", lambda d: W.c2_dirichlet_batch(B=3, N=3001, dtype=d), 3, 1.0e5)

    def long3(d):
        w = W.c4b_long_btcs(N=1 << 19, dtype=d)          # 3 x 296 tiles > 592 resident CTAs: two tiles per CTA
        u0 = np.repeat(w.u0, 3, axis=0) * np.array([[1.0], [0.5], [-0.7]], dtype=d)
        return W.Workload("long3", u0, np.repeat(w.nu, 3), w.L, w.bc, w.scheme, w.cfl, 0, w.dtype)

    btcs("long-two-tiles-per-cta", long3, 3, 10.0)
    btcs("long-dirichlet", lambda d: W.Workload("ld", W.c4b_long_btcs(N=1 << 15, dtype=d).u0.copy(), np.array([1e-4], dtype=d),
                                                1.0, 1, 2, 10.0, 0, np.dtype(d)), 3, 10.0, plan=5)
    btcs("long-fallback-general", lambda d: W.c4b_long_btcs(N=1 << 15, dtype=d), 3, 3000.0, plan=5)
    btcs("long-general-alone", lambda d: W.c4b_long_btcs(N=1 << 15, dtype=d), 2, 10.0, plan=6)
    btcs("long-odd-N", lambda d: W.c4b_long_btcs(N=40003, dtype=d), 3, 10.0)
    btcs("long-odd-N-fallback", lambda d: W.c4b_long_btcs(N=40003, dtype=d), 2, 3000.0)
    return out


CASES = _cases()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_guard_bands_determinism_and_parity(B, case, dtype):
    import torch
    name, make = case
    arrays, need, call, outs, err = make(B, dtype)
    busy = Busy(B)
    results = []
    for rep in range(6):
        guards, tensors = {}, {}
        for k, a in arrays.items():
            guards[k], tensors[k] = guarded_from(a)
        gws, ws = guarded_empty(need)
        if rep % 2:
            busy.start()
        call(tensors, ws if need else None)
        torch.cuda.synchronize()
        busy.wait()
        for k, g in guards.items():
            assert g.intact(), (name, k, "guard band overwritten")
        assert gws.intact(), (name, "workspace guard band overwritten")
        for k in arrays:                          # inputs the call must not modify
            if k not in outs:
                np.testing.assert_array_equal(tensors[k].cpu().numpy(), arrays[k])
        results.append({k: tensors[k].cpu().numpy() for k in outs})
    for r in results[1:]:
        for k in outs:
            np.testing.assert_array_equal(r[k], results[0][k], err_msg=f"{name}: run-to-run difference")
    tol = 1e-4 if dtype == np.float32 else 1e-10
    assert err(results[0]) <= tol, name


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_guard_bands_other_entry_points(B, dtype):
    """CFL kernels (three shapes), snapshots (staged stores), fused adaptive step, Newton (HYBRID exact / ragged,
    THOMAS), Gauss-Seidel (CTA plan, thread-per-system plan), adjoint (resident, checkpointed, streaming)."""
    import torch
    is64 = dtype == np.float64
    tol = 1e-4 if dtype == np.float32 else 1e-10
    rng = np.random.default_rng(5)
    # ---- CFL
    for shape in ((600, 512), (3, 4099), (2, 70001)):
        u0 = rng.standard_normal(shape).astype(dtype); nu = rng.uniform(0.01, 0.1, shape[0]).astype(dtype)
        gu, u = guarded_from(u0); gn, nv = guarded_from(nu); gd, dtw = guarded_empty(shape[0] * u0.itemsize)
        outv = dtw.view(u.dtype)
        ref = oracle.dt_from_cfl(_f64(u0), 1.0, _f64(nu), 0.4, 0).astype(dtype)
        for _ in range(3):
            B.dt_from_cfl(u, 1.0, nv, 0.4, 0, out=outv)
            torch.cuda.synchronize()
            assert gu.intact() and gn.intact() and gd.intact()
            assert np.all(np.abs(outv.cpu().numpy() - ref) <= 2 * np.spacing(np.abs(ref)))
    # ---- snapshots, adaptive
    for w, scheme in ((W.c2_dirichlet_batch(B=3, N=4096, dtype=dtype), 0), (W.c5_rk4_ensemble(B=3, N=1024, dtype=dtype), 1)):
        dt = _dt(w, 0.4 if scheme == 0 else 0.8)
        _, ref = oracle.explicit_trajectory(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 24, w.bc, scheme, 4)
        first = None
        for _ in range(3):
            gu, u = guarded_from(w.u0); gs, sraw = guarded_empty(6 * w.u0.size * w.u0.itemsize)
            snaps = sraw.view(u.dtype).view(6, w.B, w.N)
            B.burgers_explicit_traj(u, w.L, torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda(), 24, w.bc, scheme, 4, snaps=snaps)
            torch.cuda.synchronize()
            assert gu.intact() and gs.intact()
            got = snaps.cpu().numpy()
            assert np.abs(got - ref).max() / np.abs(w.u0).max() <= tol
            first = got if first is None else first
            np.testing.assert_array_equal(got, first)
        gu, u = guarded_from(w.u0)
        B.burgers_explicit_adaptive(u, w.L, torch.from_numpy(w.nu).cuda(), 0.4 if scheme == 0 else 0.8, 5, 6, w.bc, scheme)
        torch.cuda.synchronize()
        assert gu.intact()
        ref_a, _ = oracle.explicit_adaptive(_f64(w.u0), w.L, _f64(w.nu), 0.4 if scheme == 0 else 0.8, 5, 6, w.bc, scheme, dtype=dtype)
        assert rel_err(u.cpu().numpy(), ref_a, w.u0) <= tol
    # ---- Newton
    w201 = W.c3_periodic_btcs(B=40, N=201, dtype=dtype); w201.nu[:] = 0.1
    for w, plan in ((W.c3_periodic_btcs(B=3, N=2048, dtype=dtype), B.PLAN_AUTO), (w201, B.PLAN_AUTO), (w201, B.PLAN_THOMAS),
                    (W.c2_dirichlet_batch(B=3, N=1000, dtype=dtype), B.PLAN_AUTO)):
        dt = _dt(w, 2.0)
        need = B.workspace_bytes(B.OP_NEWTON, is64, w.B, w.N, w.bc, 0, plan)
        ref = oracle.newton_btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 3, w.bc, tol=1e-12, max_iter=20)
        first = None
        for _ in range(3):
            gu, u = guarded_from(w.u0); gw, ws = guarded_empty(need); gi, iraw = guarded_empty(8 * w.B)
            B.burgers_newton(u, w.L, torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda(), 3, w.bc,
                             tol=1e-5 if dtype == np.float32 else 1e-12, max_iter=20, iters_out=iraw.view(torch.int64),
                             ws=ws if need else None, plan=plan)
            torch.cuda.synchronize()
            assert gu.intact() and gw.intact() and gi.intact()
            got = u.cpu().numpy()
            assert rel_err(got, ref, w.u0) <= tol
            first = got if first is None else first
            np.testing.assert_array_equal(got, first)
    # ---- Gauss-Seidel
    for w in (W.c3_periodic_btcs(B=3, N=2048, dtype=dtype), W.c3_periodic_btcs(B=3, N=201, dtype=dtype),
              W.c3_periodic_btcs(B=40, N=24, dtype=dtype)):
        dt = _dt(w, 0.4)
        need = B.workspace_bytes(B.OP_GS, is64, w.B, w.N, w.bc)
        gtol = 1e-4 if dtype == np.float32 else 1e-9
        direct = oracle.btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 3, w.bc)
        first = None
        for _ in range(3):
            gu, u = guarded_from(w.u0); gw, ws = guarded_empty(need); gi, iraw = guarded_empty(8 * w.B)
            B.burgers_btcs_gs(u, w.L, torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda(), 3, w.bc, tol=gtol,
                              max_iter=200, iters_out=iraw.view(torch.int64), ws=ws if need else None)
            torch.cuda.synchronize()
            assert gu.intact() and gw.intact() and gi.intact()
            got = u.cpu().numpy()
            assert rel_err(got, direct, w.u0) <= 30 * gtol
            first = got if first is None else first
            np.testing.assert_array_equal(got, first)
    # ---- adjoint of RK4: resident backward kernel (eight single-barrier exchanges per step), checkpointed, streaming
    for w, seg in ((W.c5_rk4_ensemble(B=3, N=1024, dtype=dtype), 0), (W.c2_dirichlet_batch(B=3, N=1000, dtype=dtype), 4),
                   (W.c4a_long_explicit(N=40000, dtype=dtype), 0)):
        dt = _dt(w, 0.8)
        lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
        need = int(B.raw().burgers_adjoint_scheme_workspace_bytes(int(is64), w.B, w.N, w.bc, 1, 10, seg))
        ref = oracle.explicit_adjoint(_f64(w.u0), _f64(lam_T), w.L, _f64(w.nu), _f64(dt), 10, w.bc, scheme=oracle.RK4)
        first = None
        for _ in range(3):
            gu, u = guarded_from(w.u0); gl, lam = guarded_from(lam_T); gw, ws = guarded_empty(need)
            B.burgers_explicit_adjoint(u, lam, w.L, torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda(), 10, w.bc,
                                       ws=ws, segment=seg, scheme=B.SCHEME_RK4)
            torch.cuda.synchronize()
            assert gu.intact() and gl.intact() and gw.intact()
            np.testing.assert_array_equal(u.cpu().numpy(), w.u0)
            got = lam.cpu().numpy()
            assert np.abs(got - ref).max() / np.abs(ref).max() <= tol
            first = got if first is None else first
            np.testing.assert_array_equal(got, first)
    # ---- adjoint of BTCS: resident transposed solve (exact and ragged partitions), thread-per-system fallback
    for w in (W.c3_periodic_btcs(B=3, N=2048, dtype=dtype), W.c2_dirichlet_batch(B=3, N=201, dtype=dtype),
              W.c4b_long_btcs(N=20000, dtype=dtype)):
        dt = _dt(w, 10.0)
        lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
        need = int(B.raw().burgers_btcs_adjoint_workspace_bytes(int(is64), w.B, w.N, w.bc, 5))
        ref = oracle.btcs_adjoint(_f64(w.u0), _f64(lam_T), w.L, _f64(w.nu), _f64(dt), 5, w.bc)
        first = None
        for _ in range(3):
            gu, u = guarded_from(w.u0); gl, lam = guarded_from(lam_T); gw, ws = guarded_empty(need)
            B.burgers_btcs_adjoint(u, lam, w.L, torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda(), 5, w.bc, ws=ws)
            torch.cuda.synchronize()
            assert gu.intact() and gl.intact() and gw.intact()
            np.testing.assert_array_equal(u.cpu().numpy(), w.u0)
            got = lam.cpu().numpy()
            assert np.abs(got - ref).max() / np.abs(ref).max() <= tol
            first = got if first is None else first
            np.testing.assert_array_equal(got, first)
    # ---- adjoint of forward Euler
    for w, seg in ((W.c2_dirichlet_batch(B=3, N=4096, dtype=dtype), 0), (W.c3_periodic_btcs(B=3, N=1024, dtype=dtype), 5),
                   (W.c4a_long_explicit(N=40000, dtype=dtype), 0)):
        dt = _dt(w, 0.4)
        lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
        need = int(B.raw().burgers_adjoint_ckpt_workspace_bytes(int(is64), w.B, w.N, w.bc, 12, seg))
        ref = oracle.explicit_adjoint(_f64(w.u0), _f64(lam_T), w.L, _f64(w.nu), _f64(dt), 12, w.bc)
        first = None
        for _ in range(3):
            gu, u = guarded_from(w.u0); gl, lam = guarded_from(lam_T); gw, ws = guarded_empty(need)
            B.burgers_explicit_adjoint(u, lam, w.L, torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda(), 12, w.bc,
                                       ws=ws, segment=seg)
            torch.cuda.synchronize()
            assert gu.intact() and gl.intact() and gw.intact()
            np.testing.assert_array_equal(u.cpu().numpy(), w.u0)
            got = lam.cpu().numpy()
            assert np.abs(got - ref).max() / np.abs(ref).max() <= tol
            first = got if first is None else first
            np.testing.assert_array_equal(got, first)
    # ---- reverse mode of the Newton scheme (resident exact / ragged, thread-per-system), checkpoint segments of both
    #      implicit adjoints, and the trajectory kernels of the implicit schemes (snapshots staged per warp)
    wn = W.c3_periodic_btcs(B=3, N=2048, dtype=dtype)
    wd = W.c2_dirichlet_batch(B=3, N=201, dtype=dtype); wd.nu[:] = 0.05
    wl = W.c4b_long_btcs(N=20000, dtype=dtype); wl.nu[:] = 1e-3
    ntol = 2e-6 if dtype == np.float32 else 1e-13
    for w, seg in ((wn, 0), (wd, 2), (wl, 3)):
        dt = _dt(w, 4.0)
        lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
        for op, fn, ofn, kw in ((B.OP_NEWTON, B.burgers_newton_adjoint, oracle.newton_adjoint, dict(tol=ntol)),
                                (B.OP_BTCS, B.burgers_btcs_adjoint, oracle.btcs_adjoint, {})):
            need = int(B.raw().burgers_implicit_adjoint_ckpt_workspace_bytes(op, int(is64), w.B, w.N, w.bc, 5, seg))
            ref = ofn(_f64(w.u0), _f64(lam_T), w.L, _f64(w.nu), _f64(dt), 5, w.bc)
            first = None
            for _ in range(3):
                gu, u = guarded_from(w.u0); gl, lam = guarded_from(lam_T); gw, ws = guarded_empty(need)
                fn(u, lam, w.L, torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda(), 5, w.bc, ws=ws, segment=seg, **kw)
                torch.cuda.synchronize()
                assert gu.intact() and gl.intact() and gw.intact(), (w.name, op, seg)
                np.testing.assert_array_equal(u.cpu().numpy(), w.u0)
                got = lam.cpu().numpy()
                assert np.abs(got - ref).max() / np.abs(ref).max() <= tol, (w.name, op, seg)
                first = got if first is None else first
                np.testing.assert_array_equal(got, first)
    w96 = W.c3_periodic_btcs(B=2, N=96, dtype=dtype); w96.nu[:] = 0.2       # (cell Peclet number < 2 for the Newton scheme)
    for w in (wn, wd, w96):
        dt = _dt(w, 4.0)
        for which in ("btcs", "newton"):
            first = None
            for _ in range(3):
                gu, u = guarded_from(w.u0); gs, sraw = guarded_empty(3 * w.u0.size * w.u0.itemsize)
                snaps = sraw.view(u.dtype).view(3, w.B, w.N)
                dnu, ddt = torch.from_numpy(w.nu).cuda(), torch.from_numpy(dt).cuda()
                if which == "btcs":
                    B.burgers_btcs_traj(u, w.L, dnu, ddt, 7, w.bc, 2, snaps=snaps)
                    ref = oracle.btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 6, w.bc)
                else:
                    B.burgers_newton_traj(u, w.L, dnu, ddt, 7, w.bc, 2, snaps=snaps, tol=ntol)
                    ref = oracle.newton_btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 6, w.bc, tol=1e-13)
                torch.cuda.synchronize()
                assert gu.intact() and gs.intact(), (w.name, which)
                got = snaps.cpu().numpy()
                assert rel_err(got[2], ref, w.u0) <= tol, (w.name, which)      # third snapshot = state after 6 steps
                first = got if first is None else first
                np.testing.assert_array_equal(got, first)
