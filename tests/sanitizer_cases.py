"""Small invocations of every kernel family of libburgers.so, for compute-sanitizer:

    compute-sanitizer --tool racecheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool memcheck   python tests/sanitizer_cases.py
    compute-sanitizer --tool initcheck  python tests/sanitizer_cases.py

Each case is sized so that the code path the tool has to see is really taken (several warps per CTA for the
double-buffered edge exchange, two tiles per CTA for the re-used stage / PCR buffers of the LONG kernel, a time
step large enough that PCR runs to its full depth and the 2x2 ending, ...) and small enough to finish under
the tools' 10-100x slow-down.  Results are also compared with the oracle so that a case cannot pass by doing
nothing.  `python tests/sanitizer_cases.py [case ...]` runs the named cases only; summaries of the runs are kept
in profiles/r02_sanitizer.md."""
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

import oracle                                             # noqa: E402
from parity import rel_err, to_dev                        # noqa: E402
from paper_2601_12204_b200 import binding as B            # noqa: E402
from paper_2601_12204_b200 import workloads as W          # noqa: E402


FAILED = []


def _ok(what, err, tol):
    """Report instead of raising, so that one run of a tool covers every case."""
    good = bool(err <= tol)
    print(f"    {what}: err {err:.3g} (tol {tol:g}) {'ok' if good else 'FAILED'}", flush=True)
    if not good:
        FAILED.append(what)


def _dt(w, C):
    return oracle.dt_from_cfl(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), C, w.bc).astype(w.dtype)


def _f64(a):
    return a.astype(np.float64)


def _explicit(w, n, scheme, tol, **kw):
    dt = _dt(w, 0.4 if scheme == 0 else 0.8)
    u = to_dev(w.u0.copy())
    B.burgers_explicit(u, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, scheme, **kw)
    ref = oracle.explicit(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), n, w.bc, scheme)
    _ok(f"explicit {w.name} scheme {scheme} {kw}", rel_err(u.cpu().numpy(), ref, w.u0), tol)


def case_cfl():
    rng = np.random.default_rng(1)
    for shape in ((600, 512), (3, 4099), (2, 70001)):     # warp per row, CTA per row, split + atomicMax + finalize
        for dtype in (np.float32, np.float64):
            u0 = rng.standard_normal(shape).astype(dtype); nu = rng.uniform(0.01, 0.1, shape[0]).astype(dtype)
            got = B.dt_from_cfl(to_dev(u0), 1.0, to_dev(nu), 0.4, 0).cpu().numpy()
            ref = oracle.dt_from_cfl(_f64(u0), 1.0, _f64(nu), 0.4, 0).astype(dtype)
            assert np.all(np.abs(got - ref) <= 2 * np.spacing(np.abs(ref)))


def case_resident():
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        _explicit(W.c2_dirichlet_batch(B=3, N=4096, dtype=dtype), 130, 0, tol)     # 4 warps, shared edge exchange, renormalisation
        _explicit(W.c2_dirichlet_batch(B=3, N=4096, dtype=dtype), 20, 1, tol)      # RK4, 4 exchanges per step
        _explicit(W.c5_rk4_ensemble(B=4, N=1024, dtype=dtype), 20, 1, tol)         # one warp per trajectory (shuffles)
        _explicit(W.c3_periodic_btcs(B=2, N=200, dtype=dtype), 20, 0, tol)         # ragged: scalar loads, inactive threads


def case_tiled():
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        w = W.c4a_long_explicit(N=40000, dtype=dtype)                              # 5+ tiles, ragged last tile
        _explicit(w, 70, 0, tol, plan=B.PLAN_TILED, tblock=32)                     # 3 launches, ping-pong, copy back
        _explicit(w, 9, 1, tol, plan=B.PLAN_TILED, tblock=4)
        _explicit(W.c2_dirichlet_batch(B=2, N=20000, dtype=dtype), 40, 0, tol, plan=B.PLAN_TILED, tblock=16)


def case_snap():
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        for w, scheme in ((W.c2_dirichlet_batch(B=3, N=4096, dtype=dtype), 0), (W.c5_rk4_ensemble(B=3, N=1024, dtype=dtype), 1)):
            dt = _dt(w, w.cfl)
            u = to_dev(w.u0.copy())
            _, snaps = B.burgers_explicit_traj(u, w.L, to_dev(w.nu), to_dev(dt), 24, w.bc, scheme, 4)   # staged stores
            _, ref = oracle.explicit_trajectory(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 24, w.bc, scheme, 4)
            _ok(f"snap {w.name}", np.abs(snaps.cpu().numpy() - ref).max() / np.abs(w.u0).max(), tol)


def case_adapt():
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        for w, scheme in ((W.c2_dirichlet_batch(B=3, N=4096, dtype=dtype), 0), (W.c5_rk4_ensemble(B=3, N=1024, dtype=dtype), 1)):
            u = to_dev(w.u0.copy())
            _, t, _ = B.burgers_explicit_adaptive(u, w.L, to_dev(w.nu), w.cfl, 5, 6, w.bc, scheme)       # CTA-wide max, 5 evaluations
            ref, t_ref = oracle.explicit_adaptive(_f64(w.u0), w.L, _f64(w.nu), w.cfl, 5, 6, w.bc, scheme, dtype=dtype)
            _ok(f"adapt {w.name}", rel_err(u.cpu().numpy(), ref, w.u0), tol)
            assert np.allclose(t.cpu().numpy(), t_ref, rtol=1e-6)


def _btcs(w, n, C, tol, **kw):
    dt = _dt(w, C)
    u = to_dev(w.u0.copy())
    B.burgers_btcs(u, w.L, to_dev(w.nu), to_dev(dt), n, w.bc, **kw)
    ref = oracle.btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), n, w.bc)
    _ok(f"btcs {w.name} C={C} {kw}", rel_err(u.cpu().numpy(), ref, w.u0), tol)


def case_thomas():
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        _btcs(W.c3_periodic_btcs(B=70, N=201, dtype=dtype), 3, 4.0, tol, plan=B.PLAN_THOMAS)   # transposes in and out, Sherman-Morrison
        _btcs(W.c2_dirichlet_batch(B=33, N=130, dtype=dtype), 3, 4.0, tol, plan=B.PLAN_THOMAS)


def case_hybrid():
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        w = W.c3_periodic_btcs(B=3, N=2048, dtype=dtype)
        assert B.plan_query(B.OP_BTCS, dtype == np.float64, w.B, w.N, w.bc) == B.PLAN_HYBRID
        _btcs(w, 4, 10.0, tol)                                 # PCR exits early (block-wide vote)
        _btcs(w, 3, 1.0e5, tol)                                # weak dominance of the reduced rows: full depth, 2x2 ending
        _btcs(W.c2_dirichlet_batch(B=3, N=1024, dtype=dtype), 4, 10.0, tol)    # Dirichlet identity rows
        _btcs(W.c3_periodic_btcs(B=3, N=201, dtype=dtype), 4, 10.0, tol)       # the paper's N: ragged partitions (6 / 7 rows)
        _btcs(W.c2_dirichlet_batch(B=3, N=3001, dtype=dtype), 3, 1.0e5, tol)   # ragged, 256 threads, full depth


def case_long():
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        w = W.c4b_long_btcs(N=1 << 19, dtype=dtype)            # 3 systems x 296 tiles > 592 resident CTAs: two tiles per CTA,
        u0 = np.repeat(w.u0, 3, axis=0) * np.array([[1.0], [0.5], [-0.7]], dtype=dtype)   # stage and PCR buffers re-used
        w3 = W.Workload("long3", u0, np.repeat(w.nu, 3), w.L, w.bc, w.scheme, w.cfl, 0, w.dtype)
        assert B.plan_query(B.OP_BTCS, dtype == np.float64, 3, w.N, w.bc) == B.PLAN_LONG
        _btcs(w3, 3, 10.0, tol)
        wd = W.Workload("long-dirichlet", w.u0[:, :1 << 15].copy(), w.nu, 1.0, 1, w.scheme, w.cfl, 0, w.dtype)
        _btcs(wd, 3, 10.0, tol, plan=B.PLAN_LONG)              # Dirichlet edge tiles (zero-filled cp.async)
        ws = W.c4b_long_btcs(N=1 << 15, dtype=dtype)
        _btcs(ws, 3, 3000.0, tol, plan=B.PLAN_LONG)            # halo check fails at step 0: cooperative GENERAL fallback, full depth
        _btcs(ws, 2, 10.0, tol, plan=B.PLAN_LONG_GENERAL)      # GENERAL alone, early exit by the level flags
        wr = W.c4b_long_btcs(N=40003, dtype=dtype)             # odd N: element-wise wrap at the seam, ragged last tile,
        _btcs(wr, 3, 10.0, tol)                                # ragged partitions in the fallback
        _btcs(wr, 2, 3000.0 if dtype == np.float64 else 300.0, tol)   # (fp32: cond ~ 1 + 4r times eps stays under the bar)


def case_newton():
    for dtype, tol, ntol in ((np.float32, 1e-4, 1e-5), (np.float64, 1e-10, 1e-12)):
        w201 = W.c3_periodic_btcs(B=40, N=201, dtype=dtype)       # ragged partitions; nu raised so that the cell Peclet
        w201.nu[:] = 0.1                                          # number |u| dx / nu stays below 2 (D11: no pivoting)
        for w in (W.c3_periodic_btcs(B=3, N=2048, dtype=dtype), W.c2_dirichlet_batch(B=3, N=1024, dtype=dtype), w201):
            for theta in (1.0, 0.5):
                dt = _dt(w, 2.0)
                u = to_dev(w.u0.copy())
                B.burgers_newton(u, w.L, to_dev(w.nu), to_dev(dt), 3, w.bc, tol=ntol, max_iter=20, theta=theta)
                ref = oracle.newton_btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 3, w.bc, tol=1e-12, max_iter=20, theta=theta)
                _ok(f"newton {w.name} theta={theta}", rel_err(u.cpu().numpy(), ref, w.u0), tol)


def case_gs():
    import torch
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        for w in (W.c3_periodic_btcs(B=3, N=2048, dtype=dtype), W.c3_periodic_btcs(B=3, N=201, dtype=dtype),
                  W.c2_dirichlet_batch(B=3, N=512, dtype=dtype), W.c3_periodic_btcs(B=40, N=24, dtype=dtype)):
            dt = _dt(w, 0.4)
            u = to_dev(w.u0.copy())
            it = torch.zeros(w.B, dtype=torch.int64, device="cuda")
            gtol = 1e-4 if dtype == np.float32 else 1e-9
            B.burgers_btcs_gs(u, w.L, to_dev(w.nu), to_dev(dt), 3, w.bc, tol=gtol, max_iter=200, iters_out=it)
            direct = oracle.btcs(_f64(w.u0), w.L, _f64(w.nu), _f64(dt), 3, w.bc)
            _ok(f"gs {w.name}", rel_err(u.cpu().numpy(), direct, w.u0), 30 * gtol)
            assert it.min().item() >= 3


def case_adjoint():
    rng = np.random.default_rng(3)
    for dtype, tol in ((np.float32, 1e-4), (np.float64, 1e-10)):
        for w, seg in ((W.c2_dirichlet_batch(B=3, N=4096, dtype=dtype), 0), (W.c3_periodic_btcs(B=3, N=1024, dtype=dtype), 5),
                       (W.c4a_long_explicit(N=40000, dtype=dtype), 0)):      # resident, checkpointed, streaming backward
            dt = _dt(w, 0.4)
            lam_T = rng.standard_normal(w.u0.shape).astype(dtype)
            lam = to_dev(lam_T.copy())
            B.burgers_explicit_adjoint(to_dev(w.u0), lam, w.L, to_dev(w.nu), to_dev(dt), 12, w.bc, segment=seg)
            ref = oracle.explicit_adjoint(_f64(w.u0), _f64(lam_T), w.L, _f64(w.nu), _f64(dt), 12, w.bc)
            _ok(f"adjoint {w.name}", np.abs(lam.cpu().numpy() - ref).max() / np.abs(ref).max(), tol)


CASES = {k[5:]: v for k, v in sorted(globals().items()) if k.startswith("case_")}


def main(argv):
    import torch
    assert torch.cuda.is_available(), "needs a CUDA device"
    names = argv or list(CASES)
    for n in names:
        print(f"case {n}:", flush=True)
        CASES[n]()
        torch.cuda.synchronize()
    if FAILED:
        raise SystemExit(f"FAILED: {FAILED}")
    print(f"{len(names)} cases ok")


if __name__ == "__main__":
    main(sys.argv[1:])
