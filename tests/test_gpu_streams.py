"""SURVEY.md 8(b) "Asynchrony" / "Thread-safety": every device entry point only enqueues on the stream it is
given, and concurrent calls on different streams with disjoint buffers are legal.  The binding passes torch's
CURRENT stream, so `with torch.cuda.stream(s)` drives the `void* stream` argument of the C ABI."""
import threading

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


def _inputs(w, C):
    dt = oracle.dt_from_cfl(w.u0.astype(np.float64), w.L, w.nu.astype(np.float64), C, w.bc).astype(w.dtype)
    return to_dev(w.u0.copy()), to_dev(w.nu), to_dev(dt), dt


def test_non_default_stream_every_plan(B):
    """One call of each plan family on a non-default (non-blocking) stream; the default stream stays idle, and
    nothing is read back before the stream is synchronised."""
    import torch
    s = torch.cuda.Stream()
    cases = []
    with torch.cuda.stream(s):
        w = W.c2_dirichlet_batch(B=6, N=4096, dtype=np.float64)               # RESIDENT, CTA of 128 threads
        u, nu, dt, dth = _inputs(w, w.cfl)
        B.burgers_explicit(u, w.L, nu, dt, 300, w.bc, B.SCHEME_EULER)
        cases.append(("resident", u, lambda: oracle.explicit(w.u0, w.L, w.nu, dth, 300, w.bc, 0), w.u0))
        w2 = W.c4a_long_explicit(N=1 << 17, n_steps=0, dtype=np.float64)      # TILED, several launches + copy back
        u2, nu2, dt2, dth2 = _inputs(w2, w2.cfl)
        assert B.plan_query(B.OP_EXPLICIT, True, 1, w2.N, w2.bc, 0) == B.PLAN_TILED
        B.burgers_explicit(u2, w2.L, nu2, dt2, 300, w2.bc, B.SCHEME_EULER)
        cases.append(("tiled", u2, lambda: oracle.explicit(w2.u0, w2.L, w2.nu, dth2, 300, w2.bc, 0), w2.u0))
        w3 = W.c3_periodic_btcs(B=5, N=2048, n_steps=0)                       # HYBRID
        u3, nu3, dt3, dth3 = _inputs(w3, w3.cfl)
        B.burgers_btcs(u3, w3.L, nu3, dt3, 12, w3.bc)
        cases.append(("hybrid", u3, lambda: oracle.btcs(w3.u0, w3.L, w3.nu, dth3, 12, w3.bc), w3.u0))
        w4 = W.c4b_long_btcs(N=1 << 15, n_steps=0)                            # LONG: programmatic dependent launches,
        u4, nu4, dt4, dth4 = _inputs(w4, w4.cfl)                              # fix-up, cooperative kernel
        assert B.plan_query(B.OP_BTCS, True, 1, w4.N, w4.bc) == B.PLAN_LONG
        B.burgers_btcs(u4, w4.L, nu4, dt4, 7, w4.bc)
        cases.append(("long", u4, lambda: oracle.btcs(w4.u0, w4.L, w4.nu, dth4, 7, w4.bc), w4.u0))
        dtc = B.dt_from_cfl(u3, w3.L, nu3, 0.4, w3.bc)                        # CFL kernel on the same stream, after the solve
    s.synchronize()
    for name, u, ref, u0 in cases:
        assert rel_err(u.cpu().numpy(), ref(), u0) <= 1e-10, name
    ref_dt = oracle.dt_from_cfl(cases[2][1].cpu().numpy(), w3.L, w3.nu, 0.4, w3.bc)
    assert np.all(np.abs(dtc.cpu().numpy() - ref_dt) <= 2 * np.spacing(ref_dt))


def test_two_streams_two_host_threads_disjoint_buffers(B):
    """Two host threads, each with its own stream and its own buffers, call the library at the same time (long
    enough kernels that they overlap on the device); both results equal the oracle's."""
    import torch
    wa = W.c2_dirichlet_batch(B=64, N=4096, dtype=np.float64)
    wb = W.c3_periodic_btcs(B=64, N=2048, n_steps=0)
    ua, nua, dta, dtha = _inputs(wa, wa.cfl)
    ub, nub, dtb, dthb = _inputs(wb, wb.cfl)
    torch.cuda.synchronize()
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    errs = []

    def run(stream, fn):
        try:
            with torch.cuda.stream(stream):
                for _ in range(3):            # several calls back to back on each stream
                    fn()
        except Exception as ex:           # noqa: BLE001 -- reported below
            errs.append(ex)

    ta = threading.Thread(target=run, args=(sa, lambda: B.burgers_explicit(ua, wa.L, nua, dta, 1000, wa.bc, 0)))
    tb = threading.Thread(target=run, args=(sb, lambda: B.burgers_btcs(ub, wb.L, nub, dtb, 40, wb.bc)))
    ta.start(); tb.start(); ta.join(); tb.join()
    sa.synchronize(); sb.synchronize()
    assert not errs, errs
    refa = oracle.explicit(wa.u0, wa.L, wa.nu, dtha, 3000, wa.bc, 0)
    refb = oracle.btcs(wb.u0, wb.L, wb.nu, dthb, 120, wb.bc)
    assert rel_err(ua.cpu().numpy(), refa, wa.u0) <= 1e-10
    assert rel_err(ub.cpu().numpy(), refb, wb.u0) <= 1e-10
