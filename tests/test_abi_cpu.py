"""C-ABI checks that need no GPU: the library builds, loads, exports every symbol that
include/burgers.h declares, rejects bad arguments synchronously (before any CUDA call), and
its pure shape queries behave."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "burgers.h")


@pytest.fixture(scope="module")
def B():
    from paper_2601_12204_b200 import build
    build.build()
    from paper_2601_12204_b200 import binding
    return binding


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b((?:burgers|dt_from_cfl)_\w+)\s*\(", src)))


def test_header_symbols_exported(B):
    names = _declared()
    assert len(names) >= 39
    lib = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in burgers.h but not exported"
    assert sorted(B.EXPORTS) == names


def test_version_and_strerror(B):
    assert B.version() == 100
    assert B.strerror(0) == "ok"
    for st in range(-7, 0):
        assert B.strerror(st) not in ("ok", "unknown status")
    assert B.strerror(-99) == "unknown status"


def test_argument_errors_are_synchronous(B):
    lib = B.raw()
    one = ctypes.c_void_p(16)  # never dereferenced: every call below fails validation first
    f = lib.burgers_explicit_f64
    assert f(None, 1, 8, 1.0, one, one, 1, 0, 0, None, 0, None) == B.ERR_NULL
    assert f(one, 1, 8, 1.0, None, one, 1, 0, 0, None, 0, None) == B.ERR_NULL
    assert f(one, 0, 8, 1.0, one, one, 1, 0, 0, None, 0, None) == B.ERR_SHAPE
    assert f(one, 1, 2, 1.0, one, one, 1, 0, 0, None, 0, None) == B.ERR_SHAPE
    assert f(one, 1, 8, 1.0, one, one, -1, 0, 0, None, 0, None) == B.ERR_SHAPE
    assert f(one, 1, 8, 1.0, one, one, 1, 2, 0, None, 0, None) == B.ERR_ENUM
    assert f(one, 1, 8, 1.0, one, one, 1, 0, 5, None, 0, None) == B.ERR_ENUM
    assert f(one, 1, 8, 0.0, one, one, 1, 0, 0, None, 0, None) == B.ERR_VALUE
    assert f(one, 1, 8, float("nan"), one, one, 1, 0, 0, None, 0, None) == B.ERR_VALUE
    assert f(one, 1, 8, float("inf"), one, one, 1, 0, 0, None, 0, None) == B.ERR_VALUE
    g = lib.burgers_explicit_plan_f32
    assert g(one, 1, 8, 1.0, one, one, 1, 0, 0, 9, 0, 0, None, 0, None) == B.ERR_ENUM
    assert g(one, 1, 8, 1.0, one, one, 1, 0, 0, B.PLAN_RESIDENT, 0, 3, None, 0, None) == B.ERR_PLAN
    assert g(one, 1, 7, 1.0, one, one, 1, 0, 0, B.PLAN_RESIDENT, 0, 2, None, 0, None) == B.ERR_PLAN
    # TILED needs a workspace
    assert g(one, 1, 1 << 20, 1.0, one, one, 1, 0, 0, B.PLAN_TILED, 0, 0, None, 0, None) == B.ERR_WORKSPACE
    tj = lib.burgers_explicit_traj_f64
    assert tj(one, 1, 8, 1.0, one, one, 4, 0, 0, 2, None, None, 0, None) == B.ERR_NULL
    assert tj(one, 1, 8, 1.0, one, one, 4, 0, 0, 0, one, None, 0, None) == B.ERR_SHAPE
    assert tj(one, 1, 8, 1.0, one, one, 4, 0, 7, 2, one, None, 0, None) == B.ERR_ENUM
    aj = lib.burgers_explicit_adjoint_f64
    assert aj(one, None, 1, 8, 1.0, one, one, 3, 0, None, 0, None) == B.ERR_NULL
    assert aj(one, one, 1, 8, 1.0, one, one, 3, 0, None, 0, None) == B.ERR_WORKSPACE
    assert aj(one, one, 1, 8, 1.0, one, one, -3, 0, None, 0, None) == B.ERR_SHAPE
    assert lib.burgers_explicit_adjoint_ckpt_f32(one, one, 1, 8, 1.0, one, one, 3, 0, -1, one, 1 << 20, None) == B.ERR_SHAPE
    full = B.raw().burgers_adjoint_ckpt_workspace_bytes(1, 4, 100, 0, 100, 0)
    ck = B.raw().burgers_adjoint_ckpt_workspace_bytes(1, 4, 100, 0, 100, 10)
    assert full >= (2 + 99) * 4 * 100 * 8 and (2 + 9 + 9) * 4 * 100 * 8 <= ck < full // 3
    lib.burgers_adjoint_workspace_bytes.restype = ctypes.c_size_t
    assert lib.burgers_adjoint_workspace_bytes(1, 4, 100, 0, 11) >= (2 + 10) * 4 * 100 * 8
    ad = lib.burgers_explicit_adaptive_f64
    assert ad(one, 1, 8, 1.0, one, 0.4, 3, 5, 0, 0, None, None, None, 0, None) == B.ERR_NULL
    assert ad(one, 1, 8, 1.0, one, 0.4, 3, 0, 0, 0, one, None, None, 0, None) == B.ERR_SHAPE
    assert ad(one, 1, 8, 1.0, one, -0.4, 3, 5, 0, 0, one, None, None, 0, None) == B.ERR_VALUE
    assert ad(one, 1, 8, 1.0, one, 0.4, 3, 5, 0, 9, one, None, None, 0, None) == B.ERR_ENUM
    sh = lib.burgers_solve_host_f64
    assert sh(one, 1, 8, 1.0, None, 0.4, 1, 0, B.OP_EXPLICIT, 0, None) == B.ERR_NULL
    assert sh(one, 1, 8, 1.0, one, 0.4, 1, 0, B.OP_NEWTON, 0, None) == B.ERR_ENUM
    assert sh(one, 1, 8, 1.0, one, 0.4, 1, 0, B.OP_EXPLICIT, 5, None) == B.ERR_ENUM
    assert sh(one, 1, 8, 1.0, one, -0.4, 1, 0, B.OP_BTCS, 0, None) == B.ERR_VALUE
    assert sh(one, 1, 2, 1.0, one, 0.4, 1, 0, B.OP_BTCS, 0, None) == B.ERR_SHAPE
    gs = lib.burgers_btcs_gs_f64
    assert gs(one, 1, 8, 1.0, one, None, 1, 0, 1e-6, 10, None, one, 1 << 20, None) == B.ERR_NULL
    assert gs(one, 1, 8, 1.0, one, one, 1, 0, -1e-6, 10, None, one, 1 << 20, None) == B.ERR_VALUE
    assert gs(one, 1, 8, 1.0, one, one, 1, 0, 1e-6, 10, None, None, 0, None) == B.ERR_WORKSPACE
    assert B.workspace_bytes(B.OP_GS, True, 4, 100, 0) == 0                       # CTA per system: no scratch
    assert B.workspace_bytes(B.OP_GS, True, 4, 40, 0) >= 2 * 4 * 40 * 8           # thread per system
    assert B.workspace_bytes(B.OP_GS, True, 4, 5000, 0) >= 2 * 4 * 5000 * 8
    bt = lib.burgers_btcs_traj_f64
    assert bt(one, 1, 8, 1.0, one, one, 4, 0, 2, None, None, 0, None) == B.ERR_NULL
    assert bt(one, 1, 8, 1.0, one, one, 4, 0, 0, one, None, 0, None) == B.ERR_SHAPE
    h = lib.burgers_btcs_f64
    assert h(None, 1, 8, 1.0, one, one, 1, 0, None, 0, None) == B.ERR_NULL
    assert h(one, 1, 8, 1.0, one, one, 1, 7, None, 0, None) == B.ERR_ENUM
    assert h(one, 1, 8, -1.0, one, one, 1, 0, None, 0, None) == B.ERR_VALUE
    hp = lib.burgers_btcs_plan_f64
    assert hp(one, 1, 8, 1.0, one, one, 1, 0, B.PLAN_THOMAS, None, 0, None) == B.ERR_WORKSPACE
    assert hp(one, 1, 8, 1.0, one, one, 1, 0, B.PLAN_RESIDENT, None, 0, None) == B.ERR_ENUM
    assert hp(one, 1, 1000, 1.0, one, one, 1, 0, B.PLAN_LONG, None, 0, None) == B.ERR_PLAN
    assert hp(one, 1, 1 << 16, 1.0, one, one, 1, 0, B.PLAN_LONG, None, 0, None) == B.ERR_WORKSPACE
    assert hp(one, 1, 1 << 16, 1.0, one, one, 1, 0, B.PLAN_LONG_GENERAL, None, 0, None) == B.ERR_WORKSPACE
    c = lib.dt_from_cfl_f32
    assert c(None, 1, 8, 1.0, one, 0.4, 0, one, None) == B.ERR_NULL
    assert c(one, 1, 8, 1.0, one, 0.0, 0, one, None) == B.ERR_VALUE
    assert c(one, 1, 8, 1.0, one, 0.4, 3, one, None) == B.ERR_ENUM
    assert c(one, 1, 1, 1.0, one, 0.4, 0, one, None) == B.ERR_SHAPE
    nw = lib.burgers_newton_f64
    assert nw(None, 1, 8, 1.0, one, one, 1, 0, 1.0, 1e-6, 10, None, 0, None, 0, None) == B.ERR_NULL
    assert nw(one, 1, 8, 1.0, one, one, 1, 0, 1.0, -1.0, 10, None, 0, None, 0, None) == B.ERR_VALUE
    assert nw(one, 1, 8, 1.0, one, one, 1, 0, 1.0, float("nan"), 10, None, 0, None, 0, None) == B.ERR_VALUE
    assert nw(one, 1, 8, 1.0, one, one, 1, 0, 1.0, 1e-6, -1, None, 0, None, 0, None) == B.ERR_VALUE
    assert nw(one, 1, 8, 1.0, one, one, 1, 0, 1.5, 1e-6, 10, None, 0, None, 0, None) == B.ERR_VALUE
    assert nw(one, 1, 8, 1.0, one, one, 1, 0, float("nan"), 1e-6, 10, None, 0, None, 0, None) == B.ERR_VALUE
    assert nw(one, 1, 8, 1.0, one, one, 1, 0, 0.5, 1e-6, 10, None, B.PLAN_LONG, None, 0, None) == B.ERR_ENUM
    assert nw(one, 1, 5, 1.0, one, one, 1, 0, 0.5, 1e-6, 10, None, B.PLAN_HYBRID, None, 0, None) == B.ERR_PLAN
    assert nw(one, 1, 100000, 1.0, one, one, 1, 0, 0.5, 1e-6, 10, None, B.PLAN_HYBRID, None, 0, None) == B.ERR_PLAN
    assert nw(one, 1, 100000, 1.0, one, one, 1, 0, 0.5, 1e-6, 10, None, B.PLAN_AUTO, None, 0, None) == B.ERR_WORKSPACE
    assert lib.burgers_newton_host_f32(one, 1, 8, 1.0, one, one, 1, 0, 1.0, -2.0, 10, None) == B.ERR_VALUE
    assert lib.burgers_newton_host_f64(one, 1, 8, 1.0, one, one, 1, 0, -0.1, 1e-6, 10, None) == B.ERR_VALUE
    # host variants validate the same way
    assert lib.burgers_explicit_host_f32(None, 1, 8, 1.0, one, one, 1, 0, 0) == B.ERR_NULL
    assert lib.burgers_btcs_host_f64(one, 1, 8, 1.0, one, one, -2, 0) == B.ERR_SHAPE
    assert lib.dt_from_cfl_host_f64(one, 1, 8, 1.0, one, -1.0, 0, one) == B.ERR_VALUE


def test_plan_queries(B):
    # configs of BASELINE.json: C2 and C5 are resident, C4a is tiled
    assert B.plan_query(B.OP_EXPLICIT, False, 1024, 4096, B.BC_DIRICHLET, B.SCHEME_EULER) == B.PLAN_RESIDENT
    assert B.plan_query(B.OP_EXPLICIT, True, 1024, 4096, B.BC_DIRICHLET, B.SCHEME_EULER) == B.PLAN_RESIDENT
    assert B.plan_query(B.OP_EXPLICIT, False, 65536, 1024, B.BC_PERIODIC, B.SCHEME_RK4) == B.PLAN_RESIDENT
    assert B.plan_query(B.OP_EXPLICIT, False, 1, 1 << 24, B.BC_PERIODIC, B.SCHEME_EULER) == B.PLAN_TILED
    assert B.plan_query(B.OP_EXPLICIT, True, 1, 3001, B.BC_PERIODIC, B.SCHEME_EULER) == B.PLAN_TILED
    assert B.workspace_bytes(B.OP_EXPLICIT, False, 1024, 4096, B.BC_DIRICHLET, 0) == 0
    assert 4 << 24 <= B.workspace_bytes(B.OP_EXPLICIT, False, 1, 1 << 24, B.BC_PERIODIC, 0) <= (4 << 24) + 512   # + adaptive slots
    assert B.workspace_bytes(B.OP_BTCS, True, 8, 100, B.BC_PERIODIC, 0, B.PLAN_THOMAS) >= 4 * 8 * 100 * 8
    assert B.workspace_bytes(B.OP_BTCS, True, 8, 100, B.BC_DIRICHLET, 0, B.PLAN_THOMAS) >= 3 * 8 * 100 * 8
    assert B.launch_count(B.OP_EXPLICIT, False, 1024, 4096, 1, 0, n_steps=10000) == 1
    assert B.launch_count(B.OP_EXPLICIT, False, 1, 1 << 24, 0, 0, n_steps=2000, tblock=16) == 125
    assert B.launch_count(B.OP_EXPLICIT, False, 1, 1 << 24, 0, 0, n_steps=0) == 0
    # BTCS: C3 fits one CTA per system (HYBRID); C4b is one long system across CTAs (LONG).  ANY grid length
    # takes one of the two ("any N >= 3 must work"): ragged partitions on a power-of-two number
    # of threads (the paper's N = 201), ragged last tile.  Only systems of fewer than 7 rows and
    # batches of long rows that do not start on 16-byte boundaries fall back to one thread per system.
    assert B.plan_query(B.OP_BTCS, True, 4096, 2048, B.BC_PERIODIC) == B.PLAN_HYBRID
    assert B.plan_query(B.OP_BTCS, True, 1, 1 << 22, B.BC_PERIODIC) == B.PLAN_LONG
    for bc in (B.BC_PERIODIC, B.BC_DIRICHLET):
        for is64 in (False, True):
            for N in (7, 8, 24, 201, 1000, 2000, 3001, 4096):
                assert B.plan_query(B.OP_BTCS, is64, 3, N, bc) == B.PLAN_HYBRID, (N, is64)
                assert B.workspace_bytes(B.OP_BTCS, is64, 3, N, bc) == 0
            for N in (10001, 3000000, (1 << 22) + 40):
                assert B.plan_query(B.OP_BTCS, is64, 1, N, bc) == B.PLAN_LONG, (N, is64)
            assert B.plan_query(B.OP_BTCS, is64, 4, 3000000, bc) == B.PLAN_LONG
            assert B.plan_query(B.OP_BTCS, is64, 4, 3000001, bc) == B.PLAN_THOMAS      # misaligned rows
            assert B.plan_query(B.OP_BTCS, is64, 4, 5, bc) == B.PLAN_THOMAS
    assert B.plan_query(B.OP_BTCS, True, 3, 6000, 0) == B.PLAN_LONG and B.plan_query(B.OP_BTCS, False, 3, 8192, 0) == B.PLAN_HYBRID
    assert B.launch_count(B.OP_BTCS, True, 4096, 2048, 0, n_steps=1000) == 1
    # LONG: 50 launches of four steps on 512-thread tiles + fixup + GENERAL; 203 steps: + 3 single steps
    assert B.launch_count(B.OP_BTCS, True, 1, 1 << 22, 0, n_steps=200) == 52
    assert B.launch_count(B.OP_BTCS, True, 1, 1 << 22, 0, n_steps=203) == 55
    assert B.launch_count(B.OP_BTCS, True, 1, 1 << 22, 0, n_steps=1) == 3
    assert B.launch_count(B.OP_BTCS, True, 1, 6000, 0, n_steps=10) == 12     # too short for the wide tiles
    assert B.launch_count(B.OP_BTCS, True, 1, 1 << 22, 0, plan=B.PLAN_LONG_GENERAL, n_steps=200) == 1
    assert B.workspace_bytes(B.OP_BTCS, True, 1, 1 << 22, 0) >= int(2.5 * 8 * (1 << 22))
    assert B.workspace_bytes(B.OP_BTCS, True, 1, 1000, 0, 0, B.PLAN_LONG) == 0      # does not fit
    # Newton BTCS: resident plan for any 7 <= N that fits one CTA, else thread per system (workspace)
    assert B.plan_query(B.OP_NEWTON, True, 4096, 2048, B.BC_PERIODIC) == B.PLAN_HYBRID
    for N in (7, 201, 1000, 3001, 4096):
        assert B.plan_query(B.OP_NEWTON, True, 1, N, B.BC_DIRICHLET) == B.PLAN_HYBRID
        assert B.plan_query(B.OP_NEWTON, False, 1, N, B.BC_PERIODIC) == B.PLAN_HYBRID
    assert B.plan_query(B.OP_NEWTON, True, 1, 5, B.BC_DIRICHLET) == B.PLAN_THOMAS
    assert B.plan_query(B.OP_NEWTON, True, 1, 100000, B.BC_DIRICHLET) == B.PLAN_THOMAS
    assert B.workspace_bytes(B.OP_NEWTON, True, 4096, 2048, B.BC_PERIODIC) == 0
    assert B.workspace_bytes(B.OP_NEWTON, True, 2, 201, B.BC_PERIODIC) == 0
    assert B.workspace_bytes(B.OP_NEWTON, True, 2, 100001, B.BC_PERIODIC) >= 6 * 2 * 100001 * 8
    assert B.launch_count(B.OP_NEWTON, True, 4096, 2048, 0, n_steps=1000) == 1
    assert B.launch_count(B.OP_CFL, False, 1024, 4096, 1) == 1
    assert B.launch_count(B.OP_CFL, False, 1, 1 << 24, 0) == 2


def test_device_entry_points_refuse_cpu_tensors(B):
    import torch
    u = torch.zeros(2, 8, dtype=torch.float64)
    v = torch.ones(2, dtype=torch.float64)
    with pytest.raises(TypeError):
        B.burgers_explicit(u, 1.0, v, v, 1, B.BC_PERIODIC, B.SCHEME_EULER)
    with pytest.raises(TypeError):
        B.burgers_btcs(u, 1.0, v, v, 1, B.BC_PERIODIC)
    with pytest.raises(TypeError):
        B.dt_from_cfl(u, 1.0, v, 0.4, B.BC_PERIODIC)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2601_12204_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "burgers_oracle" not in txt and "liboracle" not in txt, f


def test_plain_c_client_compiles_links_and_runs(tmp_path):
    """include/burgers.h is valid C99 (-pedantic -Werror) and a C program needs nothing but the header and
    libburgers.so; argument errors are status codes, returned before any device work."""
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    libdir = os.path.join(root, "paper_2601_12204_b200")
    exe = str(tmp_path / "c_abi_client")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(root, "include"),
                    os.path.join(root, "tests", "c_abi_client.c"), "-o", exe, "-L", libdir, "-lburgers", "-lm",
                    "-Wl,-rpath," + libdir], check=True)
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.startswith("version ") and r.stdout.strip().endswith("bad 0")


def test_binding_rejects_short_per_trajectory_arrays_before_the_library_is_called(B):
    """a nu / dt / iters_out array shorter than B would be read or written out of bounds on the device;
    every binding entry point checks the lengths first (host entry points can be checked without a GPU)."""
    import numpy as np
    u = np.zeros((3, 16)); ok = np.ones(3); short = np.ones(2)
    for call in (lambda: B.burgers_explicit_host(u, 1.0, short, ok, 1, 0, 0),
                 lambda: B.burgers_explicit_host(u, 1.0, ok, short, 1, 0, 0),
                 lambda: B.burgers_btcs_host(u, 1.0, ok, short, 1, 0),
                 lambda: B.burgers_newton_host(u, 1.0, short, ok, 1, 0),
                 lambda: B.burgers_solve_host(u, 1.0, short, 0.4, 1, 0),
                 lambda: B.dt_from_cfl_host(u, 1.0, short, 0.4, 0)):
        with pytest.raises(ValueError, match="length B"):
            call()
    with pytest.raises(TypeError):                       # device entry points refuse host arrays (no CPU fallback)
        B.burgers_explicit(u, 1.0, ok, ok, 1, 0, 0)
