"""Pins of the CPU oracle against what the paper and the mathematics fix
(SURVEY.md 8(c) R1-R4, G1-G8).  No GPU; nothing here calls the CUDA path."""
import math

import numpy as np
import pytest

import oracle
from oracle import DIRICHLET, EULER, PERIODIC, RK4
from refs import amplification, colehopf_sin, read_colehopf_golden, read_golden

W = read_golden("worked_example_4node.txt")
U4 = np.array([1.0, 2.0, -1.0, 0.0])


# ---------------------------------------------------------------- G1 / G4
def test_worked_example_rhs_and_explicit_periodic():
    # PAPER.md:216 Eq.21 with the upwind rule of PAPER.md:89, exact rational values
    np.testing.assert_allclose(oracle.rhs(U4, 4.0, 0.1, PERIODIC), W["F_periodic"], rtol=0, atol=2e-15)
    e1 = oracle.explicit(U4, 4.0, 0.1, 0.1, 1, PERIODIC, EULER)
    np.testing.assert_allclose(e1, W["euler_periodic"], rtol=0, atol=2e-15)
    e2 = oracle.explicit(U4, 4.0, 0.1, 0.1, 2, PERIODIC, EULER)
    np.testing.assert_allclose(e2, W["euler2_periodic"], rtol=0, atol=4e-15)
    k = oracle.explicit(U4, 4.0, 0.1, 0.1, 1, PERIODIC, RK4)      # Eq.22
    np.testing.assert_allclose(k, W["rk4_periodic"], rtol=0, atol=4e-15)


def test_worked_example_dirichlet():
    e1 = oracle.explicit(U4, 3.0, 0.1, 0.1, 1, DIRICHLET, EULER)
    np.testing.assert_allclose(e1, W["euler_dirichlet"], rtol=0, atol=2e-15)
    k = oracle.explicit(U4, 3.0, 0.1, 0.1, 1, DIRICHLET, RK4)
    np.testing.assert_allclose(k, W["rk4_dirichlet"], rtol=0, atol=4e-15)
    x = oracle.btcs(U4, 3.0, 0.1, 0.1, 1, DIRICHLET)
    np.testing.assert_allclose(x, W["btcs_dirichlet"], rtol=0, atol=4e-15)


def test_worked_example_btcs_rows_and_solution():
    sub, diag, sup, rhs = oracle.btcs_rows(U4, 4.0, 0.1, 0.1, PERIODIC)
    np.testing.assert_allclose(sub, W["btcs_sub"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(diag, W["btcs_diag"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(sup, W["btcs_sup"], rtol=0, atol=1e-15)
    np.testing.assert_array_equal(rhs, U4)
    x = oracle.btcs(U4, 4.0, 0.1, 0.1, 1, PERIODIC)
    np.testing.assert_allclose(x, W["btcs_periodic"], rtol=0, atol=4e-15)


# ---------------------------------------------------------------- R1 / G2
def test_colehopf_reference_matches_golden():
    for nu, xf, u in read_colehopf_golden():
        got = colehopf_sin(np.array([xf * math.pi]), 1.0, nu)[0]
        assert abs(got - u) < 5e-15, (nu, xf, got, u)


def _run_c1(N, scheme, nu=0.05, T=1.0):
    L = 2 * math.pi
    u0 = np.sin(2 * math.pi * np.arange(N) / N)
    if scheme == "btcs":
        dtc = oracle.dt_from_cfl(u0, L, nu, 4.0, PERIODIC)[0]       # 10 x (0.4 x limit)
    elif scheme == "rk4":
        dtc = oracle.dt_from_cfl(u0, L, nu, 0.8, PERIODIC)[0]
    else:
        dtc = oracle.dt_from_cfl(u0, L, nu, 0.4, PERIODIC)[0]
    n = int(math.ceil(T / dtc - 1e-12))
    dt = T / n
    if scheme == "btcs":
        u = oracle.btcs(u0, L, nu, dt, n, PERIODIC)
    else:
        u = oracle.explicit(u0, L, nu, dt, n, PERIODIC, RK4 if scheme == "rk4" else EULER)
    exact = colehopf_sin(np.arange(N) * L / N, T, nu)
    err = u - exact
    return n, math.sqrt(np.mean(err ** 2)), np.abs(err).max()


def test_c1_step_counts_G5():
    # dx = 2pi/256, diffusive limit binds: 0.4 dx^2/(2 nu) = 2.409571e-3 -> n = 416; BTCS 10x -> 42
    n, _, _ = _run_c1(256, "euler")
    assert n == 416
    n, _, _ = _run_c1(256, "btcs")
    assert n == 42


@pytest.mark.parametrize("scheme,lo,hi", [("euler", 0.9e-2, 1.25e-2), ("rk4", 0.9e-2, 1.3e-2),
                                           ("btcs", 1.5e-2, 2.1e-2)])
def test_c1_error_vs_colehopf(scheme, lo, hi):
    # first-order upwind at N=256: RMS error ~1e-2 (Euler 1.07e-2, BTCS 1.8e-2); a wrong sign,
    # dropped term or transposed neighbour gives O(1) or an O(0.1) error instead
    _, rms, mx = _run_c1(256, scheme)
    assert lo < rms < hi, rms
    assert mx < 6e-2


@pytest.mark.parametrize("scheme", ["euler", "rk4", "btcs"])
def test_observed_order_is_one(scheme):
    errs = [_run_c1(N, scheme)[1] for N in (256, 512, 1024)]
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    if scheme == "btcs":
        assert 0.9 < orders[1] < 1.45 and orders[1] <= orders[0] + 0.05, orders
    else:
        assert 0.88 < orders[0] < 1.1 and 0.92 < orders[1] < 1.08, orders


# ---------------------------------------------------------------- R2 / G3
@pytest.mark.parametrize("scheme", ["euler", "rk4", "btcs"])
@pytest.mark.parametrize("adv", [0.7, -1.3])
@pytest.mark.parametrize("N,k", [(16, 1), (16, 5), (37, 11)])
def test_fourier_amplification(scheme, adv, N, k):
    L, nu, dt, nsteps, phase = 3.0, 0.02, 0.011, 7, 0.3
    dx = L / N
    theta = 2 * math.pi * k / N
    i = np.arange(N)
    u0 = np.cos(theta * i + phase)
    c, r = abs(adv) * dt / dx, nu * dt / dx ** 2
    G = amplification(scheme, theta, c, r, sigma=math.copysign(1.0, adv))
    want = np.real(G ** nsteps * np.exp(1j * (theta * i + phase)))
    if scheme == "btcs":
        got = oracle.btcs(u0, L, nu, dt, nsteps, PERIODIC, adv=adv)
    else:
        got = oracle.explicit(u0, L, nu, dt, nsteps, PERIODIC,
                              RK4 if scheme == "rk4" else EULER, adv=adv)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-13 * max(1.0, abs(G) ** nsteps))


@pytest.mark.parametrize("scheme", ["euler", "rk4", "btcs"])
def test_fourier_amplification_unstable_dt(scheme):
    # the formula holds for any dt, stable or not
    N, k, L, nu, adv, dt, nsteps = 16, 7, 1.0, 0.05, 1.0, 0.05, 5
    dx = L / N
    theta = 2 * math.pi * k / N
    i = np.arange(N)
    u0 = np.cos(theta * i)
    G = amplification(scheme, theta, abs(adv) * dt / dx, nu * dt / dx ** 2)
    want = np.real(G ** nsteps * np.exp(1j * theta * i))
    got = (oracle.btcs(u0, L, nu, dt, nsteps, PERIODIC, adv=adv) if scheme == "btcs" else
           oracle.explicit(u0, L, nu, dt, nsteps, PERIODIC, RK4 if scheme == "rk4" else EULER, adv=adv))
    np.testing.assert_allclose(got, want, rtol=1e-11, atol=1e-12 * max(1.0, abs(G) ** nsteps))


@pytest.mark.parametrize("scheme", ["euler", "rk4", "btcs"])
def test_dirichlet_heat_eigenvector(scheme):
    # adv = 0: heat equation; sin(k pi i/(N-1)) is an exact eigenvector, z = -4 r sin^2(k pi/(2(N-1)))  (G7)
    N, k, L, nu, dt, nsteps = 21, 3, 2.0, 0.3, 0.004, 9
    dx = L / (N - 1)
    r = nu * dt / dx ** 2
    z = -4 * r * math.sin(k * math.pi / (2 * (N - 1))) ** 2
    G = {"euler": 1 + z, "rk4": 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24, "btcs": 1 / (1 - z)}[scheme]
    u0 = np.sin(k * math.pi * np.arange(N) / (N - 1))
    u0[0] = u0[-1] = 0.0
    got = (oracle.btcs(u0, L, nu, dt, nsteps, DIRICHLET, adv=0.0) if scheme == "btcs" else
           oracle.explicit(u0, L, nu, dt, nsteps, DIRICHLET, RK4 if scheme == "rk4" else EULER, adv=0.0))
    np.testing.assert_allclose(got, G ** nsteps * u0, rtol=0, atol=1e-14)


def test_pure_upwind_shift_G7():
    # nu = 0, constant speed, c = 1: exactly a one-cell shift per step
    N, L = 12, 12.0
    rng = np.random.default_rng(3)
    u0 = rng.standard_normal(N)
    got = oracle.explicit(u0, L, 0.0, 1.0, 5, PERIODIC, EULER, adv=1.0)
    np.testing.assert_allclose(got, np.roll(u0, 5), rtol=0, atol=1e-14)
    got = oracle.explicit(u0, L, 0.0, 1.0, 5, PERIODIC, EULER, adv=-1.0)
    np.testing.assert_allclose(got, np.roll(u0, -5), rtol=0, atol=1e-14)


# ---------------------------------------------------------------- R3
def _dense_btcs(u, L, nu, dt, bc):
    N = len(u)
    dx = L / N if bc == PERIODIC else L / (N - 1)
    r = nu * dt / dx ** 2
    M = np.zeros((N, N))
    for i in range(N):
        c = u[i] * dt / dx
        M[i, (i - 1) % N] += -r - max(c, 0.0)
        M[i, i] += 1 + 2 * r + abs(c)
        M[i, (i + 1) % N] += -r + min(c, 0.0)
    if bc == PERIODIC:
        return np.linalg.solve(M, u)
    x = u.copy()
    rhs = u[1:-1] - M[1:-1, 0] * u[0] - M[1:-1, -1] * u[-1]
    x[1:-1] = np.linalg.solve(M[1:-1, 1:-1], rhs)
    return x


@pytest.mark.parametrize("bc", [PERIODIC, DIRICHLET])
@pytest.mark.parametrize("N", [3, 4, 5, 8, 13, 16])
def test_btcs_step_vs_dense_gaussian_elimination(bc, N):
    rng = np.random.default_rng(100 + N)
    for trial in range(12):
        u = rng.uniform(-2, 2, N)
        if trial == 0:
            u = -np.abs(u) - 0.1          # all negative
        if trial == 1:
            u = np.abs(u) + 0.1           # all positive
        L = rng.uniform(0.5, 7.0)
        dx = L / N if bc == PERIODIC else L / (N - 1)
        r = rng.uniform(0.01, 50.0)
        dt = rng.uniform(0.01, 3.0) * dx
        nu = r * dx * dx / dt
        want = _dense_btcs(u, L, nu, dt, bc)
        got = oracle.btcs(u, L, nu, dt, 1, bc)
        np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-13)


@pytest.mark.parametrize("n", [2, 3, 7, 16])
def test_thomas_and_cyclic_vs_dense(n):
    rng = np.random.default_rng(n)
    sub, sup = -rng.uniform(0.1, 3, n), -rng.uniform(0.1, 3, n)
    diag = 1.0 - sub - sup
    rhs = rng.standard_normal(n)
    M = np.diag(diag) + np.diag(sub[1:], -1) + np.diag(sup[:-1], 1)
    np.testing.assert_allclose(oracle.thomas(sub, diag, sup, rhs), np.linalg.solve(M, rhs), rtol=1e-13)
    if n >= 3:
        M[0, n - 1] += sub[0]
        M[n - 1, 0] += sup[n - 1]
        np.testing.assert_allclose(oracle.cyclic(sub, diag, sup, rhs), np.linalg.solve(M, rhs), rtol=1e-13)


# ---------------------------------------------------------------- R4 / D8
def test_dt_from_cfl_branches_and_zero_cases():
    N, L = 11, 2.0
    u = np.zeros((4, N))
    u[0, 3] = -4.0                      # convective bound binds
    u[1, 5] = 1e-3                      # diffusive bound binds
    u[2, 0] = 2.0                       # nu = 0 -> convective
    nu = np.array([1e-3, 0.5, 0.0, 0.0])
    dxp, dxd = L / N, L / (N - 1)
    got = oracle.dt_from_cfl(u, L, nu, 0.4, PERIODIC)
    assert got[0] == pytest.approx(0.4 * dxp / 4.0, rel=1e-15)
    assert got[1] == pytest.approx(0.4 * dxp ** 2 / (2 * 0.5), rel=1e-15)
    assert got[2] == pytest.approx(0.4 * dxp / 2.0, rel=1e-15)
    assert math.isinf(got[3])
    got = oracle.dt_from_cfl(u, L, nu, 1.0, DIRICHLET)   # Dirichlet: dx = L/(N-1), end nodes count
    assert got[2] == pytest.approx(dxd / 2.0, rel=1e-15)
    assert got[1] == pytest.approx(dxd ** 2 / (2 * 0.5), rel=1e-15)


def test_cfl_violation_breaks_max_principle_R4():
    # adv = 0, r = 0.51 on a +-1 sawtooth: amplitude grows by |1 - 4r| per step
    N, L = 16, 16.0
    saw = np.where(np.arange(N) % 2 == 0, 1.0, -1.0)
    u = oracle.explicit(saw, L, 0.51, 1.0, 10, PERIODIC, EULER, adv=0.0)
    assert np.abs(u).max() == pytest.approx(abs(1 - 4 * 0.51) ** 10, rel=1e-12)
    u = oracle.explicit(saw, L, 0.25, 1.0, 10, PERIODIC, EULER, adv=0.0)
    assert np.abs(u).max() <= 1.0


# ---------------------------------------------------------------- G6 invariants
@pytest.mark.parametrize("bc", [PERIODIC, DIRICHLET])
def test_constant_state_is_fixed_point(bc):
    u0 = np.full(17, 1.375)
    for sch in (EULER, RK4):
        np.testing.assert_array_equal(oracle.explicit(u0, 1.0, 0.01, 1e-3, 20, bc, sch), u0)
    np.testing.assert_allclose(oracle.btcs(u0, 1.0, 0.01, 0.5, 20, bc), u0, rtol=0, atol=1e-14)


def test_max_principle():
    rng = np.random.default_rng(5)
    N, L = 64, 1.0
    u0 = rng.uniform(-1, 2, (6, N))
    nu = rng.uniform(1e-3, 1e-1, 6)
    dt = oracle.dt_from_cfl(u0, L, nu, 0.5, PERIODIC)        # |c| + 2r <= 1
    u = oracle.explicit(u0, L, nu, dt, 200, PERIODIC, EULER)
    assert (u.max(1) <= u0.max(1) + 1e-14).all() and (u.min(1) >= u0.min(1) - 1e-14).all()
    ub = oracle.btcs(u0, L, nu, 50 * dt, 30, PERIODIC)       # any dt
    assert (ub.max(1) <= u0.max(1) + 1e-13).all() and (ub.min(1) >= u0.min(1) - 1e-13).all()
    ud = oracle.btcs(u0, L, nu, 50 * dt, 30, DIRICHLET)
    assert (ud.max(1) <= u0.max(1) + 1e-13).all() and (ud.min(1) >= u0.min(1) - 1e-13).all()
    np.testing.assert_array_equal(ud[:, [0, -1]], u0[:, [0, -1]])


def test_btcs_rows_sum_to_one_and_are_dominant():
    rng = np.random.default_rng(6)
    u = rng.uniform(-3, 3, 40)
    sub, diag, sup, _ = oracle.btcs_rows(u, 2.0, 0.03, 0.2, PERIODIC)
    np.testing.assert_allclose(sub + diag + sup, 1.0, rtol=0, atol=1e-12)
    assert (sub <= 0).all() and (sup <= 0).all() and (diag > 0).all()
    np.testing.assert_allclose(np.abs(diag) - np.abs(sub) - np.abs(sup), 1.0, atol=1e-12)


def test_odd_symmetry_is_preserved_exactly():
    # periodic, N even, u_{N-i} = -u_i constructed exactly: stays exactly odd under Euler/RK4;
    # fails for the backward-only reading of Eq.3 (Q2)
    N = 32
    rng = np.random.default_rng(7)
    h = rng.uniform(-1, 1, N // 2 - 1)
    u0 = np.zeros(N)
    u0[1:N // 2] = h
    u0[N // 2 + 1:] = -h[::-1]
    for sch in (EULER, RK4):
        u = oracle.explicit(u0, 2 * math.pi, 0.05, 2e-3, 50, PERIODIC, sch)
        np.testing.assert_array_equal(u[1:N // 2], -u[N // 2 + 1:][::-1])
        assert u[0] == 0.0 and u[N // 2] == 0.0
    ub = oracle.btcs(u0, 2 * math.pi, 0.05, 5e-2, 20, PERIODIC)
    np.testing.assert_allclose(ub[1:N // 2], -ub[N // 2 + 1:][::-1], rtol=0, atol=1e-14)


def test_steps_compose_bitwise():
    rng = np.random.default_rng(8)
    u0 = rng.uniform(-1, 1, (3, 50))
    nu = np.array([0.01, 0.02, 0.05])
    dt = oracle.dt_from_cfl(u0, 1.0, nu, 0.4, DIRICHLET)
    for sch in (EULER, RK4):
        a = oracle.explicit(oracle.explicit(u0, 1.0, nu, dt, 7, DIRICHLET, sch), 1.0, nu, dt, 5, DIRICHLET, sch)
        np.testing.assert_array_equal(a, oracle.explicit(u0, 1.0, nu, dt, 12, DIRICHLET, sch))
    a = oracle.btcs(oracle.btcs(u0, 1.0, nu, 9 * dt, 3, PERIODIC), 1.0, nu, 9 * dt, 4, PERIODIC)
    np.testing.assert_array_equal(a, oracle.btcs(u0, 1.0, nu, 9 * dt, 7, PERIODIC))


def test_threads_do_not_change_results():
    rng = np.random.default_rng(9)
    u0 = rng.uniform(-1, 1, (9, 40))
    nu = rng.uniform(0.01, 0.05, 9)
    dt = oracle.dt_from_cfl(u0, 1.0, nu, 0.4, PERIODIC)
    a = oracle.explicit(u0, 1.0, nu, dt, 30, PERIODIC, RK4, threads=1)
    b = oracle.explicit(u0, 1.0, nu, dt, 30, PERIODIC, RK4, threads=4)
    np.testing.assert_array_equal(a, b)
    c = oracle.explicit_long(u0[0], 1.0, nu[0], dt[0], 30, PERIODIC, threads=3)
    np.testing.assert_array_equal(c, oracle.explicit(u0[0], 1.0, nu[0], dt[0], 30, PERIODIC, EULER))
    d = oracle.explicit_long(u0[0], 1.0, nu[0], dt[0], 31, DIRICHLET, threads=2)
    np.testing.assert_array_equal(d, oracle.explicit(u0[0], 1.0, nu[0], dt[0], 31, DIRICHLET, EULER))


# ---------------------------------------------------------------- G8
@pytest.mark.parametrize("scheme", ["euler", "rk4", "btcs"])
def test_travelling_viscous_shock_dirichlet(scheme):
    # u = s - (D/2) tanh(D (x - x0 - s t)/(4 nu)) is an exact solution on the line (PAPER.md:399
    # describes this front); both signs of u occur, so both upwind branches are exercised
    uL, uR, nu, L, T = 1.0, -0.4, 0.02, 4.0, 1.0
    D, s = uL - uR, 0.5 * (uL + uR)
    errs = []
    for N in (201, 401):
        x = np.linspace(0.0, L, N)
        exact = lambda t: s - 0.5 * D * np.tanh(D * (x - 1.5 - s * t) / (4 * nu))
        u0 = exact(0.0)
        C = {"euler": 0.4, "rk4": 0.8, "btcs": 2.0}[scheme]
        dtc = oracle.dt_from_cfl(u0, L, nu, C, DIRICHLET)[0]
        n = int(math.ceil(T / dtc))
        dt = T / n
        u = (oracle.btcs(u0, L, nu, dt, n, DIRICHLET) if scheme == "btcs" else
             oracle.explicit(u0, L, nu, dt, n, DIRICHLET, RK4 if scheme == "rk4" else EULER))
        errs.append(math.sqrt(np.mean((u - exact(T)) ** 2)))
    assert errs[0] < 0.15 and 0.7 < math.log2(errs[0] / errs[1]) < 1.3, errs


# ---------------------------------------------------------------- E5: the step of PAPER.md:193 (Eq.20)
def test_step_function_btcs_is_stable_at_five_times_the_convective_limit():
    """"the implicit solver remained stable even for dt = 5 dx/u_max" on the step initial
    condition of Eq.20 (N = 201, nu = 0.01).  For the lagged upwind BTCS of D4 this is a
    theorem, not an observation: the matrix is an M-matrix with unit row sums (max principle for any dt) and,
    with u >= 0, the scheme has Harten's implicit TVD form (C_{i-1/2} = r + c_i >= 0, D_{i+1/2} = r >= 0), so a
    monotone profile stays monotone and its total variation cannot grow.  The explicit scheme at the same dt
    (|c| + 2r = 5 + 20 >> 1) must blow up."""
    from paper_2601_12204_b200 import workloads as WL
    w = WL.step_dirichlet()
    dx = w.L / (w.N - 1)
    dt = np.array([w.meta["dt"]])
    assert dt[0] == 5.0 * dx / np.abs(w.u0).max()                           # "dt = 5 dx/u_max", r = nu dt/dx^2 = 10
    x = np.arange(w.N) * dx
    front = []
    for n in (1, 4, 8, 16):
        u = oracle.btcs(w.u0, w.L, w.nu, dt, n, w.bc)[0]
        assert u[0] == 1.0 and u[-1] == 0.0                                 # frozen ends (Q8)
        assert u.min() >= 0.0 and u.max() <= 1.0 + 1e-14                    # max principle at C = 5
        assert np.all(np.diff(u) <= 1e-14)                                  # monotone: no oscillation at the front
        assert np.abs(np.diff(u)).sum() <= 1.0 + 1e-13                      # total variation does not grow
        i = int(np.argmax(u < 0.5))
        front.append(x[i - 1] + (u[i - 1] - 0.5) / (u[i - 1] - u[i]) * dx)
    # the front travels to the right (u > 0: backward differences), at a speed of the order of the
    # Rankine-Hugoniot value (u_L + u_R)/2 = 1/2 (the non-conservative lagged form at C = 5 is slower)
    assert np.all(np.diff(front) > 0)
    speed = (front[-1] - front[1]) / (12 * dt[0])
    assert 0.3 < speed < 0.6, speed
    blown = oracle.explicit(w.u0, w.L, w.nu, dt, 8, w.bc, EULER)[0]
    assert not (np.abs(blown).max() <= 10.0)
