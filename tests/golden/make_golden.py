"""Writes the text fixtures in this folder.  Calls neither oracle/ nor the CUDA path.

Everything here is computed from the mathematics alone, by a method different
from the oracle's:

* ``worked_example_4node.txt`` -- the 4-node worked example (periodic, N=4, L=4
  so dx=1, nu=1/10, dt=1/10, u=[1,2,-1,0]) advanced by
  Eq.21, Eq.22 and the BTCS system of
  DESIGN.md D4 in EXACT rational arithmetic (``fractions.Fraction``), the linear
  systems solved by exact Gauss-Jordan elimination on the dense matrix.
* ``colehopf_sin.txt`` -- the exact solution of Eq.1 for
  u(x,0)=sin x on [0,2pi) at t=1 through the Cole-Hopf transformation
  (PAPER.md:204, :283): u = int (x-y)/t K dy / int K dy,
  K = exp(-(x-y)^2/(4 nu t) - (1-cos y)/(2 nu)).  The stored value is the
  equivalent Bessel/Fourier series u = 4 nu sum k I_k(z) e^{-nu k^2 t} sin kx /
  (I_0(z) + 2 sum I_k(z) e^{-nu k^2 t} cos kx), z = 1/(2 nu), summed in 150-digit
  arithmetic (mpmath) and cross-checked to 1e-18 against 50-digit quadrature of
  the heat-kernel integrals above.

Run:  python tests/golden/make_golden.py
"""
from __future__ import annotations

import os
from fractions import Fraction as Fr

import mpmath as mp

HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------
# exact rational worked example
# ----------------------------------------------------------------------------
def F_exact(u, dx, nu, bc):
    N = len(u)
    F = [Fr(0)] * N
    rng = range(N) if bc == "periodic" else range(1, N - 1)
    for i in rng:
        um, up, ui = u[(i - 1) % N], u[(i + 1) % N], u[i]
        g = (ui - um) if ui > 0 else (up - ui)          # upwind rule
        F[i] = -ui * g / dx + nu * (up - 2 * ui + um) / dx ** 2   # Eq.21
    return F


def euler_exact(u, dx, nu, dt, bc):
    F = F_exact(u, dx, nu, bc)
    return [a + dt * f for a, f in zip(u, F)]


def rk4_exact(u, dx, nu, dt, bc):
    k1 = F_exact(u, dx, nu, bc)
    k2 = F_exact([a + dt / 2 * k for a, k in zip(u, k1)], dx, nu, bc)
    k3 = F_exact([a + dt / 2 * k for a, k in zip(u, k2)], dx, nu, bc)
    k4 = F_exact([a + dt * k for a, k in zip(u, k3)], dx, nu, bc)
    return [a + dt / 6 * (p + 2 * q + 2 * r + s)
            for a, p, q, r, s in zip(u, k1, k2, k3, k4)]


def solve_exact(M, rhs):
    n = len(rhs)
    A = [row[:] + [rhs[i]] for i, row in enumerate(M)]
    for c in range(n):
        piv = next(r for r in range(c, n) if A[r][c] != 0)
        A[c], A[piv] = A[piv], A[c]
        A[c] = [v / A[c][c] for v in A[c]]
        for r in range(n):
            if r != c and A[r][c] != 0:
                A[r] = [vr - A[r][c] * vc for vr, vc in zip(A[r], A[c])]
    return [A[i][n] for i in range(n)]


def btcs_exact(u, dx, nu, dt, bc):
    """(u_i^{n+1}-u_i^n)/dt + u_i^n upwind_x(u^{n+1}) = nu central_xx(u^{n+1})."""
    N = len(u)
    r = nu * dt / dx ** 2
    rows = []
    M = [[Fr(0)] * N for _ in range(N)]
    for i in range(N):
        c = u[i] * dt / dx
        sub, diag, sup = -r - max(c, 0), 1 + 2 * r + abs(c), -r + min(c, 0)
        rows.append((sub, diag, sup))
        M[i][(i - 1) % N] += sub
        M[i][i] += diag
        M[i][(i + 1) % N] += sup
    if bc == "periodic":
        return rows, solve_exact(M, list(u))
    idx = list(range(1, N - 1))
    Mi = [[M[i][j] for j in idx] for i in idx]
    rhs = [u[i] - M[i][0] * u[0] - M[i][N - 1] * u[N - 1] for i in idx]   # D5
    x = solve_exact(Mi, rhs)
    return rows, [u[0]] + x + [u[N - 1]]


def newton_exact(u, dx, nu, dt, bc, iters, theta=Fr(1)):
    """`iters` Newton iterations on the residual of PAPER.md Eq.11 (central convection, all terms at
    n+1) from w0 = u^n, with the Jacobian obtained by differentiating Eq.11 (Q5/D11).
    theta != 1: theta-scheme F = w - u + theta G(w) + (1-theta) G(u), G = dt * central operator."""
    N = len(u)
    h, r = dt / (2 * dx), nu * dt / dx ** 2
    idx = list(range(N)) if bc == "periodic" else list(range(1, N - 1))
    w = list(u)
    out = []

    def G(v, i):
        return h * v[i] * (v[(i + 1) % N] - v[(i - 1) % N]) - r * (v[(i + 1) % N] - 2 * v[i] + v[(i - 1) % N])

    for _ in range(iters):
        F = {}
        M = [[Fr(0)] * N for _ in range(N)]
        for i in idx:
            wm, wp, wi = w[(i - 1) % N], w[(i + 1) % N], w[i]
            F[i] = wi - u[i] + theta * G(w, i) + (1 - theta) * G(u, i)          # Eq.11 at theta = 1
            M[i][(i - 1) % N] += theta * (-h * wi - r)
            M[i][i] += 1 + theta * (h * (wp - wm) + 2 * r)
            M[i][(i + 1) % N] += theta * (h * wi - r)
        Mi = [[M[i][j] for j in idx] for i in idx]          # frozen end nodes: delta = 0
        d = solve_exact(Mi, [-F[i] for i in idx])           # Eq.12
        for i, di in zip(idx, d):
            w[i] = w[i] + di                                 # Eq.13
        out.append(list(w))
    return out


def write_newton_example():
    u = [Fr(1), Fr(2), Fr(-1), Fr(0)]
    dx, nu, dt = Fr(1), Fr(1, 10), Fr(1, 10)
    lines = [
        "# Newton-Raphson on PAPER.md Eq.11 (fully implicit, central convection), 4-node example:",
        "# u^n=[1,2,-1,0], dx=1, nu=0.1, dt=0.1; iterates w^1, w^2, w^3 from w^0 = u^n in exact rational",
        "# arithmetic (tests/golden/make_golden.py), rounded once to fp64.  Eq.12-13 PAPER.md:147-151.",
    ]
    N = len(u)
    h, r = dt / (2 * dx), nu * dt / dx ** 2
    F0 = [u[i] - u[i] + h * u[i] * (u[(i + 1) % N] - u[(i - 1) % N]) - r * (u[(i + 1) % N] - 2 * u[i] + u[(i - 1) % N])
          for i in range(N)]
    lines.append("F0_periodic " + fmt(F0))
    lines.append("J0_sub_periodic " + fmt([-h * u[i] - r for i in range(N)]))
    lines.append("J0_diag_periodic " + fmt([1 + h * (u[(i + 1) % N] - u[(i - 1) % N]) + 2 * r for i in range(N)]))
    lines.append("J0_sup_periodic " + fmt([h * u[i] - r for i in range(N)]))
    for k, w in enumerate(newton_exact(u, dx, nu, dt, "periodic", 3), 1):
        lines.append(f"newton{k}_periodic " + fmt(w))
    lines.append("# Dirichlet: same u, L=3 (dx=1), end nodes frozen at 1 and 0")
    for k, w in enumerate(newton_exact(u, dx, nu, dt, "dirichlet", 3), 1):
        lines.append(f"newton{k}_dirichlet " + fmt(w))
    lines.append("# theta = 1/2 (Crank-Nicolson on the central operator), same data")
    for k, w in enumerate(newton_exact(u, dx, nu, dt, "periodic", 3, Fr(1, 2)), 1):
        lines.append(f"cn{k}_periodic " + fmt(w))
    for k, w in enumerate(newton_exact(u, dx, nu, dt, "dirichlet", 3, Fr(1, 2)), 1):
        lines.append(f"cn{k}_dirichlet " + fmt(w))
    lines.append("# Gauss-Seidel sweeps on the lagged upwind BTCS system (D4/D12), same data, x0 = u^n")
    for k, x in enumerate(gs_exact(u, dx, nu, dt, "periodic", 3), 1):
        lines.append(f"gs{k}_periodic " + fmt(x))
    for k, x in enumerate(gs_exact(u, dx, nu, dt, "dirichlet", 3), 1):
        lines.append(f"gs{k}_dirichlet " + fmt(x))
    with open(os.path.join(HERE, "newton_4node.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


def gs_exact(u, dx, nu, dt, bc, sweeps):
    """`sweeps` lexicographic Gauss-Seidel sweeps on the BTCS system of D4 from x0 = u^n."""
    N = len(u)
    r = nu * dt / dx ** 2
    rows = []
    for i in range(N):
        c = u[i] * dt / dx
        rows.append((-r - max(c, 0), 1 + 2 * r + abs(c), -r + min(c, 0)))
    idx = list(range(N)) if bc == "periodic" else list(range(1, N - 1))
    x = list(u)
    out = []
    for _ in range(sweeps):
        for i in idx:
            sub, diag, sup = rows[i]
            x[i] = (u[i] - sub * x[(i - 1) % N] - sup * x[(i + 1) % N]) / diag
        out.append(list(x))
    return out


def fmt(vals):
    return " ".join(repr(float(v)) for v in vals)


def write_worked_example():
    u = [Fr(1), Fr(2), Fr(-1), Fr(0)]
    dx, nu, dt = Fr(1), Fr(1, 10), Fr(1, 10)
    lines = [
        "# 4-node worked example: periodic N=4, L=4 (dx=1), nu=0.1, dt=0.1, u=[1,2,-1,0]",
        "# exact rational arithmetic (tests/golden/make_golden.py), rounded once to fp64",
        "# Eq.21 PAPER.md:216, Eq.22 PAPER.md:224-229, BTCS rows DESIGN.md D4 (PAPER.md:237-241)",
        "F_periodic " + fmt(F_exact(u, dx, nu, "periodic")),
        "euler_periodic " + fmt(euler_exact(u, dx, nu, dt, "periodic")),
        "rk4_periodic " + fmt(rk4_exact(u, dx, nu, dt, "periodic")),
    ]
    u2 = euler_exact(euler_exact(u, dx, nu, dt, "periodic"), dx, nu, dt, "periodic")
    lines.append("euler2_periodic " + fmt(u2))
    rows, x = btcs_exact(u, dx, nu, dt, "periodic")
    for k, name in enumerate(("btcs_sub", "btcs_diag", "btcs_sup")):
        lines.append(name + " " + fmt([rw[k] for rw in rows]))
    lines.append("btcs_periodic " + fmt(x))
    # Dirichlet on the same 4 values: nodes 0 and 3 frozen at 1 and 0, dx = L/(N-1) with L=3
    lines.append("# Dirichlet: same u, L=3 (dx=1), end nodes frozen at 1 and 0")
    lines.append("euler_dirichlet " + fmt(euler_exact(u, dx, nu, dt, "dirichlet")))
    lines.append("rk4_dirichlet " + fmt(rk4_exact(u, dx, nu, dt, "dirichlet")))
    _, xd = btcs_exact(u, dx, nu, dt, "dirichlet")
    lines.append("btcs_dirichlet " + fmt(xd))
    with open(os.path.join(HERE, "worked_example_4node.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


# ----------------------------------------------------------------------------
# Cole-Hopf, u0 = sin x on [0, 2pi)
# ----------------------------------------------------------------------------
def colehopf_quad(x, t, nu):
    x, t, nu = mp.mpf(x), mp.mpf(t), mp.mpf(nu)
    s = mp.sqrt(4 * nu * t)

    def g(y):
        return mp.exp(-(1 - mp.cos(y)) / (2 * nu))

    # substitute y = x - s*eta: integrals over eta with weight exp(-eta^2)
    span = 14
    pts = [-span + k for k in range(2 * span + 1)]
    num = mp.quad(lambda e: e * mp.exp(-e * e) * g(x - s * e), pts)
    den = mp.quad(lambda e: mp.exp(-e * e) * g(x - s * e), pts)
    return (s / t) * num / den


def colehopf_series(x, t, nu, terms=400):
    x, t, nu = mp.mpf(x), mp.mpf(t), mp.mpf(nu)
    z = 1 / (2 * nu)
    num = mp.mpf(0)
    den = mp.besseli(0, z)
    for k in range(1, terms):
        ck = mp.besseli(k, z) * mp.exp(-nu * k * k * t)
        num += k * ck * mp.sin(k * x)
        den += 2 * ck * mp.cos(k * x)
    return 4 * nu * num / den


def write_colehopf():
    lines = [
        "# exact u(x, t=1) of u_t + u u_x = nu u_xx, u(x,0) = sin x, 2pi-periodic (Cole-Hopf)",
        "# columns: nu  x_as_multiple_of_pi  u   (150-digit Bessel/Fourier series; 50-digit heat-kernel quadrature agrees to 1e-18)",
    ]
    xs = [mp.mpf(1) / 4, mp.mpf(1) / 2, mp.mpf(3) / 4, mp.mpf(7) / 8, mp.mpf(1),
          mp.mpf(5) / 4, mp.mpf(13) / 8]
    for nu in ("0.05", "0.01"):
        for xf in xs:
            mp.mp.dps = 50
            uq = colehopf_quad(xf * mp.pi, 1, nu)
            mp.mp.dps = 150
            us = colehopf_series(xf * mp.pi, 1, nu)
            mp.mp.dps = 50
            assert abs(uq - us) < mp.mpf(10) ** -18, (nu, xf, uq, us)
            lines.append(f"{nu} {float(xf)!r} {mp.nstr(us, 20)}")
    with open(os.path.join(HERE, "colehopf_sin.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    write_worked_example()
    write_newton_example()
    write_colehopf()
    print("golden fixtures written to", HERE)
