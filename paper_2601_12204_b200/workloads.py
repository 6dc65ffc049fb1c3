"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic).

The paper measures on no dataset: its workloads are two analytic initial
conditions on N=201 grids (sine PAPER.md:189 Eq.19, step PAPER.md:193 Eq.20,
periodic / Dirichlet boundaries PAPER.md:171-181, nu = 0.01 PAPER.md:383).  The
configs of BASELINE.json keep that structure and scale B and N up; this module
generates exactly those inputs (recipe: DESIGN.md "Input recipe", SURVEY.md
8(d)).  Everything is drawn on the host in fp64 from
``numpy.random.default_rng(seed)`` with seed = 1220400 + config number, in the
draw order written below, then rounded to the workload's dtype.

Both the CUDA path (bench.py, tests) and the oracle (tests, cpu_baseline) read
the SAME rounded arrays from here.  The time step is NOT computed here: callers
obtain it from ``dt_from_cfl`` of whichever side they are driving.
"""
from __future__ import annotations

import hashlib
import math
from dataclasses import dataclass, field

import numpy as np

PERIODIC, DIRICHLET = 0, 1
EULER, RK4, BTCS = 0, 1, 2
SEED_BASE = 1220400


@dataclass
class Workload:
    name: str
    u0: np.ndarray            # [B][N], already rounded to `dtype`
    nu: np.ndarray            # [B]
    L: float
    bc: int
    scheme: int               # EULER / RK4 / BTCS
    cfl: float                # C of dt_from_cfl
    n_steps: int              # fixed step count (0 when final_time is used)
    dtype: np.dtype
    final_time: float = 0.0   # >0: n = ceil(T/dt_cfl), dt = T/n  (config 1)
    meta: dict = field(default_factory=dict)

    @property
    def B(self) -> int:
        return self.u0.shape[0]

    @property
    def N(self) -> int:
        return self.u0.shape[1]

    @property
    def updates(self) -> int:
        return self.B * self.N * self.n_steps

    def sha256(self) -> str:
        h = hashlib.sha256()
        h.update(np.ascontiguousarray(self.u0).tobytes())
        h.update(np.ascontiguousarray(self.nu).tobytes())
        return h.hexdigest()


def steps_for_final_time(dt_cfl: float, T: float):
    """Config-1 rule: n = ceil(T/dt_cfl), dt = T/n (fixed final time)."""
    n = int(math.ceil(T / float(dt_cfl) - 1e-12))
    return n, T / n


def _finish(name, u0, nu, L, bc, scheme, cfl, n_steps, dtype, **kw) -> Workload:
    dtype = np.dtype(dtype)
    return Workload(name, np.ascontiguousarray(u0.astype(dtype)),
                    np.ascontiguousarray(np.asarray(nu, dtype=np.float64).astype(dtype)),
                    float(L), bc, scheme, float(cfl), int(n_steps), dtype, **kw)


def c1_sine(N: int = 256, nu: float = 0.05, scheme: int = EULER, cfl: float = 0.4,
            dtype=np.float64) -> Workload:
    """Config 1: one trajectory, periodic [0,2pi), u0 = sin x, final time T=1."""
    L = 2.0 * math.pi
    i = np.arange(N, dtype=np.float64)
    u0 = np.sin(2.0 * math.pi * i / N)[None, :]
    return _finish(f"C1-sine-N{N}", u0, [nu], L, PERIODIC, scheme, cfl, 0, dtype,
                   final_time=1.0)


def step_dirichlet(N: int = 201, nu: float = 0.01, cfl: float = 5.0, n_steps: int = 16, L: float = 1.0,
                   dtype=np.float64) -> Workload:
    """The paper's step initial condition (Eq.20): u0 = 1 for x < L/2, 0 otherwise, on the
    paper's grid N = 201, nu = 0.01, Dirichlet ends (a = 1, b = 0 as found in u0).
    ``cfl`` = 5 is the factor of "dt = 5 dx/u_max": a multiple of the CONVECTIVE bound alone
    (at this N and nu the diffusive bound dx^2/(2 nu) is four times smaller, so dt_from_cfl would not give
    it); callers form dt = meta["dt"] = cfl * dx / max|u0| themselves."""
    dx = L / (N - 1)
    x = np.arange(N, dtype=np.float64) * dx
    u0 = np.where(x < 0.5 * L, 1.0, 0.0)[None, :]
    return _finish(f"step-dirichlet-N{N}", u0, [nu], L, DIRICHLET, BTCS, cfl, n_steps, dtype,
                   meta={"dt": cfl * dx / 1.0})


def c2_dirichlet_batch(B: int = 1024, N: int = 4096, n_steps: int = 10000,
                       dtype=np.float32, seed: int = SEED_BASE + 2, rows=None) -> Workload:
    """Config 2: B Dirichlet trajectories on [0,1], 8 sine modes, nu log-uniform.

    ``rows``: optional index array -- only those trajectories of the B-trajectory batch (all
    random draws are made for the whole batch first, so a subset / shard is bit-identical to
    the same rows of the full workload)."""
    rng = np.random.default_rng(seed)
    Z = rng.standard_normal((B, 8))
    k = np.arange(1, 9, dtype=np.float64)
    A = Z / np.sqrt(k)[None, :]                       # amplitudes ~ N(0, 1/k) (variance)
    lognu = rng.uniform(math.log(1e-3), math.log(1e-1), B)
    nu = np.exp(lognu)
    if rows is not None:
        rows = np.asarray(rows)
        A, nu = A[rows], nu[rows]
    x = np.arange(N, dtype=np.float64) / (N - 1)
    u0 = np.zeros((len(nu), N))
    for m in range(8):
        u0 += A[:, m:m + 1] * np.sin(k[m] * math.pi * x)[None, :]
    u0[:, 0] = 0.0
    u0[:, -1] = 0.0
    return _finish(f"C2-dirichlet-B{len(nu)}of{B}-N{N}", u0, nu, 1.0, DIRICHLET, EULER, 0.4,
                   n_steps, dtype)


def c3_periodic_btcs(B: int = 4096, N: int = 2048, n_steps: int = 1000,
                     dtype=np.float64, seed: int = SEED_BASE + 3, rows=None) -> Workload:
    """Config 3: B periodic trajectories, 1 + 0.5 sum of 4 random-phase modes k<=16.
    ``rows`` as in :func:`c2_dirichlet_batch`."""
    rng = np.random.default_rng(seed)
    ks = np.stack([rng.permutation(16)[:4] + 1 for _ in range(B)]).astype(np.float64)
    phi = rng.uniform(0.0, 2.0 * math.pi, (B, 4))
    if rows is not None:
        rows = np.asarray(rows)
        ks, phi = ks[rows], phi[rows]
    B = len(ks)
    L = 2.0 * math.pi
    x = np.arange(N, dtype=np.float64) * (L / N)
    u0 = np.ones((B, N))
    for j in range(4):
        u0 += 0.5 * np.cos(ks[:, j:j + 1] * x[None, :] + phi[:, j:j + 1])
    nu = np.full(B, 0.01)
    return _finish(f"C3-periodic-btcs-B{B}-N{N}", u0, nu, L, PERIODIC, BTCS, 10.0,
                   n_steps, dtype)


def _tophat(N: int, width_cells: float = 20.0):
    L = 2.0 * math.pi
    dx = L / N
    x = np.arange(N, dtype=np.float64) * dx
    delta = width_cells * dx
    return L, 0.5 * (np.tanh((x - L / 4) / delta) - np.tanh((x - 3 * L / 4) / delta))


def c4a_long_explicit(N: int = 1 << 24, n_steps: int = 2000, dtype=np.float32) -> Workload:
    """Config 4a: single long periodic grid, two-sided tanh step, shock width 20 dx."""
    L, u = _tophat(N)
    return _finish(f"C4a-long-euler-N{N}", u[None, :], [1e-4], L, PERIODIC, EULER, 0.4,
                   n_steps, dtype)


def c4b_long_btcs(N: int = 1 << 22, n_steps: int = 200, dtype=np.float64) -> Workload:
    """Config 4b: BTCS on the same profile, one long cyclic tridiagonal system."""
    L, u = _tophat(N)
    return _finish(f"C4b-long-btcs-N{N}", u[None, :], [1e-4], L, PERIODIC, BTCS, 10.0,
                   n_steps, dtype)


def c5_rk4_ensemble(B: int = 65536, N: int = 1024, n_steps: int = 5000,
                    dtype=np.float32, seed: int = SEED_BASE + 5,
                    rows=None) -> Workload:
    """Config 5: Gaussian pulses, periodic, L=1, RK4 at CFL 0.8.

    ``rows``: optional index array -- generate only those trajectories of the
    full B-trajectory ensemble (the draws are always made for all B first, so a
    subset is bit-identical to the same rows of the full workload)."""
    rng = np.random.default_rng(seed)
    L = 1.0
    amp = rng.uniform(0.5, 2.0, B)
    wid = rng.uniform(0.05, 0.2, B) * L
    nu = rng.uniform(5e-3, 5e-2, B)
    x0 = rng.uniform(0.0, L, B)
    if rows is not None:
        rows = np.asarray(rows)
        amp, wid, nu, x0 = amp[rows], wid[rows], nu[rows], x0[rows]
    x = np.arange(N, dtype=np.float64) * (L / N)
    d = np.mod(x[None, :] - x0[:, None] + L / 2, L) - L / 2
    u0 = amp[:, None] * np.exp(-0.5 * (d / wid[:, None]) ** 2)
    return _finish(f"C5-rk4-B{len(amp)}of{B}-N{N}", u0, nu, L, PERIODIC, RK4, 0.8,
                   n_steps, dtype)


def shard_rows(B_global: int, rank: int, world: int) -> np.ndarray:
    """Rows of a B_global-trajectory batch owned by `rank` of `world` (contiguous, balanced to
    within one row).  Trajectories are independent: sharding needs no collective."""
    if not (0 <= rank < world) or B_global < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(B_global, world)
    lo = rank * base + min(rank, rem)
    return np.arange(lo, lo + base + (1 if rank < rem else 0))
