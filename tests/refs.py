"""References the oracle is pinned against (closed forms; no oracle code here)."""
from __future__ import annotations

import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            key, *vals = line.split()
            out[key] = np.array([float(v) for v in vals])
    return out


def read_colehopf_golden():
    rows = []
    with open(os.path.join(GOLDEN, "colehopf_sin.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            nu, xf, u = line.split()
            rows.append((float(nu), float(xf), float(u)))
    return rows


def colehopf_sin(x, t, nu, nodes=80):
    """Exact solution of Eq.1 for u(x,0)=sin x, 2pi-periodic
    (Cole-Hopf), heat-kernel form by Gauss-Hermite quadrature:
    s = sqrt(4 nu t), g(y) = exp(-(1-cos y)/(2 nu)),
    u = (s/t) sum_j w_j eta_j g(x - s eta_j) / sum_j w_j g(x - s eta_j)."""
    eta, w = np.polynomial.hermite.hermgauss(nodes)
    x = np.asarray(x, dtype=np.float64)
    s = np.sqrt(4.0 * nu * t)
    y = x[..., None] - s * eta
    g = np.exp(-(1.0 - np.cos(y)) / (2.0 * nu))
    return (s / t) * (g * (w * eta)).sum(-1) / (g * w).sum(-1)


def amplification(scheme, theta, c, r, sigma=1.0):
    """Exact one-step Fourier amplification factor of the linearised schemes
    (constant advection speed, |a| dt/dx = c, sign sigma; r = nu dt/dx^2):
    z = -c (1 - e^{-i sigma theta}) - 4 r sin^2(theta/2)."""
    z = -c * (1.0 - np.exp(-1j * sigma * theta)) - 4.0 * r * np.sin(theta / 2.0) ** 2
    if scheme == "euler":
        return 1.0 + z
    if scheme == "rk4":
        return 1.0 + z + z ** 2 / 2.0 + z ** 3 / 6.0 + z ** 4 / 24.0
    if scheme == "btcs":
        return 1.0 / (1.0 - z)
    raise ValueError(scheme)
