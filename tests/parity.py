"""Helpers of the GPU parity tests: run the CUDA path (through the C ABI binding) and the CPU
oracle on the same seeded inputs and compare element by element.

Tolerances are BASELINE.json's north_star:  max|u_gpu - u_ref| <= 1e-10 max|u0| (fp64),
<= 1e-4 max|u0| (fp32; the oracle runs in fp64 on the fp32-rounded inputs)."""
from __future__ import annotations

import numpy as np

TOL = {np.dtype(np.float64): 1e-10, np.dtype(np.float32): 1e-4}


def rel_err(u_gpu, u_ref, u0):
    """worst over trajectories of max_i |u_gpu - u_ref| / max_i |u0|."""
    u_gpu = np.asarray(u_gpu, dtype=np.float64).reshape(u_ref.shape)
    scale = np.abs(np.asarray(u0, dtype=np.float64)).reshape(u_ref.shape[0], -1).max(axis=1)
    scale = np.where(scale > 0, scale, 1.0)
    err = np.abs(u_gpu - u_ref).reshape(u_ref.shape[0], -1).max(axis=1)
    assert np.all(np.isfinite(u_gpu)), "non-finite values from the CUDA path"
    return float((err / scale).max())


def to_dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle_dt(u0, L, nu, C, bc, dtype):
    """dt from the oracle on the (rounded) inputs, rounded to the workload dtype."""
    import oracle
    return oracle.dt_from_cfl(u0.astype(np.float64), L, nu.astype(np.float64), C, bc).astype(dtype)
