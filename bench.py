#!/usr/bin/env python
"""bench.py -- grid-point updates/s of the Burgers hot path on B200 (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload c2_f32|c2_f64|c3|c4a|c4b|c5|...] [--no-extras] [--no-cpu] [--peaks]

A "step" is ONE pass of the hot path over one batch of the seeded synthetic workload:
dt_from_cfl (CFL reduction) followed by the time-stepping call (all n_steps of the config).
Headline workload at N=1: BASELINE.json configs[1] (C2: B=1024 Dirichlet trajectories, N=4096,
10,000 forward-Euler steps, fp32).  `value` = grid-point updates/s (B*N*n_steps per step) with
the inputs resident in HBM; `e2e` = the same through the host-buffer C-ABI calls (H2D + D2H inside
the timed region); `roofline` = the dominant kernel against its bound (DESIGN.md 6 / 8);
`cpu_baseline` = the fp64 CPU oracle timed on this box's cores on a bounded sample (all cores, and
one thread); `pipe_peaks` = the FP-pipe micro-benchmarks measured in this run; `schemes` = every
other config with the same set of numbers (median of >= 5 repetitions).

--gpus N > 1: launched under torchrun (RANK / WORLD_SIZE set) every rank runs its own shard of an
N-times larger batch (trajectories are independent: no collective on the data path; weak scaling);
launched plainly, bench.py re-executes itself under torch.distributed.run with N ranks.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SM_COUNT = 148
FP32_LANES, FP64_LANES = 128, 64
# Algorithmic instruction counts per update (DESIGN.md 6.1 / 6.3):
#   fp32 Euler: 7 issue slots (FADD, FADD, FSETP, FSEL, FFMA, FFMA + FADD of the compensated sum)
#   fp32 RK4:   4 stages x 8 (FADD, FADD, FSETP, FSEL, FMUL, FFMA + 2 FFMA for accumulator / next stage)
#   fp64 Euler: 5 FP64-pipe instructions (DADD, DADD, DMUL, DFMA, DFMA; the select runs on the integer pipe)
#   fp64 BTCS, partition + PCR solvers: per row 19 (assembly 5, forward elimination 6 + 3 for the reciprocal,
#     backward recurrence 3, back substitution 2) + per thread (23 + 12 per PCR level) / P rows:
#     HYBRID P = 16, 4 levels: 19 + 71/16 = 23.4;  LONG P = 16, <= 3 levels: 19 + 59/16 = 22.7  -> 23
I_EULER_F32, I_EULER_F64, I_RK4_F32, I_BTCS_HYBRID, I_BTCS_LONG = 7, 5, 32, 23, 23
# Tests drive the multi-rank logic of run_ours on CPU by replacing these two (tests/test_sharding_gloo.py):
BACKEND = "nccl"            # torch.distributed backend of the timing barrier / max-over-ranks
RUNNER = None               # class with GpuRunner's interface; None -> GpuRunner
HOT = ("c2_f32", "c2_f64", "c3", "c4a", "c4b", "c5")
NEXT = ("c3_newton", "c3_cn", "c2_traj", "c3_gs", "c2_adjoint")
MORE = ("c5_adjoint", "c3_btcs_adjoint", "c3_newton_adjoint")        # --workload only (not in the default table)
WORKLOADS = HOT + NEXT


def sig(x, n=5):
    """Round to n significant digits (keeps the one JSON line short enough for the driver's tail)."""
    if x is None or isinstance(x, (int, str, bool)):
        return x
    x = float(x)
    if x == 0.0 or not np.isfinite(x):
        return x
    return float(f"{x:.{n}g}")


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm_gbs": float(p["hbm_gbs"]), "sm_max_mhz": float(p.get("sm_max_mhz", 1965.0)),
                "source": "MEASURED_PEAKS.json"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback of B200_PROFILING.md"}


def ncu_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of each time-stepping kernel, from the
    `ncu --set full` captures summarised under profiles/ (the file names the commit they were taken at)."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    out = {"commit": None, "bytes_per_launch": {}}
    try:
        for line in open(path):
            line = line.strip()
            if line.startswith("# commit:"):
                out["commit"] = line.split(":", 1)[1].strip()
            elif line and not line.startswith("#") and not line.startswith("workload"):
                k, v = line.split(",")
                out["bytes_per_launch"][k] = float(v)
    except (OSError, ValueError):
        pass
    return out


# ------------------------------------------------------------------------------- workloads
def make_workload(name, rank=0, world=1, reduced=False):
    """(workload, spec) -- spec: op, scheme, bound, algorithmic instr/update, pipe lanes."""
    from paper_2601_12204_b200 import workloads as W
    if name in ("c2_f32", "c2_f64"):
        dtype = np.float32 if name == "c2_f32" else np.float64
        Bg = 1024 * world
        w = W.c2_dirichlet_batch(B=Bg, dtype=dtype, rows=W.shard_rows(Bg, rank, world),
                                 n_steps=1000 if reduced else 10000)
        return w, dict(op="explicit", scheme=0, bound="alu", instr=I_EULER_F32 if dtype == np.float32 else I_EULER_F64,
                       lanes=FP32_LANES if dtype == np.float32 else FP64_LANES)
    if name == "c3":
        Bg = 4096 * world
        w = W.c3_periodic_btcs(B=Bg, rows=W.shard_rows(Bg, rank, world), n_steps=100 if reduced else 1000)
        return w, dict(op="btcs", scheme=None, bound="alu", instr=I_BTCS_HYBRID, lanes=FP64_LANES)
    if name == "c3_gs":          # C3's trajectories, CFL-sized dt (C = 0.4, the regime of the paper's
        Bg = 4096 * world        #   "5-7 iterations"), BTCS with Gauss-Seidel sweeps to max residual < 1e-6, 100 steps
        w = W.c3_periodic_btcs(B=Bg, rows=W.shard_rows(Bg, rank, world), n_steps=10 if reduced else 100)
        w.cfl = 0.4
        return w, dict(op="gs", scheme=None, bound="alu", instr=None, lanes=FP64_LANES, tol=1e-6, max_iter=1000)
    if name == "c2_adjoint":     # SURVEY 8(f) NEXT-4c: reverse-mode derivative of 1000 Euler steps of 256 C2 trajectories
        Bg = 256 * world
        w = W.c2_dirichlet_batch(B=Bg, dtype=np.float32, rows=W.shard_rows(Bg, rank, world),
                                 n_steps=100 if reduced else 1000)
        return w, dict(op="adjoint", scheme=0, bound="hbm", instr=None, lanes=FP32_LANES)
    if name == "c5_adjoint":     # adjoint of 100 RK4 steps of 4096 of C5's pulses (D14; streaming backward sweep)
        Bg = 4096 * world
        w = W.c5_rk4_ensemble(B=65536 * world, rows=np.arange(0, 65536 * world, 16)[W.shard_rows(Bg, rank, world)],
                              n_steps=10 if reduced else 100)
        return w, dict(op="adjoint", scheme=1, bound="hbm", instr=None, lanes=FP32_LANES)
    if name in ("c3_btcs_adjoint", "c3_newton_adjoint"):   # reverse mode of ALL of C3 (D15 / D16): 4096 trajectories, 1000
        Bg = 4096 * world                                  # implicit steps; 67 GB of states -> checkpointed (32-step segments)
        w = W.c3_periodic_btcs(B=Bg, rows=W.shard_rows(Bg, rank, world), n_steps=100 if reduced else 1000)
        if name == "c3_newton_adjoint":
            w.cfl = 4.0
        return w, dict(op="adjoint", scheme=2 if name == "c3_btcs_adjoint" else 3, bound="hbm", instr=None, lanes=FP64_LANES)
    if name == "c2_traj":        # SURVEY 8(f) NEXT-4b: C2 fp32 with a snapshot of all trajectories every 50 steps
        Bg = 1024 * world
        w = W.c2_dirichlet_batch(B=Bg, dtype=np.float32, rows=W.shard_rows(Bg, rank, world),
                                 n_steps=1000 if reduced else 10000)
        return w, dict(op="explicit", scheme=0, bound="alu", instr=I_EULER_F32, lanes=FP32_LANES, snap_every=50)
    if name in ("c3_newton", "c3_cn"):   # SURVEY 8(f) NEXT-1 / NEXT-2 on C3's inputs: Newton solve of the fully implicit
        Bg = 4096 * world                #   (theta = 1) / Crank-Nicolson (theta = 1/2) central scheme, tol 1e-6
        w = W.c3_periodic_btcs(B=Bg, rows=W.shard_rows(Bg, rank, world), n_steps=100 if reduced else 1000)
        return w, dict(op="newton", scheme=None, bound="alu", instr=None, lanes=FP64_LANES, tol=1e-6, max_iter=50,
                       theta=1.0 if name == "c3_newton" else 0.5)
    if name == "c4a":
        w = W.c4a_long_explicit(n_steps=200 if reduced else 2000)
        return w, dict(op="explicit", scheme=0, bound="alu", instr=I_EULER_F32, lanes=FP32_LANES)
    if name == "c4b":            # one HBM-accounting round trip per step (state stays in L2): north_star's bound is HBM
        w = W.c4b_long_btcs(n_steps=20 if reduced else 200)
        return w, dict(op="btcs", scheme=None, bound="hbm", instr=I_BTCS_LONG, lanes=FP64_LANES)
    if name == "c5":
        Bg = 65536 * world
        w = W.c5_rk4_ensemble(B=Bg, rows=W.shard_rows(Bg, rank, world), n_steps=500 if reduced else 5000)
        return w, dict(op="explicit", scheme=1, bound="alu", instr=I_RK4_F32, lanes=FP32_LANES)
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled for the whole run; `window(t0, t1)` reports one region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self):
        if self.proc is not None:
            time.sleep(0.1)
            self.proc.terminate()

    def window(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)                       # let the sample that covers t1 arrive
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in list(self.rows):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                clk, smax = float(f[0]), float(f[1])
            except ValueError:
                continue
            if t0 - 0.03 <= ts <= t1 + 0.06:
                sm.append(clk)
                for n, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": smax,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return model


def metric_name(spec):
    base = "grid-point updates/s (B*N*steps/s), "
    if spec["op"] == "explicit":
        return base + ("forward Euler upwind/central" if spec["scheme"] == 0 else "RK4")
    return base + {"btcs": "BTCS", "newton": "Newton BTCS (central convection, theta-scheme)",
                   "gs": "Gauss-Seidel BTCS",
                   "adjoint": ("adjoint of forward Euler", "adjoint of RK4", "adjoint of BTCS",
                               "reverse mode of Newton BTCS")[spec["scheme"] or 0]}[spec["op"]]


# ------------------------------------------------------------------------------- oracle leg
def oracle_sample_run(w, spec, target_s=12.0, threads=None):
    """Times the CPU oracle (as it stands) on a bounded sample of workload `w`: whole trajectories
    (all n_steps) for batched configs, a shortened step count for the single long grids.
    Returns (updates, seconds, threads, description)."""
    import oracle
    threads = threads or oracle.default_threads()
    u0 = w.u0.astype(np.float64)
    nu = w.nu.astype(np.float64)
    dt = oracle.dt_from_cfl(u0, w.L, nu, w.cfl, w.bc).astype(w.dtype).astype(np.float64)

    def run(rows, n):
        t0 = time.perf_counter()
        if spec["op"] == "btcs":
            oracle.btcs(u0[rows], w.L, nu[rows], dt[rows], n, w.bc, threads=threads)
        elif spec["op"] == "gs":
            oracle.btcs_gs(u0[rows], w.L, nu[rows], dt[rows], n, w.bc, tol=spec["tol"], max_iter=spec["max_iter"],
                           threads=threads)
        elif spec["op"] == "adjoint":
            lam = np.random.default_rng(1220404).standard_normal(u0[rows].shape)
            if spec["scheme"] == 2:
                oracle.btcs_adjoint(u0[rows], lam, w.L, nu[rows], dt[rows], n, w.bc, threads=threads)
            elif spec["scheme"] == 3:
                oracle.newton_adjoint(u0[rows], lam, w.L, nu[rows], dt[rows], n, w.bc, threads=threads)
            else:
                oracle.explicit_adjoint(u0[rows], lam, w.L, nu[rows], dt[rows], n, w.bc, threads=threads, scheme=spec["scheme"])
        elif spec["op"] == "newton":
            oracle.newton_btcs(u0[rows], w.L, nu[rows], dt[rows], n, w.bc, tol=spec["tol"],
                               max_iter=spec["max_iter"], threads=threads, theta=spec["theta"])
        elif w.B == 1:
            oracle.explicit_long(u0[0], w.L, nu[0], dt[0], n, w.bc, threads=threads)
        else:
            oracle.explicit(u0[rows], w.L, nu[rows], dt[rows], n, w.bc, spec["scheme"], threads=threads)
        return time.perf_counter() - t0

    if w.B == 1:      # long grid: calibrate on 1 step, then as many steps as fit the budget
        rows = np.arange(1)
        t = run(rows, 1)
        n = int(max(1, min(w.n_steps, target_s / max(t, 1e-9))))
        sec = run(rows, n)
        return w.N * n, sec, threads, f"{n} of {w.n_steps} steps of the full N={w.N} grid"
    nb = min(w.B, threads)
    ncal = max(1, min(w.n_steps, 100))
    t = run(np.arange(nb), ncal) / (nb * ncal)                 # seconds per trajectory-step (all threads busy)
    want = int(target_s / max(t * w.n_steps, 1e-12))
    nb = int(max(threads, min(w.B, want // threads * threads)))
    nb = min(nb, w.B)
    sec = run(np.arange(nb), w.n_steps)
    return nb * w.N * w.n_steps, sec, threads, f"first {nb} of {w.B} trajectories, all {w.n_steps} steps"


def cpu_baseline(w, spec, all_core_s, single_s):
    """two figures per config -- all host cores, and a single thread."""
    upd, sec, threads, desc = oracle_sample_run(w, spec, target_s=all_core_s)
    out = {"value": sig(upd / sec), "unit": "updates/s", "cores": threads, "kind": "oracle", "sample": desc,
           "seconds": sig(sec, 3)}
    if single_s > 0:
        upd1, sec1, _, desc1 = oracle_sample_run(w, spec, target_s=single_s, threads=1)
        out["single_thread"] = {"value": sig(upd1 / sec1), "cores": 1, "sample": desc1, "seconds": sig(sec1, 3)}
    return out


# ------------------------------------------------------------------------------- GPU legs
class GpuRunner:
    def __init__(self, w, spec, device):
        import torch
        from paper_2601_12204_b200 import binding as B
        self.torch, self.B, self.w, self.spec = torch, B, w, spec
        self.dev = device
        self.u0 = torch.from_numpy(w.u0).to(device)
        self.nu = torch.from_numpy(w.nu).to(device)
        self.u = torch.empty_like(self.u0)
        self.dt = torch.empty_like(self.nu)
        is64 = w.dtype == np.float64
        if spec["op"] == "explicit":
            self.plan = B.plan_query(B.OP_EXPLICIT, is64, w.B, w.N, w.bc, spec["scheme"])
            need = B.workspace_bytes(B.OP_EXPLICIT, is64, w.B, w.N, w.bc, spec["scheme"])
            self.launches = B.launch_count(B.OP_EXPLICIT, is64, w.B, w.N, w.bc, spec["scheme"], n_steps=w.n_steps)
        elif spec["op"] == "adjoint":
            self.plan = 0
            if spec["scheme"] >= 2:      # implicit schemes: forward sweep (one launch when the system fits one CTA: the
                #                          kernel writes the states; else one per step) + one backward launch
                q = B.raw().burgers_btcs_adjoint_workspace_bytes if spec["scheme"] == 2 else B.raw().burgers_newton_adjoint_workspace_bytes
                need = int(q(int(is64), w.B, w.N, w.bc, w.n_steps))
                fits = B.plan_query(B.OP_BTCS if spec["scheme"] == 2 else B.OP_NEWTON, is64, w.B, w.N, w.bc) == B.PLAN_HYBRID
                one = w.n_steps * w.B * w.N * w.u0.dtype.itemsize <= (8 << 30)       # one segment (binding: segment = 0)
                m = w.n_steps if one else math.ceil(math.sqrt(w.n_steps))
                K = -(-w.n_steps // m)
                # per segment: forward (one launch if the kernel writes the states, else one per step) + backward
                self.launches = (1 if K > 1 and fits else 0) + K * ((1 if fits else m) + 1)
            else:
                need = int(B.raw().burgers_adjoint_scheme_workspace_bytes(int(is64), w.B, w.N, w.bc, spec["scheme"], w.n_steps, 0))
                # Euler: forward trajectory kernel + resident backward kernel; RK4: forward + 7 launches per step
                self.launches = 2 if spec["scheme"] == 0 else 1 + 7 * w.n_steps
            self.lam0 = torch.randn(self.u0.shape, dtype=self.u0.dtype, device=device,
                                    generator=torch.Generator(device=device).manual_seed(1220404))
        elif spec["op"] == "gs":
            self.plan = B.plan_query(B.OP_GS, is64, w.B, w.N, w.bc)
            need = B.workspace_bytes(B.OP_GS, is64, w.B, w.N, w.bc)
            self.launches = B.launch_count(B.OP_GS, is64, w.B, w.N, w.bc, n_steps=w.n_steps)
            self.iters = torch.zeros(w.B, dtype=torch.int64, device=device)
        elif spec["op"] == "newton":
            self.plan = B.plan_query(B.OP_NEWTON, is64, w.B, w.N, w.bc)
            need = B.workspace_bytes(B.OP_NEWTON, is64, w.B, w.N, w.bc)
            self.launches = B.launch_count(B.OP_NEWTON, is64, w.B, w.N, w.bc, n_steps=w.n_steps)
            self.iters = torch.zeros(w.B, dtype=torch.int64, device=device)
        else:
            self.plan = B.plan_query(B.OP_BTCS, is64, w.B, w.N, w.bc)
            need = B.workspace_bytes(B.OP_BTCS, is64, w.B, w.N, w.bc)
            self.launches = B.launch_count(B.OP_BTCS, is64, w.B, w.N, w.bc, n_steps=w.n_steps)
        self.op_launches = int(self.launches)
        self.launches += B.launch_count(B.OP_CFL, is64, w.B, w.N, w.bc)
        self.ws = torch.empty(need, dtype=torch.uint8, device=device) if need else None
        self.snaps = None
        if spec.get("snap_every"):
            self.snaps = torch.empty((w.n_steps // spec["snap_every"], w.B, w.N), dtype=self.u0.dtype, device=device)
        self.flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)   # > 126 MB L2

    def reset(self):
        self.u.copy_(self.lam0 if self.spec["op"] == "adjoint" else self.u0)     # adjoint: u holds lambda
        self.flush.zero_()          # L2 flush between timed iterations (outside the event pairs)

    def cfl(self):
        src = self.u0 if self.spec["op"] == "adjoint" else self.u
        self.B.dt_from_cfl(src, self.w.L, self.nu, self.w.cfl, self.w.bc, out=self.dt)

    def op(self):
        w, B = self.w, self.B
        if self.spec["op"] == "explicit" and self.snaps is not None:
            B.burgers_explicit_traj(self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, self.spec["scheme"],
                                    self.spec["snap_every"], snaps=self.snaps, ws=self.ws)
        elif self.spec["op"] == "explicit":
            B.burgers_explicit(self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, self.spec["scheme"], ws=self.ws)
        elif self.spec["op"] == "adjoint" and self.spec["scheme"] == 2:
            B.burgers_btcs_adjoint(self.u0, self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, ws=self.ws)
        elif self.spec["op"] == "adjoint" and self.spec["scheme"] == 3:
            B.burgers_newton_adjoint(self.u0, self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, ws=self.ws)
        elif self.spec["op"] == "adjoint":
            B.burgers_explicit_adjoint(self.u0, self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, ws=self.ws,
                                       scheme=self.spec["scheme"])
        elif self.spec["op"] == "gs":
            B.burgers_btcs_gs(self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, tol=self.spec["tol"],
                              max_iter=self.spec["max_iter"], iters_out=self.iters, ws=self.ws)
        elif self.spec["op"] == "newton":
            B.burgers_newton(self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, tol=self.spec["tol"],
                             max_iter=self.spec["max_iter"], iters_out=self.iters, ws=self.ws, theta=self.spec["theta"])
        else:
            B.burgers_btcs(self.u, w.L, self.nu, self.dt, w.n_steps, w.bc, ws=self.ws)

    def timed(self, steps, warmup):
        """Returns (list of step ms, list of op-only ms) from CUDA events on the launching stream."""
        torch = self.torch
        for _ in range(warmup):
            self.reset(); self.cfl(); self.op()
        torch.cuda.synchronize()
        step_ms, op_ms = [], []
        for _ in range(steps):
            self.reset()
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            e0.record(); self.cfl(); e1.record(); self.op(); e2.record()
            e2.synchronize()
            step_ms.append(e0.elapsed_time(e2)); op_ms.append(e1.elapsed_time(e2))
        return step_ms, op_ms

    def e2e(self, steps, warmup):
        """Same step through the host-buffer C-ABI calls: pinned host arrays in, result read back."""
        torch, B, w = self.torch, self.B, self.w
        hu0 = torch.from_numpy(w.u0).pin_memory()
        hnu = torch.from_numpy(w.nu).pin_memory()
        hu = torch.empty_like(hu0).pin_memory()
        u_np, nu_np = hu.numpy(), hnu.numpy()
        ms = []
        for i in range(warmup + steps):
            hu.copy_(hu0)
            self.flush.zero_(); torch.cuda.synchronize()
            t0 = time.perf_counter()
            if self.spec["op"] in ("gs", "adjoint"):   # no _host entry point: pinned host -> device, device calls, device -> pinned host
                du, dnu = hu.to(self.dev, non_blocking=True), hnu.to(self.dev, non_blocking=True)
                ddt = B.dt_from_cfl(du, w.L, dnu, w.cfl, w.bc)
                if self.spec["op"] == "gs":
                    B.burgers_btcs_gs(du, w.L, dnu, ddt, w.n_steps, w.bc, tol=self.spec["tol"],
                                      max_iter=self.spec["max_iter"], ws=self.ws)
                else:                                  # (the seed lambda is already on the device)
                    dl = self.lam0.clone()
                    if self.spec["scheme"] == 2:
                        B.burgers_btcs_adjoint(du, dl, w.L, dnu, ddt, w.n_steps, w.bc, ws=self.ws)
                    elif self.spec["scheme"] == 3:
                        B.burgers_newton_adjoint(du, dl, w.L, dnu, ddt, w.n_steps, w.bc, ws=self.ws)
                    else:
                        B.burgers_explicit_adjoint(du, dl, w.L, dnu, ddt, w.n_steps, w.bc, ws=self.ws, scheme=self.spec["scheme"])
                    du = dl
                hu.copy_(du); torch.cuda.synchronize()
            elif self.spec["op"] == "newton":
                dt = B.dt_from_cfl_host(u_np, w.L, nu_np, w.cfl, w.bc)
                B.burgers_newton_host(u_np, w.L, nu_np, dt, w.n_steps, w.bc, tol=self.spec["tol"],
                                      max_iter=self.spec["max_iter"], theta=self.spec["theta"])
            else:                                      # the hot path in one host call: one upload, CFL + stepping
                B.burgers_solve_host(u_np, w.L, nu_np, w.cfl, w.n_steps, w.bc,
                                     op=B.OP_EXPLICIT if self.spec["op"] == "explicit" else B.OP_BTCS,
                                     scheme=self.spec["scheme"] or 0)
            t1 = time.perf_counter()
            if i >= warmup:
                ms.append((t1 - t0) * 1e3)
        esz = w.u0.dtype.itemsize
        if self.spec["op"] == "newton":
            h2d = 2 * w.B * w.N * esz + 3 * w.B * esz  # cfl: u, nu; step: u, nu, dt
            d2h = w.B * w.N * esz + w.B * esz          # cfl: dt; step: u
        else:
            h2d = w.B * w.N * esz + w.B * esz          # u, nu
            d2h = w.B * w.N * esz                      # u
        return ms, h2d, d2h


def measure_pipe_peaks(device, pk):
    """The FP-pipe micro-benchmarks of burgers_pipe_peak, timed with CUDA events (best of 3 launches of ~2 ms)."""
    import torch
    from paper_2601_12204_b200 import binding as B
    sink = torch.zeros(2, dtype=torch.float64, device=device)
    out = {}
    for k, name in enumerate(B.PEAK_KINDS):
        nominal = SM_COUNT * (FP32_LANES if k < 3 else FP64_LANES) * pk["sm_max_mhz"] * 1e6
        iters = 2000 if k < 3 else 1000          # (kind 6, DFMA + select mix: fraction of the FP64 rate left to the DFMAs)
        B.pipe_peak(k, 50, sink)
        torch.cuda.synchronize()
        best = 0.0
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); n = B.pipe_peak(k, iters, sink); e1.record(); e1.synchronize()
            best = max(best, n / (e0.elapsed_time(e1) * 1e-3))
        out[name] = {"ginst_s": sig(best / 1e9), "frac_of_nominal": sig(best / nominal, 4)}
    return out


def roofline(name, spec, w, op_ms, pk, traffic, launches, pipe=None, verbose=True):
    """Dominant kernel = the time-stepping kernel(s) of the op call.  `achieved` = algorithmic work per launch /
    average launch duration (CUDA events around the op call: the kernels run back to back on one stream)."""
    sec = statistics.median(op_ms) * 1e-3
    ups = w.updates / sec
    esz = w.u0.dtype.itemsize
    hbm_acc = ups * 2 * esz / (pk["hbm_gbs"] * 1e9)
    tr = traffic.get("bytes_per_launch", {}).get(name)
    out = {"bound": spec["bound"], "kernel_launches": int(launches),
           "avg_launch_us": sig(sec * 1e6 / max(1, launches)),
           "traffic": tr, "traffic_source": f"ncu dram rd+wr per launch, profiles/ncu_traffic.csv @ {str(traffic.get('commit'))[:7]}",
           "hbm_accounting_frac": sig(hbm_acc, 4)}
    if not verbose:            # per-scheme entries: the sources are those of the headline's roofline
        out.pop("traffic_source")
    if spec["bound"] == "hbm":
        if spec["op"] == "adjoint":          # every stored forward state is written once and read once
            byt = 2 * (w.n_steps - 1) * w.B * w.N * esz
            note = "forward states written once + read once / time of both sweeps"
        else:                                # one round trip of the state per step
            byt = 2 * esz * w.updates
            note = f"{2 * esz} B per update (read u^n, write u^n+1) x updates / kernel time"
        ach = byt / sec / 1e9
        out.update({"achieved": sig(ach), "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": sig(ach / pk["hbm_gbs"], 4),
                    "peak_source": pk["source"] + " (measured copy bandwidth)", "note": note})
        if not verbose:
            out.pop("note"); out["peak_source"] = "measured copy"
        if spec["instr"]:
            out["alu_frac"] = sig(ups * spec["instr"] / (SM_COUNT * spec["lanes"] * pk["sm_max_mhz"] * 1e6), 4)
        return out
    peak = SM_COUNT * spec["lanes"] * pk["sm_max_mhz"] * 1e6 / 1e9        # G lane-instr/s
    pipe_name = "fp64" if spec["lanes"] == FP64_LANES else "fp32"
    src = f"nominal issue rate {SM_COUNT} SMs x {spec['lanes']} lanes x {pk['sm_max_mhz']:.0f} MHz"
    if pipe:
        chain = pipe["dfma_chain" if pipe_name == "fp64" else "ffma_chain"]["frac_of_nominal"]
        three = pipe["dfma_3reg" if pipe_name == "fp64" else "ffma_3reg"]["frac_of_nominal"]
        src += f"; measured in this run: FMA chain {chain} of it, FMA with 3 register operands {three}"
    if not verbose:
        src = f"nominal {pipe_name} issue rate"
    if spec["instr"] is None:                # 8(f) rows without an instruction-count model: time and accounting only
        out.update({"achieved": None, "peak": sig(peak), "unit": "Ginst/s", "frac": None, "peak_source": src})
        return out
    ach = ups * spec["instr"] / 1e9
    out.update({"achieved": sig(ach), "peak": sig(peak), "unit": "Ginst/s", "frac": sig(ach / peak, 4),
                "peak_source": src, "instr_per_update": spec["instr"]})
    if verbose:
        out["note"] = f"{spec['instr']} algorithmic {pipe_name}-pipe instr/update x updates / kernel time"
    return out


def measure(name, device, args, pk, traffic, sampler, pipe, steps, warmup, rank=0, world=1, cpu=(0.0, 0.0), e2e_steps=0):
    """Everything bench.py reports about one config.  Returns (record, step_ms list, workload, runner info)."""
    import torch
    w, spec = make_workload(name, rank, world, args.reduced)
    r = GpuRunner(w, spec, device)
    if spec["op"] == "btcs" and w.B == 1 and r.plan == r.B.PLAN_THOMAS:
        raise RuntimeError("single long system would run on one thread (no LONG plan for this N)")
    r.timed(0, warmup)
    t0 = time.time()
    step_ms, op_ms = r.timed(steps, 0)
    t1 = time.time()
    ck = sampler.window(t0, t1)
    rec = {"dtype": "f32" if w.dtype == np.float32 else "f64", "B": w.B, "N": w.N, "n_steps": w.n_steps,
           "plan": int(r.plan), "reps": steps, "ms_median": sig(statistics.median(step_ms)),
           "ms_min_max": [sig(min(step_ms)), sig(max(step_ms))],
           "updates_per_s": sig(w.updates / (statistics.median(step_ms) * 1e-3)),
           "gpu_launches_per_step": int(r.launches),
           "roofline": roofline(name, spec, w, op_ms, pk, traffic, r.op_launches, pipe, verbose=False),
           "clocks": {"sm_mhz": ck.get("sm_mhz"), "reasons": ck.get("reasons")}}
    if not rec["clocks"]["reasons"]:
        rec["clocks"] = {"sm_mhz": ck.get("sm_mhz")}            # (no throttle reason in this config's window)
    cfl_ms = max(1e-6, statistics.median(step_ms) - statistics.median(op_ms))
    rec["cfl_ms"] = sig(cfl_ms, 3)
    if r.snaps is not None:
        rec["snapshots"] = int(r.snaps.shape[0]); rec["snapshot_bytes"] = int(r.snaps.numel() * r.snaps.element_size())
    if spec["op"] == "btcs" and r.plan == r.B.PLAN_LONG and r.op_launches > 2:
        rec["steps_per_launch"] = sig(w.n_steps / (r.op_launches - 2), 3)       # LONG: S steps per HBM round trip
    if spec["op"] == "gs":
        sw = float(r.iters.double().mean().item()) / w.n_steps
        rec["gs_sweeps_per_step"] = sig(sw, 4); rec["tol"] = spec["tol"]
        # FP64 instructions per update, counted from btcs_gs.cu (CTA plan, 16 rows per thread) for the measured sweep count:
        # per step rows + reciprocal + scaled coefficients 12; per residual pass (one more than sweeps) 6 + the scan of
        # the thread maps 14/16; per sweep the second pass 1
        spec = dict(spec, instr=round(12 + (sw + 1) * (6 + 14.0 / 16) + sw, 1))
        rec["roofline"] = roofline(name, spec, w, op_ms, pk, traffic, r.op_launches, pipe, verbose=False)
    if spec["op"] == "newton":
        its = float(r.iters.double().mean().item()) / w.n_steps
        rec["newton_iterations_per_step"] = sig(its, 4)
        rec["tol"] = spec["tol"]; rec["theta"] = spec["theta"]
        # FP64 instructions per update, counted from newton.cu for the measured iteration count: one
        # residual pass per iteration + one final (10 per row), per iteration Jacobian rows 4 + elimination 9 +
        # backward recurrence 3 + back substitution 2 + update 1, + the interface solve (23 + 12 x 4 levels) / 16 rows
        spec = dict(spec, instr=round(its * (10 + 19 + 71.0 / 16) + 10, 1))
        rec["roofline"] = roofline(name, spec, w, op_ms, pk, traffic, r.op_launches, pipe, verbose=False)
    if e2e_steps:
        e_ms, h2d, d2h = r.e2e(e2e_steps, 1)
        rec["e2e"] = {"value": sig(w.updates * world / (statistics.median(e_ms) * 1e-3)),
                      "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                      "ms_per_step": sig(statistics.median(e_ms))}
    rec["roofline"].pop("peak_source", None)                      # (as in the headline's roofline)
    rec["roofline"].pop("unit", None)                             # (Ginst/s for "alu", GB/s for "hbm")
    rec.pop("cfl_ms", None)
    rec["roofline"].pop("kernel_launches", None)                  # (= gpu_launches_per_step minus the CFL launches)
    if rec["roofline"].get("bound") == "hbm":
        rec["roofline"].pop("hbm_accounting_frac", None)          # (= frac)
    rec["roofline"] = {k: v for k, v in rec["roofline"].items() if v is not None}
    info = {"w": w, "spec": spec, "launches": int(r.launches), "plan": int(r.plan), "step_ms": step_ms}
    del r
    torch.cuda.empty_cache()
    if cpu[0] > 0:
        c = cpu_baseline(w, spec, cpu[0], cpu[1])
        rec["cpu_baseline"] = {"value": c["value"], "cores": c["cores"],
                               "sample": c["sample"].split(",")[0].replace("trajectories", "traj").replace(" of the full", ""),
                               "single_thread": c.get("single_thread", {}).get("value")}
    return rec, info


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", 0)); world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if world != max(1, args.gpus):
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with --nproc-per-node {args.gpus}")
    on_gpu = BACKEND == "nccl"
    if on_gpu:
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback; see --impl reference)")
        torch.cuda.set_device(local)
        device = torch.device("cuda", local)
    else:
        device = torch.device("cpu")
    if world > 1:
        dist.init_process_group(BACKEND, **({"device_id": device} if on_gpu else {}))
    if on_gpu:
        from paper_2601_12204_b200 import build as _b
        if rank == 0:
            _b.build()
    if world > 1:
        dist.barrier()
    pk = peaks()
    traffic = ncu_traffic()
    Runner = RUNNER or GpuRunner

    def barrier():
        if world > 1:
            dist.barrier()
        if on_gpu:
            torch.cuda.synchronize()

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    sampler = ClockSampler(local)
    sampler.start()
    pipe = measure_pipe_peaks(device, pk) if (rank == 0 and on_gpu) else None
    barrier()
    # headline: W warm-ups, then EXACTLY K timed steps between two barriers; mean over the K steps, max over ranks
    w, spec = make_workload(args.workload, rank, world, args.reduced)
    r = Runner(w, spec, device)
    r.timed(0, args.warmup)
    barrier()
    t0 = time.time()
    step_ms, op_ms = r.timed(args.steps, 0)
    barrier()
    t1 = time.time()
    clocks = sampler.window(t0, t1)
    ms = max_over_ranks(statistics.mean(step_ms))
    value = w.updates * world / (ms * 1e-3)
    out = {
        "metric": metric_name(spec),
        "value": sig(value, 7), "unit": "updates/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": sig(ms, 6), "ms_median": sig(statistics.median(step_ms), 6), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if w.dtype == np.float32 else "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: {w.name}, {w.n_steps} time steps per bench step, "
                               f"bc={'periodic' if w.bc == 0 else 'dirichlet'}, CFL {w.cfl}",
                   "B_per_gpu": w.B, "N": w.N, "n_steps": w.n_steps, "plan": int(r.plan),
                   "parallelism": f"batch-sharded x{world} (no collective)" if world > 1 else "single GPU",
                   "l2": "flushed between timed steps (512 MiB memset)",
                   "input_sha256": w.sha256()[:16]},
        "gpu_launches": int(r.launches * args.steps),
        "clocks": clocks,
    }
    if spec["op"] == "gs" and hasattr(r, "iters"):              # instruction count for the measured sweep count (see measure())
        sw = float(r.iters.double().mean().item()) / w.n_steps
        spec = dict(spec, instr=round(12 + (sw + 1) * (6 + 14.0 / 16) + sw, 1))
        out["gs_sweeps_per_step"] = sig(sw, 4)
    if spec["op"] == "newton" and hasattr(r, "iters"):          # instruction count for the measured iteration count (see measure())
        its = float(r.iters.double().mean().item()) / w.n_steps
        spec = dict(spec, instr=round(its * (10 + 19 + 71.0 / 16) + 10, 1))
        out["newton_iterations_per_step"] = sig(its, 4)
    if rank == 0:
        out["roofline"] = roofline(args.workload, spec, w, op_ms, pk, traffic, r.op_launches, pipe)
        if spec["op"] == "btcs" and r.plan == r.B.PLAN_LONG and r.op_launches > 2:
            out["roofline"]["steps_per_launch"] = sig(w.n_steps / (r.op_launches - 2), 3)
        e_ms, h2d, d2h = r.e2e(max(1, min(args.steps, 5)), 1)
        out["e2e"] = {"value": sig(w.updates * world / (statistics.median(e_ms) * 1e-3), 6), "unit": "updates/s",
                      "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                      "ms_per_step": sig(statistics.median(e_ms)),
                      "note": "burgers_solve_host_*: pinned host buffers, upload + CFL + stepping + download; rank 0"}
        cfl_ms = max(1e-6, statistics.median(step_ms) - statistics.median(op_ms))
        out["cfl"] = {"ms": sig(cfl_ms, 3), "hbm_frac": sig(w.B * w.N * w.u0.dtype.itemsize / (cfl_ms * 1e-3) / 1e9 / pk["hbm_gbs"], 3)}
        out["pipe_peaks"] = pipe
    del r
    if on_gpu:
        torch.cuda.empty_cache()
    if world == 1 and not args.no_extras:
        extras = {}
        for name in WORKLOADS:
            if name == args.workload:
                continue
            hot = name in HOT
            try:
                rec, _ = measure(name, device, args, pk, traffic, sampler, pipe, steps=5, warmup=1,
                                 cpu=(0.0, 0.0) if args.no_cpu else ((4.0, 2.5) if hot else (2.0, 1.5)),
                                 e2e_steps=3 if hot else 0)
                extras[name] = rec
            except Exception as ex:  # a missing plan must not hide the headline number
                extras[name] = {"error": f"{type(ex).__name__}: {ex}"}
        out["schemes"] = extras
        # the fractions again inside a key the driver keeps whole: [ms, bound, frac]
        out["roofline"]["other_configs"] = {k: [v.get("ms_median"), v["roofline"]["bound"], v["roofline"].get("frac")]
                                            for k, v in extras.items() if "roofline" in v}
    if rank == 0 and world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(w, spec, 12.0, 4.0)
        out["cpu_baseline"]["cpu"] = cpu_info()
    sampler.stop()
    if rank == 0:
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_reference(args):
    """The reference arm of this tier is the CPU oracle, as it stands, on the host cores."""
    if int(os.environ.get("RANK", 0)) != 0:
        return
    import oracle
    oracle.build()
    w, spec = make_workload(args.workload, 0, 1, args.reduced)
    per = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    vals, desc, threads = [], "", 1
    for i in range(args.warmup + args.steps):
        upd, sec, threads, desc = oracle_sample_run(w, spec, target_s=per)
        if i >= args.warmup:
            vals.append((upd, sec))
    upd = sum(v[0] for v in vals); sec = sum(v[1] for v in vals)
    value = upd / sec
    out = {"impl": "reference",
           "metric": metric_name(spec),
           "value": value, "unit": "updates/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": sec / max(1, len(vals)) * 1e3, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"{args.workload}: {w.name}, {w.n_steps} time steps per bench step, "
                                  f"bc={'periodic' if w.bc == 0 else 'dirichlet'}, CFL {w.cfl}",
                      "B_per_gpu": w.B, "N": w.N, "n_steps": w.n_steps, "sample": desc,
                      "input_sha256": w.sha256()[:16]},
           "cpu_baseline": {"value": value, "unit": "updates/s", "cores": threads, "kind": "oracle",
                            "sample": desc, "cpu": cpu_info()},
           "e2e": {"value": value, "unit": "updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def run_peaks(args):
    """`--peaks`: only the FP-pipe micro-benchmarks (profiles/r02_peaks.md)."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --peaks needs a CUDA device")
    torch.cuda.set_device(0)
    from paper_2601_12204_b200 import build as _b
    _b.build()
    pk = peaks()
    sampler = ClockSampler(0)
    sampler.start(); t0 = time.time()
    pipe = measure_pipe_peaks(torch.device("cuda", 0), pk)
    for _ in range(20):                    # long enough for nvidia-smi to see the clocks under this load
        measure_pipe_peaks(torch.device("cuda", 0), pk)
    t1 = time.time()
    clocks = sampler.window(t0, t1)
    sampler.stop()
    print(json.dumps({"pipe_peaks": pipe, "clocks": clocks, "sm_max_mhz": pk["sm_max_mhz"],
                      "nominal_ginst_s": {"fp32": SM_COUNT * FP32_LANES * pk["sm_max_mhz"] / 1e3,
                                          "fp64": SM_COUNT * FP64_LANES * pk["sm_max_mhz"] / 1e3}}), flush=True)


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def respawn_under_torchrun(args, argv):
    """`python bench.py --gpus N` without torchrun: start N ranks of this same file, one GPU each."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(sys.argv[0]), *argv]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                 # the communicator log lets the driver count the ranks
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    return subprocess.call(cmd, env=env)


def main(argv=None):
    argv = list(sys.argv[1:] if argv is None else argv)
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2_f32", choices=list(WORKLOADS + MORE))
    ap.add_argument("--no-extras", action="store_true", help="skip the per-scheme table of the other configs")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline legs")
    ap.add_argument("--reduced", action="store_true", help="10x fewer time steps per bench step (debug only)")
    ap.add_argument("--peaks", action="store_true", help="only the FP-pipe micro-benchmarks")
    args = ap.parse_args(argv)
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if args.peaks:
        return run_peaks(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(respawn_under_torchrun(args, argv))
    run_ours(args)


if __name__ == "__main__":
    main()
