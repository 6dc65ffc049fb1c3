"""N>1 host logic on CPU: two `gloo` ranks (world_size 2) shard a batched workload the way
`bench.py --gpus 2` does (the last two tests run bench.py's own entry point: `--gpus 2` launched without
torchrun starts two ranks itself, with the GPU stepper replaced by a stub and gloo as the backend) (contiguous trajectory slices, no data-path
collective), and the pieces are checked against the unsharded batch:
  - every rank's shard is bit-identical to the same rows of the full workload,
  - the shards tile the batch exactly (no row lost or duplicated),
  - stepping the shards independently (here: with the CPU oracle, the only stepper that runs
    without a GPU) and concatenating equals stepping the whole batch -- i.e. sharding needs no
    exchange,
  - the max-over-ranks reduction bench.py uses for its timing returns the slowest rank's value.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2601_12204_b200 import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, Bg, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        rows = W.shard_rows(Bg, rank, world)
        results = {}
        for name, make, stepper in (
            ("c2", lambda r: W.c2_dirichlet_batch(B=Bg, N=128, dtype=np.float64, rows=r),
             lambda w, dt: oracle.explicit(w.u0, w.L, w.nu, dt, 40, w.bc, oracle.EULER, threads=1)),
            ("c3", lambda r: W.c3_periodic_btcs(B=Bg, N=64, rows=r),
             lambda w, dt: oracle.btcs(w.u0, w.L, w.nu, dt, 5, w.bc, threads=1)),
            ("c5", lambda r: W.c5_rk4_ensemble(B=Bg, N=64, dtype=np.float64, rows=r),
             lambda w, dt: oracle.explicit(w.u0, w.L, w.nu, dt, 20, w.bc, oracle.RK4, threads=1)),
        ):
            w = make(rows)
            dt = oracle.dt_from_cfl(w.u0, w.L, w.nu, w.cfl, w.bc)      # per trajectory: no all-reduce
            u = stepper(w, dt)
            # gather (rows, u0, dt, u) on every rank -- test plumbing only, not the data path
            gathered = [None] * world
            dist.all_gather_object(gathered, (rows, w.u0, dt, u))
            results[name] = gathered
        # bench.py's timing reduction: max over ranks
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        results["max_ms"] = float(t.item())
        dist.barrier()
        if rank == 0:
            torch.save(results, out)
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_batch_sharding_matches_full_batch(tmp_path):
    import oracle
    oracle.build()
    world, Bg = 2, 7                      # odd batch: ragged shards (4 + 3)
    out = str(tmp_path / "res.pt")
    mp.spawn(_rank_main, args=(world, _free_port(), Bg, out), nprocs=world, join=True)
    res = torch.load(out, weights_only=False)
    assert res["max_ms"] == 11.0
    full = {
        "c2": (W.c2_dirichlet_batch(B=Bg, N=128, dtype=np.float64),
               lambda w, dt: oracle.explicit(w.u0, w.L, w.nu, dt, 40, w.bc, oracle.EULER)),
        "c3": (W.c3_periodic_btcs(B=Bg, N=64), lambda w, dt: oracle.btcs(w.u0, w.L, w.nu, dt, 5, w.bc)),
        "c5": (W.c5_rk4_ensemble(B=Bg, N=64, dtype=np.float64),
               lambda w, dt: oracle.explicit(w.u0, w.L, w.nu, dt, 20, w.bc, oracle.RK4)),
    }
    for name, (w, stepper) in full.items():
        parts = res[name]
        rows = np.concatenate([p[0] for p in parts])
        np.testing.assert_array_equal(rows, np.arange(Bg))                      # exact tiling
        np.testing.assert_array_equal(np.concatenate([p[1] for p in parts]), w.u0)   # same inputs
        dt = oracle.dt_from_cfl(w.u0, w.L, w.nu, w.cfl, w.bc)
        np.testing.assert_array_equal(np.concatenate([p[2] for p in parts]), dt)
        np.testing.assert_array_equal(np.concatenate([p[3] for p in parts]), stepper(w, dt))


def test_shard_rows_properties():
    for Bg in (0, 1, 5, 1024, 65536 + 3):
        for world in (1, 2, 3, 8):
            parts = [W.shard_rows(Bg, r, world) for r in range(world)]
            np.testing.assert_array_equal(np.concatenate(parts), np.arange(Bg))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        W.shard_rows(8, 2, 2)


ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_STUB = """
import sys
sys.path.insert(0, {root!r})
import os
import bench


class StubRunner:                       # GpuRunner's interface, no device: rank r "takes" 10 + r ms per step
    def __init__(self, w, spec, device):
        self.w, self.plan, self.launches, self.op_launches = w, 1, 2, 1
        assert w.B == 1024 and str(device) == "cpu"

    def timed(self, steps, warmup):
        r = int(os.environ["RANK"])
        return [10.0 + r] * steps, [9.0 + r] * steps

    def e2e(self, steps, warmup):
        return [12.0] * steps, 7, 5


bench.BACKEND = "gloo"
bench.RUNNER = StubRunner
bench.main()
"""


@pytest.mark.timeout(300)
def test_bench_gpus_2_spawns_two_ranks_by_itself(tmp_path):
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment re-executes itself under
    torch.distributed.run with two ranks; each builds its own shard, the timing is the max over ranks and the
    value counts the updates of both."""
    stub = tmp_path / "bench_stub.py"
    stub.write_text(_STUB.format(root=ROOT))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    p = subprocess.run([sys.executable, str(stub), "--gpus", "2", "--steps", "2", "--warmup", "1", "--no-extras",
                        "--no-cpu", "--reduced"], capture_output=True, text=True, env=env, timeout=280)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, p.stdout                       # rank 0 alone prints, once
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["scaling"] == "weak"
    assert out["ms_per_step"] == 11.0                       # max over ranks of (10, 11)
    assert out["config"]["B_per_gpu"] == 1024 and "x2" in out["config"]["parallelism"]
    assert out["value"] == pytest.approx(2 * 1024 * 4096 * 1000 / 11.0e-3, rel=1e-6)
    assert out["gpu_launches"] == 4 and out["e2e"]["h2d_bytes_per_step"] == 7


def test_bench_refuses_a_world_size_that_contradicts_gpus():
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "3", "--no-extras", "--no-cpu"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert p.returncode != 0 and "WORLD_SIZE=2" in (p.stderr + p.stdout)
