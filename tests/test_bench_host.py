"""Host-side logic of bench.py on CPU: the replica aggregation over ranks (world size 2, gloo), the locked
roofline arithmetic, and the reference arm's JSON line.  No GPU, no CUDA calls."""
from __future__ import annotations

import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.dist_env() == (rank, rank, world)

    def reduce_max(x: float) -> float:
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    dist.barrier()
    ms_local = 2.0 if rank == 0 else 3.0        # the slower rank sets the job's step time
    value, ms = bench.aggregate(1_537_200, ms_local, world, reduce_max)
    q.put((rank, value, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms in got:
        assert ms == 3.0                                          # max over ranks
        assert value == 2 * 1_537_200 / 3.0e-3                    # whole-job solves/s over both replicas


def test_algorithmic_work_is_the_locked_count():
    sys.path.insert(0, str(ROOT))
    import bench
    meta = dict(n_columns=2562, n_layers=40, n_bins=30, n_gauss=20)
    mu = np.r_[np.full(1281, 0.5), np.full(1281, -0.5)]
    slots = bench.algorithmic_slots(meta, 1, mu)
    assert slots == 40 * 600 * (1281 * 156.0 + 1281 * 108.0)
    assert bench.algorithmic_slots(meta, 3, mu) == 40 * 600 * (1281 * 368.0 + 1281 * 272.0)
    cfg = dict(ktab=np.zeros((20, 30, 30, 20)))
    b = bench.algorithmic_bytes(meta, cfg, toa=False)
    assert b == 8 * (2 * 2562 * 40 + 2562 + 30) + 8 * (3 * 2562 * 41 + 2562 * 40) + 20 * 30 * 600 * 8


def test_reference_arm_prints_one_json_line():
    """`bench.py --impl reference` = the oracle on the host cores (tier's reference arm); config 5's shape is
    skipped here for time, config 2 with one step."""
    env = dict(os.environ, OMP_NUM_THREADS=str(min(8, os.cpu_count() or 1)))
    res = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, env=env, cwd=str(ROOT))
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "solves/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0
    assert d["gpu_launches"] == 0 and d["vs_baseline"] is None


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    res = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=120, env=env, cwd=str(ROOT))
    assert res.returncode == 0 and res.stdout.strip() == ""
