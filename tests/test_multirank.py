"""N > 1 host logic on CPU (the path shards over (B,H) with no exchange step -> replicas only).
What the multi-rank bench adds to the one-GPU path is (a) a barrier and a MAX over ranks of the device time,
(b) the whole-job aggregate, (c) distinct data per rank, (d) the reference arm running on rank 0 only.
world_size-2 `gloo` processes on 127.0.0.1 cover (a)-(c); (d) is run as the driver runs it (RANK in the env)."""
from __future__ import annotations

import json
import os
import subprocess
import sys
from pathlib import Path

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2605_30409_b200 import inputs as gin
    wl = gin.config(2)
    local_ms = 10.0 + 5.0 * rank                     # rank 1 is the slow one
    dist.barrier()
    ms = bench.max_over_ranks(local_ms, dist)
    q.put((rank, ms, bench.job_tokens_per_s(world, wl, 4, ms), bench.rank_seed(wl, rank, 3)))
    dist.destroy_process_group()


def test_two_gloo_ranks_agree_on_the_slowest_time_and_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ms0, v0, s0), (r1, ms1, v1, s1) = res
    assert (r0, r1) == (0, 1)
    assert ms0 == ms1 == 15.0                        # MAX over ranks, on every rank
    assert v0 == v1 == 2 * 1 * 3520 * 4 / 15e-3      # whole-job tokens / slowest rank's time
    assert s0 != s1                                  # every replica streams its own data


def test_max_over_ranks_without_process_group_is_identity():
    import bench
    assert bench.max_over_ranks(3.25, None) == 3.25


def _run_reference(rank: str):
    env = dict(os.environ, RANK=rank, WORLD_SIZE="2", LOCAL_RANK=rank, OMP_NUM_THREADS="4")
    return subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                          capture_output=True, text=True, env=env, timeout=600)


def test_reference_arm_runs_on_rank0_only():
    r1 = _run_reference("1")
    assert r1.returncode == 0 and r1.stdout.strip() == ""       # other ranks exit 0 without work
    r0 = _run_reference("0")
    assert r0.returncode == 0, r0.stderr[-2000:]
    line = json.loads([l for l in r0.stdout.splitlines() if l.startswith("{")][-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
