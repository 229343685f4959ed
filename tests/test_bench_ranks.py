"""world_size-2 gloo tests (CPU) of bench.py's multi-rank host logic: the path shards by giving every
rank its own independent frame sequence (weak scaling, no data-path collective), times
are reduced with MAX over ranks, and only rank 0 reports."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    from paper_1607_00908_b200 import workloads as W
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = bench.rank_workload(W.scaled(5, 256), rank)
        frames = list(w.frames(2))
        sig = torch.tensor([int(frames[0][0].astype(np.int64).sum()), int(frames[1][1].astype(np.int64).sum())])
        sigs = [torch.zeros_like(sig) for _ in range(world)]
        dist.all_gather(sigs, sig)
        ms = bench.reduce_max(10.0 + 5.0 * rank, world, "cpu")          # rank 1 is the slow one
        val = bench.whole_job_value(world, 4, w.L * w.L, ms)
        out[rank] = dict(seed=w.seed, n=w.n_sites, L=w.L, sigs=[s.tolist() for s in sigs], ms=ms, val=val)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_by_independent_sequences():
    world, port = 2, 29500 + os.getpid() % 2000
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0["seed"] != r1["seed"] and r0["n"] == r1["n"] and r0["L"] == r1["L"]   # same config, own data
    assert r0["sigs"] == r1["sigs"] and r0["sigs"][0] != r0["sigs"][1]               # inputs really differ
    assert r0["ms"] == r1["ms"] == 15.0                                              # MAX over ranks
    assert r0["val"] == pytest.approx(2 * 4 * 256 * 256 / 15e-3)                     # whole-job aggregate


def _run_reference(rank):
    env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                           "--steps", "1", "--warmup", "0", "--workload", "cfg5@256"],
                          env=env, capture_output=True, text=True, timeout=300)


def test_reference_arm_runs_on_rank0_only():
    r1 = _run_reference(1)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = _run_reference(0)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0


def test_gpus_flag_spawns_the_ranks():
    """`bench.py --gpus 2` without a launcher starts two ranks itself (torch.distributed.run on 127.0.0.1):
    rank 0 prints the one line with n_gpus = 2, rank 1 prints nothing.  The reference arm needs no GPU."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0", "--workload", "cfg5@256"],
                       env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    line = json.loads(lines[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0


def test_gpus_flag_must_match_world_size():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0",
                        "--workload", "cfg5@256"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stderr + r.stdout)
