"""The N > 1 path of bench.py on CPU: world_size 2 over gloo (replicas only, no collective on the
data path).  Covers the rank logic: independent replica per rank, MAX over ranks of the device time, whole-job value,
and the reference arm under torchrun (rank 0 alone runs and prints)."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import workloads


def _worker(rank: int, world: int, port: int, out: str):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    w = workloads.config(0, replica=rank)                    # what cuda_arm gives this rank
    ms_local = 10.0 * (rank + 1)                             # rank 1 is the slow one
    ms_max, value = bench.whole_job_value(ms_local, w.n_atoms, 50, world, device="cpu")
    dist.barrier()
    np.save(out + f".{rank}.npy", np.concatenate([[ms_max, value], w.positions[:4].ravel()]))
    dist.destroy_process_group()


def test_two_ranks_max_time_and_whole_job_value(tmp_path):
    import torch.multiprocessing as mp
    out = str(tmp_path / "r")
    mp.spawn(_worker, args=(2, 29611, out), nprocs=2, join=True)
    a, b = np.load(out + ".0.npy"), np.load(out + ".1.npy")
    n = workloads.config(0).n_atoms
    assert a[0] == b[0] == 20.0                              # MAX over ranks, the same on every rank
    assert a[1] == b[1] == 2 * n * 50 / 20e-3                # all ranks' atom-steps over the slowest rank's time
    assert not np.allclose(a[2:], b[2:])                     # every rank runs its own replica (different seed)
    assert np.array_equal(a[2:], workloads.config(0).positions[:4].ravel())   # replica 0 is the plain config


def test_reference_arm_under_torchrun_prints_once():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29612", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2",
           "--warmup", "1", "--workload", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone runs and prints; rank 1 exits 0 without work
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["unit"] == "atom-steps/s"


def test_world_size_must_match_gpus():
    env = {**os.environ, "RANK": "0", "WORLD_SIZE": "2", "LOCAL_RANK": "0"}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "4"], capture_output=True,
                       text=True, env=env, timeout=120, cwd=ROOT)
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stderr + r.stdout)
