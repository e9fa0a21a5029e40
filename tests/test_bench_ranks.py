"""Host logic of bench.py's N > 1 path on the CPU: two gloo ranks.  Every rank runs its own
independent problem; the job's time is the max over ranks and the value the sum of the units over that time.  Also the
reference arm under torchrun: rank 0 alone prints the JSON line."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, world, local = bench.rank_env()
dist.init_process_group("gloo")
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))
val = bench.job_value(1_000_000_000, world, ms * 1e-3)
dist.barrier()
if rank == 0:
    print(json.dumps({{"ms": ms, "value": val, "world": world}}))
dist.destroy_process_group()
'''


def _torchrun(args, timeout=600):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29531"] + args
    env = dict(os.environ, OMP_NUM_THREADS="2")
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, cwd=ROOT, env=env)


def test_max_over_ranks_and_job_value_two_gloo_ranks(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["world"] == 2 and d["ms"] == 15.0                 # the slower rank's time
    assert d["value"] == pytest.approx(2 * 1.0 / 15e-3)         # GB of both ranks over the max time


def test_reference_arm_under_torchrun_prints_once():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup",
                   "0", "--ref-ne", "8"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["unit"] == "GB/s" and d["n_gpus"] == 2
