"""-m gpu: bench.py's multi-rank entry points on the one GPU of the test box (two processes share it; the transport is the
library's peer mailboxes through CUDA IPC, torch.distributed (gloo) only combines the timings)."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench(*args):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, cwd=ROOT,
                       env=env, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, p.stdout[-2000:]          # rank 0 alone prints, exactly one line
    return json.loads(lines[0])


def test_bench_gpus_2_partitioned_spawns_its_own_ranks():
    """`python bench.py --gpus 2 --mode partitioned` outside torchrun: starts two ranks itself, solves ONE lattice cut over
    them with hisq_cg."""
    d = _bench("--gpus", "2", "--mode", "partitioned", "--config", "C1", "--steps", "1", "--warmup", "3", "--step-iters", "16")
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and d["value"] > 0
    assert d["step"]["iterations"] == 16 and d["config"]["mode"] == "partitioned"
    assert d["gpu_launches"] > 16 * 8


def test_bench_gpus_2_replicas_spawns_its_own_ranks():
    d = _bench("--gpus", "2", "--config", "C1", "--steps", "1", "--warmup", "3", "--step-iters", "16", "--no-full-solve",
               "--no-configs", "--no-extras", "--no-cpu-baseline")
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["value"] > 0
    assert d["config"]["parallelism"] == "replicas only"
