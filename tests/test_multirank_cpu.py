"""N > 1 path on CPU (gloo, world_size 2): the path shards as independent replicas with no data-path
collective; the only cross-rank step is combining timings (max) and work (sum) in bench.aggregate."""
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, fl = bench.aggregate(10.0 + 5.0 * rank, 100.0 * (rank + 1), dist, torch.device("cpu"))
    q.put((rank, ms, fl))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_is_max_time_and_sum_work_over_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, ms, fl in res:
        assert ms == 15.0 and fl == 300.0


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_replicas_use_distinct_seeded_inputs():
    from paper_2306_01098_b200 import inputs
    s = torch.arange(64, dtype=torch.int64)
    a = inputs.fat_links((4, 4, 4, 4), 0, s)
    b = inputs.fat_links((4, 4, 4, 4), 1, s)
    assert not torch.equal(a, b)
