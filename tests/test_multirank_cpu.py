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


# ---- row f3: halo exchange routing over a periodic ring of ranks (gloo, CPU tensors) ----
def _halo_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2306_01098_b200 import partition
    dist.init_process_group("gloo", rank=rank, world_size=world)
    slo = torch.full((2, 3, 8), 10.0 * rank + 1, dtype=torch.complex128)   # my lowest interior slices
    shi = torch.full((2, 3, 8), 10.0 * rank + 2, dtype=torch.complex128)   # my highest interior slices
    rlo, rhi = torch.zeros_like(slo), torch.zeros_like(slo)
    partition.exchange_halos(slo, shi, rlo, rhi, rank, world, dist)
    q.put((rank, rlo[0, 0, 0].real.item(), rhi[0, 0, 0].real.item()))
    dist.barrier()
    dist.destroy_process_group()


import pytest


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_ring_routing(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000 + world
    ps = [ctx.Process(target=_halo_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = {r: (lo, hi) for r, lo, hi in (q.get(timeout=120) for _ in ps)}
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        lo, hi = res[r]
        assert lo == 10.0 * ((r - 1) % world) + 2      # lower halo <- previous rank's highest slices
        assert hi == 10.0 * ((r + 1) % world) + 1      # upper halo <- next rank's lowest slices


def test_global_sites_of_rank_cover_the_lattice_once():
    from paper_2306_01098_b200 import layout, partition
    L, G = (4, 6, 4, 16), 4
    Le = partition.extended_lattice(L, G)
    V, Ve = layout.volume(L), layout.volume(Le)
    S2 = Ve // Le[3]
    count = torch.zeros(V, dtype=torch.int64)
    for r in range(G):
        sites = partition.global_sites_of_rank(L, r, G)
        lex_e = layout.lex_of_eo(Le)
        t_e = lex_e // (Le[0] * Le[1] * Le[2])
        interior = (t_e >= partition.HALO_T) & (t_e < Le[3] - partition.HALO_T)
        count.index_add_(0, sites[interior], torch.ones(int(interior.sum()), dtype=torch.int64))
        # parity is preserved by the even halo depth: local parity half == global parity
        x = sites % L[0]; y = (sites // L[0]) % L[1]; z = (sites // (L[0] * L[1])) % L[2]; t = sites // (L[0] * L[1] * L[2])
        gpar = (x + y + z + t) & 1
        assert torch.all(gpar[: Ve // 2] == 0) and torch.all(gpar[Ve // 2:] == 1)
    assert torch.all(count == 1)


# ---- a 2 x 2 grid of ranks (cut along z and t): both directions of the exchange, gloo, CPU tensors ----
def _grid_worker(rank, grid, port, q):
    world = grid[0] * grid[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from paper_2306_01098_b200 import partition
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nb = partition.grid_neighbours(rank, grid)
    got = {}
    for d, (nr, base) in {"t": (grid[1], 0), "z": (grid[0], 2)}.items():
        code = 100.0 * rank + (10.0 if d == "z" else 0.0)
        slo = torch.full((1, 3, 4), code + 1, dtype=torch.complex128)      # my lowest owned slices / planes
        shi = torch.full((1, 3, 4), code + 2, dtype=torch.complex128)      # my highest
        rlo, rhi = torch.zeros_like(slo), torch.zeros_like(slo)
        partition.begin_exchange(slo, shi, rlo, rhi, rank, nr, dist, up=nb[d + "_up"], down=nb[d + "_down"], tag_base=base).finish()
        got[d] = (rlo[0, 0, 0].real.item(), rhi[0, 0, 0].real.item())
    q.put((rank, nb, got))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("grid", [(2, 2), (2, 1)])
def test_halo_exchange_grid_routing(grid):
    nz, nt = grid
    world = nz * nt
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 32500 + os.getpid() % 2000 + 3 * world
    ps = [ctx.Process(target=_grid_worker, args=(r, grid, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = {r: (nb, got) for r, nb, got in (q.get(timeout=120) for _ in ps)}
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        rz, rt = r % nz, r // nz
        nb, got = res[r]
        assert nb == {"t_down": rz + nz * ((rt - 1) % nt), "t_up": rz + nz * ((rt + 1) % nt),
                      "z_down": (rz - 1) % nz + nz * rt, "z_up": (rz + 1) % nz + nz * rt}
        # lower halo <- the "down" neighbour's highest slices, upper halo <- the "up" neighbour's lowest
        assert got["t"] == (100.0 * nb["t_down"] + 2, 100.0 * nb["t_up"] + 1)
        assert got["z"] == (100.0 * nb["z_down"] + 12, 100.0 * nb["z_up"] + 11)
