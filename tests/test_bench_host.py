"""Host logic of bench.py and of the rank-grid plumbing that needs no GPU: the traffic table refuses captures taken from
other kernel sources, the oracle's sample lattice, the (nz, nt) grid choice and the site bookkeeping of a z x t cut."""
import os

import numpy as np
import pytest
import torch

import bench
from paper_2306_01098_b200 import binding, layout, partition


def test_traffic_rows_are_tied_to_the_kernel_sources(tmp_path, monkeypatch):
    prof = tmp_path / "profiles"
    prof.mkdir()
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    os.makedirs(tmp_path / "paper_2306_01098_b200" / "csrc")
    for f in ("dslash.cuh", "dslash_launch_impl.cuh", "common.cuh"):
        (tmp_path / "paper_2306_01098_b200" / "csrc" / f).write_text("// " + f)
    h = bench.kernel_source_hash()
    (prof / "r2_traffic.csv").write_text(f"workload,kernel_source_hash,dram_bytes_per_launch,capture\nC5:fp64:8,{h},123,cap.md\nC3:fp32:8,deadbeef0000,9,old.md\n")
    assert bench.ncu_traffic("C5", "fp64", 8) == (123, "cap.md")
    val, why = bench.ncu_traffic("C3", "fp32", 8)
    assert val is None and "stale" in why
    val, why = bench.ncu_traffic("C2", "fp64", 1)
    assert val is None and "no row" in why
    (tmp_path / "paper_2306_01098_b200" / "csrc" / "dslash.cuh").write_text("// changed kernel")
    assert bench.ncu_traffic("C5", "fp64", 8)[0] is None          # the kernel changed: the old capture no longer counts


def test_committed_traffic_table_matches_the_committed_kernel():
    """profiles/r2_traffic.csv must describe the kernel in this tree (bench.py prints traffic = null otherwise)."""
    val, src = bench.ncu_traffic("C5", "fp64", 8)
    assert val is not None, src
    assert 0.9 * bench.dslash_bytes(96 ** 3 * 24 // 2, 8, 8) < val < 2.0 * bench.dslash_bytes(96 ** 3 * 24 // 2, 8, 8)


def test_oracle_sample_lattice_and_algorithmic_bytes():
    assert bench.oracle_block(bench.CONFIGS["C5"]) == (48, 48, 48, 12)
    assert bench.oracle_block(bench.CONFIGS["C2"]) == (32, 32, 32, 8)
    assert bench.dslash_bytes(131072, 1, 8) == 314572800          # C2: (288 + 12) words x 8 B x Vh
    assert bench.dslash_bytes(10616832, 8, 8) == (288 + 96) * 8 * 10616832


def test_rank_grid_choice():
    assert binding.rank_grid((96, 96, 96, 24), 8) == (2, 4)       # C5 on a full node: t alone would leave Lt_loc = 3
    assert binding.rank_grid((96, 96, 96, 24), 6) == (1, 6)
    assert binding.rank_grid((32, 32, 32, 8), 2) == (1, 2)
    assert binding.rank_grid((48, 48, 48, 12), 8) == (4, 2)
    with pytest.raises(ValueError):
        binding.rank_grid((4, 4, 4, 4), 8)


@pytest.mark.parametrize("grid", [(2, 2), (3, 1), (1, 2)])
def test_grid_site_bookkeeping_covers_the_lattice_once(grid):
    """Every global site is owned by exactly one rank of the grid, and halo sites are copies of the right neighbours."""
    L = (4, 4, 12, 8)
    nz, nt = grid
    V = layout.volume(L)
    seen = np.zeros(V, dtype=int)
    Le = partition.extended_lattice(L, grid)
    z_lo, z_cnt, t_lo, t_cnt = partition.owned_box(L, grid)
    for r in range(nz * nt):
        g = partition.global_sites_of_rank(L, r, grid).numpy()
        lex = layout.lex_of_eo(Le).numpy()                        # local lexicographic site of every memory slot
        z, t = (lex // (Le[0] * Le[1])) % Le[2], lex // (Le[0] * Le[1] * Le[2])
        own = (z >= z_lo) & (z < z_lo + z_cnt) & (t >= t_lo) & (t < t_lo + t_cnt)
        seen[g[own]] += 1
        # a local hop of +1 in t from an owned site lands on the global +t neighbour, also across the rank boundary
        gt = g // (L[0] * L[1] * L[2])
        rt = r // nz
        assert np.array_equal(gt, (rt * (L[3] // nt) + t - partition.HALO_T) % L[3])
        if nz > 1:
            gz = (g // (L[0] * L[1])) % L[2]
            assert np.array_equal(gz, ((r % nz) * (L[2] // nz) + z - partition.HALO_T) % L[2])
    assert np.all(seen == 1)
