"""-m gpu: row f3 first step -- the Dslash on a lattice partitioned along t.  The ranks are EMULATED on one GPU as
separate contexts run one after the other (no kernel waits on another); the exchange that torch.distributed does
between processes is a direct copy here.  Every rank's interior must reproduce the single-lattice result bit for bit
(same per-site arithmetic) and agree with the oracle."""
import numpy as np
import pytest
import torch

import oracle
from paper_2306_01098_b200 import binding, layout, partition
from tests.gpu_helpers import rel_l2
from tests.helpers import oracle_field, oracle_links

pytestmark = pytest.mark.gpu


def _run(L, prec, nranks, nrhs, parity, seed):
    dev = torch.device("cuda:0")
    ctxs, fields, bufs = [], [], []
    for r in range(nranks):
        ctx = binding.Hisq(L, prec, nrhs, dev, part=(r, nranks))
        fat, naik = partition.make_links_part(L, seed, r, nranks, dev, ctx.cdtype)
        ctx.set_links(fat, naik)
        src = partition.make_sources_part(L, seed + 1, nrhs, 1 - parity, r, nranks, dev, ctx.cdtype)
        f = ctx.pack(src)
        slo, shi = ctx.halo_buffers(nrhs)
        ctx.halo_pack(f, slo, shi)
        ctxs.append(ctx); fields.append(f); bufs.append((slo, shi))
    outs = []
    for r, ctx in enumerate(ctxs):
        rlo = bufs[(r - 1) % nranks][1]      # previous rank's highest interior slices
        rhi = bufs[(r + 1) % nranks][0]      # next rank's lowest interior slices
        ctx.halo_unpack(fields[r], rlo, rhi)
        out = ctx.new_field(nrhs)
        out.zero_()
        ctx.dslash(fields[r], parity, out=out)
        outs.append(ctx.unpack(out).cpu().numpy().astype(np.complex128))
    # gather the interiors into a global full-lattice field
    V = layout.volume(L)
    full = np.zeros((nrhs, V, 3), dtype=np.complex128)
    seen = np.zeros(V, dtype=np.int64)
    Le = partition.extended_lattice(L, nranks)
    Vh_e = layout.volume(Le) // 2
    S = Vh_e // Le[3]
    for r in range(nranks):
        sites = partition.global_sites_of_rank(L, r, nranks).numpy()[parity * Vh_e:(parity + 1) * Vh_e]
        interior = np.zeros(Vh_e, dtype=bool)
        interior.reshape(Le[3], S)[partition.HALO_T:Le[3] - partition.HALO_T] = True
        full[:, sites[interior]] = outs[r][:, interior]
        seen[sites[interior]] += 1
        # halo slices of the output are left untouched (zero here)
        assert np.all(outs[r][:, ~interior] == 0)
    for c in ctxs:
        c.close()
    return full, seen


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
@pytest.mark.parametrize("nranks", [1, 2, 4])
def test_partitioned_dslash_equals_single_lattice_and_oracle(nranks, prec):
    L, nrhs, seed = (8, 4, 6, 16), 2, 3
    X, W = oracle_links(L, seed)
    if prec == "fp32":
        X, W = X.astype(np.complex64).astype(np.complex128), W.astype(np.complex64).astype(np.complex128)
    par_sites = oracle.site_parity(L)
    for parity in (0, 1):
        full, seen = _run(L, prec, nranks, nrhs, parity, seed)
        assert np.all(seen[par_sites == parity] == 1) and np.all(seen[par_sites != parity] == 0)
        src = oracle_field(L, seed + 1, nrhs, parity=1 - parity)
        if prec == "fp32":
            src = src.astype(np.complex64).astype(np.complex128)
        ref = oracle.dslash_parity(L, X, W, src, parity)
        assert rel_l2(full, ref) <= (1e-14 if prec == "fp64" else 1e-6)
        # single-lattice CUDA result: identical per-site arithmetic -> bitwise equal
        ctx = binding.Hisq(L, prec, nrhs)
        fat, naik = binding.make_links(L, seed, ctx.device, ctx.cdtype)
        ctx.set_links(fat, naik)
        s1 = ctx.pack(binding.make_sources(L, seed + 1, nrhs, 1 - parity, ctx.device, ctx.cdtype))
        one = oracle.half_to_full(L, ctx.unpack(ctx.dslash(s1, parity)).cpu().numpy().astype(np.complex128), parity)
        ctx.close()
        assert np.array_equal(full, one)


def test_partitioned_context_rejects_solvers_and_bad_splits():
    L = (4, 4, 4, 16)
    ctx = binding.Hisq(L, "fp64", 1, part=(0, 2))
    fat, naik = partition.make_links_part(L, 0, 0, 2, ctx.device)
    ctx.set_links(fat, naik)
    with pytest.raises(binding.HisqError) as e:
        ctx.cg(ctx.new_field(1), 0.1, 1e-8)
    assert e.value.code == -1
    ctx.close()
    with pytest.raises(ValueError):
        binding.Hisq((4, 4, 4, 12), "fp64", 1, part=(0, 4))      # Lt_loc = 3: odd
    with pytest.raises(ValueError):
        binding.Hisq((4, 4, 4, 8), "fp64", 1, part=(0, 4))       # Lt_loc = 2 < 4
