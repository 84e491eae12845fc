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


def _run(L, prec, nranks, nrhs, parity, seed, overlap=False, peer=False):
    dev = torch.device("cuda:0")
    ctxs, fields, bufs = [], [], []
    for r in range(nranks):
        ctx = binding.Hisq(L, prec, nrhs, dev, part=(r, nranks))
        fat, naik = partition.make_links_part(L, seed, r, nranks, dev, ctx.cdtype)
        ctx.set_links(fat, naik)
        src = partition.make_sources_part(L, seed + 1, nrhs, 1 - parity, r, nranks, dev, ctx.cdtype)
        f = ctx.pack(src)
        slo, shi = ctx.halo_buffers(nrhs)
        if not peer:
            ctx.halo_pack(f, slo, shi)
        ctxs.append(ctx); fields.append(f); bufs.append((slo, shi))
    if peer:
        # mailboxes in the one process: plain device pointers.  All sends are enqueued before any recv (one stream).
        boxes = [c.peer_mailbox(nrhs) for c in ctxs]
        for r, c in enumerate(ctxs):
            c.peer_attach(boxes, nrhs)
        for c, f in zip(ctxs, fields):
            c.halo_send(f)
    outs = []
    nt, w = L[3] // nranks, partition.HOP_MAX
    for r, ctx in enumerate(ctxs):
        rlo = bufs[(r - 1) % nranks][1]      # previous rank's highest interior slices
        rhi = bufs[(r + 1) % nranks][0]      # next rank's lowest interior slices
        out = ctx.new_field(nrhs)
        out.zero_()
        if overlap and nt > 2 * w:
            # the slices that read no halo BEFORE the halo arrives (it holds NaN until then), the rest after
            S = ctx.Vh // ctx.L[3]
            v = fields[r].view(nrhs, 3, ctx.L[3], S)
            v[:, :, :partition.HALO_T] = float("nan")
            v[:, :, ctx.L[3] - partition.HALO_T:] = float("nan")
            ctx.dslash_slices(fields[r], parity, out, w, nt - 2 * w)
            ctx.halo_recv(fields[r]) if peer else ctx.halo_unpack(fields[r], rlo, rhi)
            ctx.dslash_edges(fields[r], parity, out, w)
        else:
            ctx.halo_recv(fields[r]) if peer else ctx.halo_unpack(fields[r], rlo, rhi)
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
        # interior / boundary split around the exchange (hisq_dslash_slices): the same bits
        full_o, seen_o = _run(L, prec, nranks, nrhs, parity, seed, overlap=True)
        assert np.array_equal(seen_o, seen) and np.array_equal(full_o, full)
        # halos moved through the mailboxes (hisq_halo_send / recv) instead of pack / copy / unpack: the same bits
        full_p, seen_p = _run(L, prec, nranks, nrhs, parity, seed, overlap=(parity == 0), peer=True)
        assert np.array_equal(seen_p, seen) and np.array_equal(full_p, full)


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_dslash_slices_compose_to_the_full_dslash(prec):
    L, nrhs, seed = (6, 4, 4, 10), 3, 8
    ctx = binding.Hisq(L, prec, nrhs)
    fat, naik = binding.make_links(L, seed, ctx.device, ctx.cdtype)
    ctx.set_links(fat, naik)
    S = ctx.Vh // L[3]
    for parity in (0, 1):
        src = ctx.pack(binding.make_sources(L, seed + 1, nrhs, 1 - parity, ctx.device, ctx.cdtype))
        ref = ctx.dslash(src, parity)
        out = ctx.new_field(nrhs)
        out.fill_(7.0)
        ctx.dslash_slices(src, parity, out, 2, 5)
        v, vr = out.view(nrhs, 3, L[3], S), ref.view(nrhs, 3, L[3], S)
        assert torch.equal(v[:, :, 2:7], vr[:, :, 2:7])
        assert torch.all(v[:, :, :2] == 7.0) and torch.all(v[:, :, 7:] == 7.0)     # the other slices are untouched
        ctx.dslash_slices(src, parity, out, 0, 2)
        ctx.dslash_slices(src, parity, out, 7, 3)
        ctx.dslash_slices(src, parity, out, 4, 0)                                 # empty range: nothing happens
        assert torch.equal(out, ref)
        out.fill_(7.0)
        ctx.dslash_edges(src, parity, out, 3)                                     # slices 0-2 and 7-9
        assert torch.equal(v[:, :, :3], vr[:, :, :3]) and torch.equal(v[:, :, 7:], vr[:, :, 7:])
        assert torch.all(v[:, :, 3:7] == 7.0)
        ctx.dslash_edges(src, parity, out, 5)                                     # 2 * width >= Lt: everything
        assert torch.equal(out, ref)
    for bad in ((-1, 2), (0, 11), (9, 2), (3, -1)):
        with pytest.raises(binding.HisqError) as e:
            ctx.dslash_slices(src, 0, out, *bad)
        assert e.value.code == -1
    ctx.close()


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


def _emulated_cg(L, prec, nranks, nrhs, m, tol, seed, overlap=False, peer=False):
    """All ranks in lockstep on one GPU: every phase is run for rank 0..G-1 in turn, the cross-rank steps (ring halo
    exchange, all-reduce) are done by hand between the phases -- the same sequence as partition.PartitionedCG.solve."""
    dev = torch.device("cuda:0")
    ctxs, bs, xs = [], [], []
    for r in range(nranks):
        ctx = binding.Hisq(L, prec, nrhs, dev, part=(r, nranks))
        fat, naik = partition.make_links_part(L, seed, r, nranks, dev, ctx.cdtype)
        ctx.set_links(fat, naik)
        b = ctx.pack(partition.make_sources_part(L, seed + 1, nrhs, 0, r, nranks, dev, ctx.cdtype, fill_halo=True))
        x = ctx.new_field(nrhs)
        ctx.cgp_begin(x, b, tol)
        ctxs.append(ctx); bs.append(b); xs.append(x)

    def allreduce(which):
        if peer:      # every rank stores into every mailbox, then every rank sums in rank order
            for c in ctxs: c.peer_reduce_send(which, nrhs)
            for c in ctxs: c.peer_reduce_recv(which, nrhs)
            return
        ts = [c.cgp_tensor(which, nrhs) for c in ctxs]
        tot = ts[0].clone()
        for t in ts[1:]:      # rank order, as the mailbox all-reduce adds
            tot += t
        for t in ts:
            t.copy_(tot)

    if peer:
        boxes = [c.peer_mailbox(nrhs) for c in ctxs]
        for r, c in enumerate(ctxs):
            c.peer_attach(boxes, nrhs)

    def halo(which, between=None):
        fields = [c.cgp_tensor(which, nrhs) for c in ctxs]
        if peer:
            for c, f in zip(ctxs, fields): c.halo_send(f)
            if between is not None:
                for c in ctxs: c.cgp_phase(between, m)
            for c, f in zip(ctxs, fields): c.halo_recv(f)
            return
        bufs = []
        for c, f in zip(ctxs, fields):
            slo, shi = c.halo_buffers(nrhs)
            c.halo_pack(f, slo, shi)
            bufs.append((slo, shi))
        if between is not None:      # what a rank computes while its halo is in flight
            for c in ctxs: c.cgp_phase(between, m)
        for r, (c, f) in enumerate(zip(ctxs, fields)):
            c.halo_unpack(f, bufs[(r - 1) % nranks][1], bufs[(r + 1) % nranks][0])

    allreduce(2)
    for c in ctxs:
        c.cgp_phase(0, m)
    st = ctxs[0].cgp_status(nrhs)
    while not st["done"] and st["iterations"] < 5000:
        for _ in range(16):
            for c in ctxs: c.cgp_phase(1, m)
            if overlap:
                halo(0, between=20)
                for c in ctxs: c.cgp_phase(21, m)
                halo(1, between=30)
                for c in ctxs: c.cgp_phase(31, m)
            else:
                halo(0)
                for c in ctxs: c.cgp_phase(2, m)
                halo(1)
                for c in ctxs: c.cgp_phase(3, m)
            allreduce(3)
            for c in ctxs: c.cgp_phase(4, m)
            allreduce(4)
            for c in ctxs: c.cgp_phase(5, m)
        st = ctxs[0].cgp_status(nrhs)
    for c in ctxs[1:]:
        assert c.cgp_status(nrhs)["iterations"] == st["iterations"]
    # gather the interiors of x
    V = layout.volume(L)
    full = np.zeros((nrhs, V, 3), dtype=np.complex128)
    Le = partition.extended_lattice(L, nranks)
    Vh_e = layout.volume(Le) // 2
    S = Vh_e // Le[3]
    for r, c in enumerate(ctxs):
        sites = partition.global_sites_of_rank(L, r, nranks).numpy()[:Vh_e]
        interior = np.zeros(Vh_e, dtype=bool)
        interior.reshape(Le[3], S)[partition.HALO_T:Le[3] - partition.HALO_T] = True
        full[:, sites[interior]] = c.unpack(xs[r]).cpu().numpy().astype(np.complex128)[:, interior]
        c.close()
    return full, st


@pytest.mark.parametrize("nranks", [1, 2, 4])
def test_partitioned_cg_matches_oracle_and_single_lattice(nranks):
    L, nrhs, m, tol, seed = (4, 6, 4, 16), 2, 0.1, 1e-10, 5
    x, st = _emulated_cg(L, "fp64", nranks, nrhs, m, tol, seed)
    X, W = oracle_links(L, seed)
    b = oracle_field(L, seed + 1, nrhs, parity=0)
    r = b - oracle.apply_A(L, X, W, m, x)
    for k in range(nrhs):
        assert np.linalg.norm(r[k]) / np.linalg.norm(b[k]) <= 1.05 * tol, (k, st)
    xo, it_o, _, ok, _ = oracle.cg(L, X, W, m, tol, b)
    assert ok == 0 and rel_l2(x, xo) <= 10 * tol
    assert abs(st["iterations"] - int(it_o.max())) <= 16 + 3      # status is polled every 16 iterations
    # Dslashes split around the halo exchange (phases 20/21, 30/31): same sums in the same order -> the same iterates
    x2, st2 = _emulated_cg(L, "fp64", nranks, nrhs, m, tol, seed, overlap=True)
    assert st2["iterations"] == st["iterations"] and np.array_equal(x2, x)
    # ... and with the halos moved through peer mailboxes (double-buffered: hundreds of exchanges reuse two slots)
    x3, st3 = _emulated_cg(L, "fp64", nranks, nrhs, m, tol, seed, overlap=True, peer=True)
    assert st3["iterations"] == st["iterations"] and np.array_equal(x3, x)


def test_partitioned_cg_driver_single_rank_equals_hisq_cg():
    """partition.PartitionedCG itself (dist = None: the ring closes on the rank) against hisq_cg on the plain lattice."""
    L, m, tol, seed = (4, 4, 6, 8), 0.2, 1e-10, 6
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, "fp64", 1, dev, part=(0, 1))
    fat, naik = partition.make_links_part(L, seed, 0, 1, dev)
    ctx.set_links(fat, naik)
    b = ctx.pack(partition.make_sources_part(L, seed + 1, 1, 0, 0, 1, dev))
    x, st = partition.PartitionedCG(ctx, 0, 1).solve(b, m, tol, check_every=8)
    assert st["done"] and max(st["rel_resid"]) <= tol
    ref = binding.Hisq(L, "fp64", 1, dev)
    f2, n2 = binding.make_links(L, seed, dev)
    ref.set_links(f2, n2)
    xr, info = ref.cg(ref.pack(binding.make_sources(L, seed + 1, 1, 0, dev)), m, tol)
    # interior of the partitioned solution == the plain solution
    Le = partition.extended_lattice(L, 1)
    S = ctx.Vh // Le[3]
    xi = ctx.unpack(x).view(1, Le[3], S, 3)[:, partition.HALO_T:Le[3] - partition.HALO_T].reshape(1, -1, 3)
    assert rel_l2(xi.cpu().numpy(), ref.unpack(xr).cpu().numpy()) <= 1e-9
    assert abs(st["iterations"] - info["iterations"]) <= 8 + 2
    ctx.close(); ref.close()


def test_hisq_cg_on_a_partitioned_context_single_rank_ring():
    """hisq_cg itself on a partitioned context (mailboxes attached; one rank, the ring closes on itself): the whole
    iteration, halos and all-reduces included, runs on the stream.  Against hisq_cg on the plain lattice."""
    L, m, tol, seed, n = (4, 4, 6, 12), 0.2, 1e-10, 16, 3
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, "fp64", n, dev, part=(0, 1))
    fat, naik = partition.make_links_part(L, seed, 0, 1, dev)
    ctx.set_links(fat, naik)
    b = ctx.pack(partition.make_sources_part(L, seed + 1, n, 0, 0, 1, dev))
    with pytest.raises(binding.HisqError):
        ctx.cg(b, m, tol)                         # no mailboxes yet
    peer = partition.PeerHalo(ctx, 0, 1, n)
    x, info = ctx.cg(b, m, tol)
    assert max(info["true_rel_resid"]) <= tol and info["reliable_updates"] >= 1     # confirmed with b - A x
    ref = binding.Hisq(L, "fp64", n, dev)
    f2, n2 = binding.make_links(L, seed, dev)
    ref.set_links(f2, n2)
    xr, iref = ref.cg(ref.pack(binding.make_sources(L, seed + 1, n, 0, dev)), m, tol)
    Le = partition.extended_lattice(L, 1)
    S = ctx.Vh // Le[3]
    xi = ctx.unpack(x).view(n, Le[3], S, 3)[:, partition.HALO_T:Le[3] - partition.HALO_T].reshape(n, -1, 3)
    assert rel_l2(xi.cpu().numpy(), ref.unpack(xr).cpu().numpy()) <= 1e-9
    assert abs(info["iterations"] - iref["iterations"]) <= 32 + 2          # polled every check_interval iterations
    assert np.allclose(info["true_rel_resid"], iref["true_rel_resid"], rtol=0.5)   # true residuals, both
    # max_iter on the partitioned path: not converged is reported as such
    ctx.set_option("max_iter", 3)
    with pytest.raises(binding.HisqError) as e:
        ctx.cg(b, m, 1e-14)
    assert e.value.code == -5
    peer.close()
    ctx.close(); ref.close()


def test_peer_calls_out_of_order_are_refused():
    """The two-slot mailbox protocol is only safe if sends and recvs alternate strictly: the library enforces it."""
    L, n = (4, 4, 4, 8), 2
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, "fp64", n, dev, part=(0, 1))
    f = ctx.new_field(n)
    f.zero_()
    with pytest.raises(binding.HisqError):
        ctx.halo_send(f)                                   # no mailboxes attached
    box = ctx.peer_mailbox(n)
    with pytest.raises(binding.HisqError):
        ctx.peer_attach([box, box], n)                     # one rank, two boxes
    with pytest.raises(binding.HisqError):
        ctx.peer_attach([box[8:]], n)                      # misaligned
    ctx.peer_attach([box], n)
    with pytest.raises(binding.HisqError):
        ctx.halo_recv(f)                                   # nothing sent
    ctx.halo_send(f)
    with pytest.raises(binding.HisqError):
        ctx.halo_send(f)                                   # two sends in a row
    ctx.halo_recv(f)
    with pytest.raises(binding.HisqError):
        ctx.peer_reduce_recv(3, n)                         # nothing sent
    with pytest.raises(binding.HisqError):
        ctx.peer_reduce_send(7, n)                         # not a state array
    ctx.peer_reduce_send(3, n)
    with pytest.raises(binding.HisqError):
        ctx.peer_reduce_send(4, n)                         # one reduce at a time
    ctx.peer_reduce_recv(3, n)
    torch.cuda.synchronize()
    # a plain (not partitioned) context has no mailbox
    plain = binding.Hisq(L, "fp64", n, dev)
    with pytest.raises(binding.HisqError):
        plain.peer_mailbox(n)
    plain.close(); ctx.close()


def test_peer_allreduce_sums_in_rank_order_same_bits_everywhere():
    """Emulated ranks: values chosen so that the floating-point sum depends on the order; every rank must end up with
    the rank-order sum, bit for bit."""
    L, n, nranks = (4, 4, 4, 16), 3, 4
    dev = torch.device("cuda:0")
    ctxs = [binding.Hisq(L, "fp64", n, dev, part=(r, nranks)) for r in range(nranks)]
    boxes = [c.peer_mailbox(n) for c in ctxs]
    for c in ctxs:
        c.peer_attach(boxes, n)
    vals = torch.tensor([[1e16, 1.0, -3.5], [1.0, 1e-16, 2.25], [-1e16, 1.0, 1e8], [1.0, -1.0, -1e8]], dtype=torch.float64, device=dev)
    for rep in range(5):                                   # several rounds: both slots are reused
        for r, c in enumerate(ctxs):
            c.cgp_tensor(3, n).copy_(vals[r] * (rep + 1))
        for c in ctxs: c.peer_reduce_send(3, n)
        for c in ctxs: c.peer_reduce_recv(3, n)
        want = torch.zeros(n, dtype=torch.float64, device=dev)
        for r in range(nranks):
            want = want + vals[r] * (rep + 1)
        for c in ctxs:
            assert torch.equal(c.cgp_tensor(3, n), want)
    for c in ctxs:
        c.close()


def _mp_worker(rank, world, port, L, m, tol, seed, q, transport):
    import os, sys
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda:0")                       # both ranks share the one GPU; no kernel waits on another
    ctx = binding.Hisq(L, "fp64", 1, dev, part=(rank, world))
    fat, naik = partition.make_links_part(L, seed, rank, world, dev)
    ctx.set_links(fat, naik)
    b = ctx.pack(partition.make_sources_part(L, seed + 1, 1, 0, rank, world, dev))
    peer = partition.PeerHalo(ctx, rank, world, 1, dist) if transport != "dist" else None
    if transport == "native":      # hisq_cg drives the iteration itself: no torch.distributed call inside the solve
        x, info = ctx.cg(b, m, tol)
        st = dict(done=info["status"] == 0, breakdown=False, iterations=info["iterations"])
    else:
        x, st = partition.PartitionedCG(ctx, rank, world, dist, peer=peer).solve(b, m, tol, check_every=8)
    if peer is not None:
        peer.close()
    Le = partition.extended_lattice(L, world)
    S = ctx.Vh // Le[3]
    xi = ctx.unpack(x).view(1, Le[3], S, 3)[:, partition.HALO_T:Le[3] - partition.HALO_T].reshape(1, -1, 3).cpu()
    xr = torch.view_as_real(xi).contiguous()
    parts = [torch.empty_like(xr) for _ in range(world)] if rank == 0 else None
    dist.gather(xr, parts, dst=0)
    if rank == 0:
        q.put((st, [torch.view_as_complex(p).numpy() for p in parts]))
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("transport", ["dist", "peer", "native"])
def test_partitioned_cg_two_processes_gloo_on_one_gpu(transport):
    """The real thing minus the second GPU: two PROCESSES, each with its own context, exchanging halos and all-reducing
    through torch.distributed (gloo here, NCCL between GPUs), run partition.PartitionedCG.solve.
    transport = "peer": the halos go through mailboxes mapped into the other process by CUDA IPC (partition.PeerHalo;
    the packing kernel stores into the neighbour's memory, stream memory operations signal) -- no kernel waits on
    another one, the streams do."""
    import torch.multiprocessing as mp
    L, m, tol, seed, world = (4, 4, 6, 16), 0.15, 1e-9, 8, 2
    ctxmp = mp.get_context("spawn")
    q = ctxmp.Queue()
    port = 33500 + __import__("os").getpid() % 2000 + {"dist": 0, "peer": 17, "native": 31}[transport]
    ps = [ctxmp.Process(target=_mp_worker, args=(r, world, port, L, m, tol, seed, q, transport)) for r in range(world)]
    for p in ps:
        p.start()
    try:
        st, parts = q.get(timeout=150)
        for p in ps:
            p.join(timeout=120)
            assert p.exitcode == 0
    finally:
        for p in ps:          # exactly the processes started above
            if p.is_alive():
                p.kill()
    assert st["done"] and not st["breakdown"]
    # rank r's interior = global even sites with t in [r*Lt_loc, (r+1)*Lt_loc), in global half-index order
    xh = np.concatenate(parts, axis=1).astype(np.complex128)
    x = oracle.half_to_full(L, xh, 0)
    X, W = oracle_links(L, seed)
    b = oracle_field(L, seed + 1, 1, parity=0)
    r = b - oracle.apply_A(L, X, W, m, x)
    assert np.linalg.norm(r) / np.linalg.norm(b) <= 1.05 * tol


def _abort_worker(rank, world, port, L, q, case):
    import os
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, "fp64", 2, dev, part=(rank, world))
    fat, naik = partition.make_links_part(L, 3, rank, world, dev)
    ctx.set_links(fat, naik)
    peer = partition.PeerHalo(ctx, rank, world, 1, dist)            # mailboxes sized for ONE right-hand side
    n = 2 if (case == "badcall" and rank == 1) else 1                # rank 1 asks for more than the mailboxes hold
    if case == "options" and rank == 1:
        ctx.set_option("max_iter", 77)                               # the ranks would run different numbers of exchanges
    b = ctx.pack(partition.make_sources_part(L, 4, n, 0, rank, world, dev))
    code = 0
    try:
        ctx.cg(b, 0.2, 1e-8)
    except binding.HisqError as e:
        code = e.code
    reattach = 0
    try:
        ctx.peer_attach(ctx._mailboxes, 1)                           # a mailbox that has been used / poisoned is refused
    except binding.HisqError as e:
        reattach = e.code
    q.put((rank, code, reattach))
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("case", ["badcall", "options"])
def test_multi_rank_solve_fails_on_every_rank_instead_of_hanging(case):
    """an early error return on one rank used to leave the other rank's stream parked in a stream wait for ever.
    badcall: rank 1's hisq_cg fails its argument check (HISQ_EINVAL) -> it poisons the counters, rank 0 returns HISQ_EPEER.
    options: the ranks were given different max_iter -> both see it in the option exchange and return HISQ_EINVAL."""
    import torch.multiprocessing as mp
    L, world = (4, 4, 4, 16), 2
    ctxmp = mp.get_context("spawn")
    q = ctxmp.Queue()
    port = 35600 + __import__("os").getpid() % 2000 + (0 if case == "badcall" else 13)
    ps = [ctxmp.Process(target=_abort_worker, args=(r, world, port, L, q, case)) for r in range(world)]
    for p in ps:
        p.start()
    try:
        res = dict((r, (c, ra)) for r, c, ra in (q.get(timeout=120) for _ in range(world)))
        for p in ps:
            p.join(timeout=60)
            assert p.exitcode == 0
    finally:
        for p in ps:
            if p.is_alive():
                p.kill()
    if case == "badcall":
        assert res[1][0] == binding.HISQ_EINVAL and res[0][0] == binding.HISQ_EPEER
    else:
        assert res[0][0] == binding.HISQ_EINVAL and res[1][0] == binding.HISQ_EINVAL
    assert res[0][1] == binding.HISQ_EINVAL and res[1][1] == binding.HISQ_EINVAL


def _interior(ctx, L, world, field, n):
    Le = partition.extended_lattice(L, world)
    S = ctx.Vh // Le[3]
    return ctx.unpack(field).view(n, Le[3], S, 3)[:, partition.HALO_T:Le[3] - partition.HALO_T].reshape(n, -1, 3)


def test_mixed_precision_and_multishift_on_a_single_rank_ring():
    """PAPER.md:135 / :141 on partitioned contexts: HISQ_MIXED hisq_cg and hisq_cg_multishift with the
    mailboxes attached (one rank, the ring closes on itself), against the same calls on the plain lattice and the oracle
    operator."""
    L, m, seed = (4, 4, 6, 12), 0.05, 21
    dev = torch.device("cuda:0")
    X, W = oracle_links(L, seed)
    # mixed precision, 2 right-hand sides, reliable updates every 20 iterations
    n, tol = 2, 1e-10
    ctx = binding.Hisq(L, "mixed", n, dev, part=(0, 1))
    ctx.set_links(*partition.make_links_part(L, seed, 0, 1, dev))
    ctx.set_option("reliable_interval", 20)
    b = ctx.pack(partition.make_sources_part(L, seed + 1, n, 0, 0, 1, dev))
    peer = partition.PeerHalo(ctx, 0, 1, n)
    x, info = ctx.cg(b, m, tol)
    assert info["reliable_updates"] >= info["iterations"] // 20 and max(info["true_rel_resid"]) <= tol
    xf = oracle.half_to_full(L, _interior(ctx, L, 1, x, n).cpu().numpy(), 0)
    bf = oracle_field(L, seed + 1, n, parity=0)
    r = bf - oracle.apply_A(L, X, W, m, xf)
    for k in range(n):
        assert np.linalg.norm(r[k]) / np.linalg.norm(bf[k]) <= tol
    peer.close(); ctx.close()
    # multi-shift, 4 shifts
    shifts, tol = [0.0, 0.01, 0.3, 2.0], 1e-9
    ctx = binding.Hisq(L, "fp64", len(shifts), dev, part=(0, 1))
    ctx.set_links(*partition.make_links_part(L, seed, 0, 1, dev))
    b = ctx.pack(partition.make_sources_part(L, seed + 2, 1, 0, 0, 1, dev))
    peer = partition.PeerHalo(ctx, 0, 1, 1)
    xs, info = ctx.cg_multishift(b, m, shifts, tol)
    assert max(info["true_rel_resid"]) <= tol
    xf = oracle.half_to_full(L, _interior(ctx, L, 1, xs, len(shifts)).cpu().numpy(), 0)
    bf = oracle_field(L, seed + 2, 1, parity=0)
    for k, sg in enumerate(shifts):
        rk = bf[0] - oracle.apply_A(L, X, W, float(np.sqrt(m * m + sg)), xf[k:k + 1])[0]
        assert np.linalg.norm(rk) / np.linalg.norm(bf[0]) <= tol
    peer.close(); ctx.close()


def _mp_worker2(rank, world, port, L, m, tol, seed, q, mode, shifts):
    import os
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda:0")
    nx = len(shifts) if mode == "multishift" else 1
    ctx = binding.Hisq(L, "mixed" if mode == "mixed" else "fp64", nx, dev, part=(rank, world))
    ctx.set_links(*partition.make_links_part(L, seed, rank, world, dev))
    if mode == "mixed":
        ctx.set_option("reliable_interval", 25)
    b = ctx.pack(partition.make_sources_part(L, seed + 1, 1, 0, rank, world, dev))
    peer = partition.PeerHalo(ctx, rank, world, 1, dist)
    if mode == "mixed":
        x, info = ctx.cg(b, m, tol)
    else:
        x, info = ctx.cg_multishift(b, m, shifts, tol)
    peer.close()
    xr = torch.view_as_real(_interior(ctx, L, world, x, nx).cpu()).contiguous()
    parts = [torch.empty_like(xr) for _ in range(world)] if rank == 0 else None
    dist.gather(xr, parts, dst=0)
    if rank == 0:
        q.put((info, [torch.view_as_complex(p).numpy() for p in parts]))
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("mode", ["mixed", "multishift"])
def test_mixed_and_multishift_two_processes_on_one_gpu(mode):
    """Two PROCESSES, mailboxes mapped through CUDA IPC, hisq_cg (HISQ_MIXED) and hisq_cg_multishift driving the iteration
    from C across the two ranks; judged by the oracle operator on the reassembled solution."""
    import torch.multiprocessing as mp
    L, m, tol, seed, world = (4, 4, 6, 16), 0.1, 1e-9, 11, 2
    shifts = [0.0, 0.02, 0.5]
    ctxmp = mp.get_context("spawn")
    q = ctxmp.Queue()
    port = 36700 + __import__("os").getpid() % 2000 + (0 if mode == "mixed" else 19)
    ps = [ctxmp.Process(target=_mp_worker2, args=(r, world, port, L, m, tol, seed, q, mode, shifts)) for r in range(world)]
    for p in ps:
        p.start()
    try:
        info, parts = q.get(timeout=150)
        for p in ps:
            p.join(timeout=120)
            assert p.exitcode == 0
    finally:
        for p in ps:
            if p.is_alive():
                p.kill()
    assert info["status"] == 0
    xh = np.concatenate(parts, axis=1).astype(np.complex128)
    X, W = oracle_links(L, seed)
    b = oracle_field(L, seed + 1, 1, parity=0)
    if mode == "mixed":
        assert info["reliable_updates"] >= info["iterations"] // 25
        r = b - oracle.apply_A(L, X, W, m, oracle.half_to_full(L, xh, 0))
        assert np.linalg.norm(r) / np.linalg.norm(b) <= 1.05 * tol
    else:
        xf = oracle.half_to_full(L, xh, 0)
        for k, sg in enumerate(shifts):
            rk = b[0] - oracle.apply_A(L, X, W, float(np.sqrt(m * m + sg)), xf[k:k + 1])[0]
            assert np.linalg.norm(rk) / np.linalg.norm(b[0]) <= 1.05 * tol


# ---- second cut, along z: a (nz x nt) grid of ranks (the t-only split cannot use an 8-GPU node on C5) --------
def _run_grid(L, prec, grid, nrhs, parity, seed, peer=False):
    """Emulated ranks of an nz x nt grid: Dslash of every rank on its box, halos by pack / copy / unpack (or through the
    mailboxes), reassembled into the global field."""
    dev = torch.device("cuda:0")
    nz, nt = grid
    nranks = nz * nt
    ctxs, fields, tb, zb = [], [], [], []
    for r in range(nranks):
        ctx = binding.Hisq(L, prec, nrhs, dev, part=(r, nz, nt))
        ctx.set_links(*partition.make_links_part(L, seed, r, grid, dev, ctx.cdtype))
        f = ctx.pack(partition.make_sources_part(L, seed + 1, nrhs, 1 - parity, r, grid, dev, ctx.cdtype))
        if not peer:
            t2 = ctx.halo_buffers(nrhs); ctx.halo_pack(f, *t2)
            z2 = ctx.zhalo_buffers(nrhs) if nz > 1 else None
            if nz > 1:
                ctx.zhalo_pack(f, *z2)
            tb.append(t2); zb.append(z2)
        ctxs.append(ctx); fields.append(f)
    if peer:
        boxes = [c.peer_mailbox(nrhs) for c in ctxs]
        for c in ctxs:
            c.peer_attach(boxes, nrhs)
        for c, f in zip(ctxs, fields):
            c.halo_send(f)
    V = layout.volume(L)
    full = np.zeros((nrhs, V, 3), dtype=np.complex128)
    seen = np.zeros(V, dtype=np.int64)
    Le = partition.extended_lattice(L, grid)
    Vh_e = layout.volume(Le) // 2
    z_lo, z_cnt, t_lo, t_cnt = partition.owned_box(L, grid)
    for r, ctx in enumerate(ctxs):
        rz, rt = r % nz, r // nz
        if peer:
            ctx.halo_recv(fields[r])
        else:
            ctx.halo_unpack(fields[r], tb[rz + nz * ((rt - 1) % nt)][1], tb[rz + nz * ((rt + 1) % nt)][0])
            if nz > 1:
                ctx.zhalo_unpack(fields[r], zb[(rz - 1) % nz + nz * rt][1], zb[(rz + 1) % nz + nz * rt][0])
        out = ctx.new_field(nrhs)
        out.zero_()
        ctx.dslash(fields[r], parity, out=out)
        o = ctx.unpack(out).cpu().numpy().astype(np.complex128)
        sites = partition.global_sites_of_rank(L, r, grid).numpy()[parity * Vh_e:(parity + 1) * Vh_e]
        own = np.zeros((Le[3], Le[2], Vh_e // (Le[3] * Le[2])), dtype=bool)
        own[t_lo:t_lo + t_cnt, z_lo:z_lo + z_cnt] = True
        own = own.reshape(-1)
        full[:, sites[own]] = o[:, own]
        seen[sites[own]] += 1
        assert np.all(o[:, ~own] == 0)            # nothing outside the owned box is written
    for c in ctxs:
        c.close()
    return full, seen


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
@pytest.mark.parametrize("grid", [(2, 1), (2, 2), (3, 2)])
def test_zt_partitioned_dslash_equals_single_lattice(grid, prec):
    L, nrhs, seed = (8, 4, 24, 16), 2, 5
    par_sites = oracle.site_parity(L)
    for parity in (0, 1):
        full, seen = _run_grid(L, prec, grid, nrhs, parity, seed)
        assert np.all(seen[par_sites == parity] == 1) and np.all(seen[par_sites != parity] == 0)
        ctx = binding.Hisq(L, prec, nrhs)
        ctx.set_links(*binding.make_links(L, seed, ctx.device, ctx.cdtype))
        s1 = ctx.pack(binding.make_sources(L, seed + 1, nrhs, 1 - parity, ctx.device, ctx.cdtype))
        one = oracle.half_to_full(L, ctx.unpack(ctx.dslash(s1, parity)).cpu().numpy().astype(np.complex128), parity)
        ctx.close()
        assert np.array_equal(full, one)          # identical per-site arithmetic: bit for bit
        full_p, seen_p = _run_grid(L, prec, grid, nrhs, parity, seed, peer=True)
        assert np.array_equal(seen_p, seen) and np.array_equal(full_p, full)
    if prec == "fp64" and grid == (2, 2):         # and against the oracle
        X, W = oracle_links(L, seed)
        ref = oracle.dslash_parity(L, X, W, oracle_field(L, seed + 1, nrhs, parity=0), 1)
        assert rel_l2(_run_grid(L, prec, grid, nrhs, 1, seed)[0], ref) <= 1e-14


def _mp_worker_grid(rank, grid, port, L, m, tol, seed, q, prec):
    import os
    world = grid[0] * grid[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, prec, 2, dev, part=(rank, grid[0], grid[1]))
    ctx.set_links(*partition.make_links_part(L, seed, rank, grid, dev))
    b = ctx.pack(partition.make_sources_part(L, seed + 1, 2, 0, rank, grid, dev))
    peer = partition.PeerHalo(ctx, rank, world, 2, dist)
    x, info = ctx.cg(b, m, tol)
    peer.close()
    xi = partition.interior(ctx, L, grid, ctx.unpack(x)).contiguous().cpu()
    xr = torch.view_as_real(xi).contiguous()
    parts = [torch.empty_like(xr) for _ in range(world)] if rank == 0 else None
    dist.gather(xr, parts, dst=0)
    if rank == 0:
        q.put((info, [torch.view_as_complex(p).numpy() for p in parts]))
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("grid,prec", [((2, 1), "fp64"), ((2, 2), "mixed")])
def test_zt_partitioned_cg_processes_on_one_gpu(grid, prec):
    """hisq_cg across the ranks of a (z, t) grid, one PROCESS per rank on the one GPU, mailboxes through CUDA IPC; the
    solution reassembled from the ranks' boxes is judged by the oracle operator."""
    import torch.multiprocessing as mp
    L, m, tol, seed = (4, 4, 16, 8), 0.1, 1e-9, 13
    world = grid[0] * grid[1]
    ctxmp = mp.get_context("spawn")
    q = ctxmp.Queue()
    port = 37800 + __import__("os").getpid() % 2000 + 7 * world
    ps = [ctxmp.Process(target=_mp_worker_grid, args=(r, grid, port, L, m, tol, seed, q, prec)) for r in range(world)]
    for p in ps:
        p.start()
    try:
        info, parts = q.get(timeout=200)
        for p in ps:
            p.join(timeout=120)
            assert p.exitcode == 0
    finally:
        for p in ps:
            if p.is_alive():
                p.kill()
    assert info["status"] == 0
    nz, nt = grid
    Lz_loc, Lt_loc, HLy = L[2] // nz, L[3] // nt, L[0] // 2 * L[1]
    xh = np.zeros((2, L[3], L[2], HLy, 3), dtype=np.complex128)       # global even half-index order [t][z][y, xh]
    for r, part in enumerate(parts):
        rz, rt = r % nz, r // nz
        xh[:, rt * Lt_loc:(rt + 1) * Lt_loc, rz * Lz_loc:(rz + 1) * Lz_loc] = part
    X, W = oracle_links(L, seed)
    b = oracle_field(L, seed + 1, 2, parity=0)
    r = b - oracle.apply_A(L, X, W, m, oracle.half_to_full(L, xh.reshape(2, -1, 3), 0))
    for k in range(2):
        assert np.linalg.norm(r[k]) / np.linalg.norm(b[k]) <= 1.05 * tol


def _mp_worker_grid_dslash(rank, grid, port, L, seed, q):
    import os
    world = grid[0] * grid[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cuda:0")
    ctx = binding.Hisq(L, "fp64", 2, dev, part=(rank, grid[0], grid[1]))
    ctx.set_links(*partition.make_links_part(L, seed, rank, grid, dev))
    f = ctx.pack(partition.make_sources_part(L, seed + 1, 2, 0, rank, grid, dev))
    # no mailboxes: both halos travel through torch.distributed (gloo here, staged through the host; NCCL between GPUs)
    out = partition.dslash_partitioned(ctx, f, 1, rank, grid, dist)
    xr = torch.view_as_real(partition.interior(ctx, L, grid, ctx.unpack(out)).contiguous().cpu()).contiguous()
    parts = [torch.empty_like(xr) for _ in range(world)] if rank == 0 else None
    dist.gather(xr, parts, dst=0)
    if rank == 0:
        q.put([torch.view_as_complex(p).numpy() for p in parts])
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


def test_zt_partitioned_dslash_through_torch_distributed_four_processes():
    """partition.dslash_partitioned on a 2 x 2 grid of ranks with the torch.distributed transport for both halo directions
    (grid_neighbours + begin_exchange): four processes on the one GPU, the reassembled output bit-equal to the single lattice."""
    import torch.multiprocessing as mp
    L, seed, grid = (4, 4, 16, 8), 17, (2, 2)
    nz, nt = grid
    ctxmp = mp.get_context("spawn")
    q = ctxmp.Queue()
    port = 38900 + __import__("os").getpid() % 2000
    ps = [ctxmp.Process(target=_mp_worker_grid_dslash, args=(r, grid, port, L, seed, q)) for r in range(nz * nt)]
    for p in ps:
        p.start()
    try:
        parts = q.get(timeout=200)
        for p in ps:
            p.join(timeout=120)
            assert p.exitcode == 0
    finally:
        for p in ps:
            if p.is_alive():
                p.kill()
    Lz_loc, Lt_loc, HLy = L[2] // nz, L[3] // nt, L[0] // 2 * L[1]
    got = np.zeros((2, L[3], L[2], HLy, 3), dtype=np.complex128)
    for r, part in enumerate(parts):
        rz, rt = r % nz, r // nz
        got[:, rt * Lt_loc:(rt + 1) * Lt_loc, rz * Lz_loc:(rz + 1) * Lz_loc] = part
    ctx = binding.Hisq(L, "fp64", 2)
    ctx.set_links(*binding.make_links(L, seed, ctx.device))
    one = ctx.unpack(ctx.dslash(ctx.pack(binding.make_sources(L, seed + 1, 2, 0, ctx.device)), 1)).cpu().numpy()
    ctx.close()
    assert np.array_equal(got.reshape(2, -1, 3), one)
