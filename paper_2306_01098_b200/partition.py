"""Row f3, first step: the Dslash on a lattice partitioned along t over several ranks (one process per GPU), the
paper's sub-lattice + halo scheme (Eq. (6)/(7)).  The kernels and the halo pack / unpack
are in libhisq (hisq_create_part, hisq_halo_pack, hisq_halo_unpack); this module is the plumbing around them:
which global sites a rank's extended lattice holds, and the neighbour exchange through torch.distributed
(NCCL on GPUs, gloo in the CPU test).  No method arithmetic here."""
from __future__ import annotations

from typing import Sequence

import torch

from . import inputs, layout

HALO_T = 4
HOP_MAX = 3   # reach of the stencil along one direction (Naik term)


def grid_of(nranks):
    """nranks = an int (cut along t only) or a pair (nz, nt) (cut along z and t; rank = rz + nz * rt) -> (nz, nt)."""
    return (1, int(nranks)) if isinstance(nranks, int) else (int(nranks[0]), int(nranks[1]))


def extended_lattice(L: Sequence[int], nranks):
    nz, nt = grid_of(nranks)
    return (int(L[0]), int(L[1]), int(L[2]) // nz + (2 * HALO_T if nz > 1 else 0), int(L[3]) // nt + 2 * HALO_T)


def owned_box(L: Sequence[int], nranks):
    """(z_lo, z_cnt, t_lo, t_cnt): the owned planes / slices inside the extended local lattice."""
    nz, nt = grid_of(nranks)
    return (HALO_T if nz > 1 else 0, int(L[2]) // nz, HALO_T, int(L[3]) // nt)


def global_sites_of_rank(L: Sequence[int], rank: int, nranks, device="cpu") -> torch.Tensor:
    """For every memory index eo of rank's EXTENDED lattice (Eq. 4 on that lattice), the GLOBAL lexicographic site
    it is a copy of (halo slices / planes wrap around the global lattice)."""
    nz, nt = grid_of(nranks)
    rz, rt = rank % nz, rank // nz
    Le = extended_lattice(L, nranks)
    lex = layout.lex_of_eo(Le, device=device)
    x = lex % Le[0]
    r = lex // Le[0]
    y = r % Le[1]
    r = r // Le[1]
    z = r % Le[2]
    t = r // Le[2]
    tg = (rt * (L[3] // nt) + t - HALO_T) % L[3]
    zg = (rz * (L[2] // nz) + z - HALO_T) % L[2] if nz > 1 else z
    return x + L[0] * (y + L[1] * (zg + L[2] * tg))


def interior(ctx, L: Sequence[int], nranks, canonical: torch.Tensor) -> torch.Tensor:
    """The owned sites of a CANONICAL half-lattice field [n, Vh_ext, 3] of a partitioned context, as [n, t_cnt, z_cnt, H*Ly, 3]."""
    Le = extended_lattice(L, nranks)
    z_lo, z_cnt, t_lo, t_cnt = owned_box(L, nranks)
    HLy = Le[0] // 2 * Le[1]
    v = canonical.view(canonical.shape[0], Le[3], Le[2], HLy, 3)
    return v[:, t_lo:t_lo + t_cnt, z_lo:z_lo + z_cnt]


def make_links_part(L, seed: int, rank: int, nranks, device, cdtype=torch.complex128, gen_device=None):
    """(fat, naik) canonical on rank's extended lattice: [4, V_ext, 3, 3]."""
    g = torch.device(gen_device) if gen_device is not None else torch.device("cpu")
    sites = global_sites_of_rank(L, rank, nranks, device=g)
    fat = inputs.fat_links(L, seed, sites).permute(1, 0, 2, 3).to(cdtype).contiguous().to(device)
    naik = inputs.naik_links(L, seed, sites).permute(1, 0, 2, 3).to(cdtype).contiguous().to(device)
    return fat, naik


def make_sources_part(L, seed: int, nrhs: int, parity: int, rank: int, nranks, device, cdtype=torch.complex128,
                      gen_device=None, fill_halo: bool = False):
    """Gaussian sources on one parity of rank's extended lattice, canonical [nrhs, Vh_ext, 3]; halo slices are zero
    unless fill_halo (they are what the exchange must deliver)."""
    g = torch.device(gen_device) if gen_device is not None else torch.device("cpu")
    Le = extended_lattice(L, nranks)
    Vh = layout.volume(Le) // 2
    sites = global_sites_of_rank(L, rank, nranks, device=g)[parity * Vh:(parity + 1) * Vh]
    src = inputs.sources(L, seed, sites, nrhs).to(cdtype)
    if not fill_halo:
        z_lo, z_cnt, t_lo, t_cnt = owned_box(L, nranks)
        v = src.view(nrhs, Le[3], Le[2], -1, 3)
        v[:, :t_lo] = 0
        v[:, t_lo + t_cnt:] = 0
        v[:, :, :z_lo] = 0
        v[:, :, z_lo + z_cnt:] = 0
    return src.contiguous().to(device)


class HaloExchange:
    """A halo exchange in flight (begin_exchange): finish() makes the received halos visible to the current stream."""

    def __init__(self, works=(), staged=None):
        self.works, self.staged = list(works), staged

    def finish(self):
        for w in self.works:
            w.wait()
        if self.staged is not None:
            for dst, src in self.staged:
                dst.copy_(src)
        self.works, self.staged = [], None


def grid_neighbours(rank: int, nranks):
    """Neighbours of `rank` on the nz x nt grid (rank = rz + nz * rt), periodic in both directions."""
    nz, nt = grid_of(nranks)
    rz, rt = rank % nz, rank // nz
    return {"t_down": rz + nz * ((rt - 1) % nt), "t_up": rz + nz * ((rt + 1) % nt),
            "z_down": (rz - 1) % nz + nz * rt, "z_up": (rz + 1) % nz + nz * rt}


def begin_exchange(send_lo: torch.Tensor, send_hi: torch.Tensor, recv_lo: torch.Tensor, recv_hi: torch.Tensor,
                   rank: int, nranks: int, dist=None, up=None, down=None, tag_base: int = 0) -> HaloExchange:
    """One direction of the halo exchange over a periodic ring: my send_hi goes to `up`'s recv_lo, my send_lo to `down`'s
    recv_hi.  up / down default to the ring of `nranks` ranks along t (rank +- 1); pass grid_neighbours(...) for a rank grid
    (tag_base keeps the messages of the two directions apart).
    dist = torch.distributed (initialised) or None for a single rank (own halos: periodic wrap onto itself).
    With NCCL the transfers are enqueued behind what the current stream holds so far (the pack kernel) and run on
    NCCL's own stream: kernels launched between begin_exchange and finish() overlap them.  Other backends (gloo: CPU
    tests, or processes sharing one GPU) go through the host and complete inside this call."""
    if up is None:
        up, down = (rank + 1) % nranks, (rank - 1) % nranks
    if dist is None or (up == rank and down == rank):
        recv_lo.copy_(send_hi)
        recv_hi.copy_(send_lo)
        return HaloExchange()
    stage = send_lo.is_cuda and dist.get_backend() != "nccl"
    # communicate as real arrays (not every backend knows complex dtypes)
    real = lambda t: torch.view_as_real(t) if t.is_complex() else t
    s_lo, s_hi = (real(send_lo.cpu()), real(send_hi.cpu())) if stage else (real(send_lo), real(send_hi))
    r_lo, r_hi = (torch.empty_like(s_lo), torch.empty_like(s_hi)) if stage else (real(recv_lo), real(recv_hi))
    staged = [(real(recv_lo), r_lo), (real(recv_hi), r_hi)] if stage else None
    if up == down and dist.get_backend() != "nccl":
        # both neighbours are the same peer: two tagged exchanges, lower rank sends first (no reliance on message order)
        for i, (snd, rcv) in enumerate(((s_hi, r_lo), (s_lo, r_hi))):
            if rank < up:
                dist.send(snd, up, tag=tag_base + i)
                dist.recv(rcv, up, tag=tag_base + i)
            else:
                dist.recv(rcv, up, tag=tag_base + i)
                dist.send(snd, up, tag=tag_base + i)
        return HaloExchange(staged=staged)
    # one grouped call: NCCL matches sends and receives between a pair of ranks in issue order, the same on both sides
    # (hi -> lo first, then lo -> hi), which also covers up == down
    ops = [dist.P2POp(dist.isend, s_hi, up, tag=tag_base), dist.P2POp(dist.irecv, r_lo, down, tag=tag_base),
           dist.P2POp(dist.isend, s_lo, down, tag=tag_base + 1), dist.P2POp(dist.irecv, r_hi, up, tag=tag_base + 1)]
    return HaloExchange(dist.batch_isend_irecv(ops), staged)


def exchange_halos(send_lo, send_hi, recv_lo, recv_hi, rank: int, nranks: int, dist=None):
    begin_exchange(send_lo, send_hi, recv_lo, recv_hi, rank, nranks, dist).finish()


def dslash_partitioned(ctx, field_in: torch.Tensor, parity: int, rank: int, nranks, dist=None, out=None,
                       overlap: bool = True, peer=None):
    """What one rank does per Dslash application: pack the halos of `field_in`, exchange them, compute.  nranks: an int (cut
    along t) or (nz, nt).  overlap (t cut only): the owned slices that read no halo are computed while the exchange is in
    flight, the first and last 3 afterwards (hisq_dslash_slices; PAPER.md:340-348 'communication hidden behind computation')."""
    n = field_in.shape[0]
    nz, nt = grid_of(nranks)
    if peer is not None:             # PeerHalo: the pack kernels write into the neighbours' mailboxes (both directions)
        peer.send(field_in)
        arrive = lambda: peer.recv(field_in)
    else:
        nb = grid_neighbours(rank, nranks)
        slo, shi = ctx.halo_buffers(n)
        rlo, rhi = ctx.halo_buffers(n)
        ctx.halo_pack(field_in, slo, shi)
        ex = begin_exchange(slo, shi, rlo, rhi, rank, nt, dist, up=nb["t_up"], down=nb["t_down"])
        exz = None
        if nz > 1:
            zslo, zshi = ctx.zhalo_buffers(n)
            zrlo, zrhi = ctx.zhalo_buffers(n)
            ctx.zhalo_pack(field_in, zslo, zshi)
            exz = begin_exchange(zslo, zshi, zrlo, zrhi, rank, nz, dist, up=nb["z_up"], down=nb["z_down"], tag_base=2)

        def arrive():
            ex.finish()
            ctx.halo_unpack(field_in, rlo, rhi)
            if exz is not None:
                exz.finish()
                ctx.zhalo_unpack(field_in, zrlo, zrhi)
    t_cnt = ctx.L[3] - 2 * HALO_T
    if not overlap or nz > 1 or t_cnt <= 2 * HOP_MAX:
        arrive()
        return ctx.dslash(field_in, parity, out=out)
    if out is None:
        out = ctx.new_field(n)
    ctx.dslash_slices(field_in, parity, out, HOP_MAX, t_cnt - 2 * HOP_MAX)
    arrive()
    ctx.dslash_edges(field_in, parity, out, HOP_MAX)
    return out


class PeerHalo:
    """Halo exchange through mailboxes in peer-mapped device memory (include/hisq.h, hisq_peer_*): the packing kernel
    stores straight into the neighbours' memory over NVLink and stream memory operations do the signalling -- no
    communication-library call on the data path.  This class is the plumbing: it allocates this rank's mailbox,
    hands a CUDA IPC mapping of it to the other ranks of the node (through `dist`'s object collectives; one process per
    GPU) and attaches all ranks' mappings to the context (t-neighbours for the halos, everybody for the all-reduce).  dist = None or one rank: the ring closes on itself."""

    def __init__(self, ctx, rank: int, nranks: int, nrhs: int, dist=None):
        self.ctx, self.dist, self.nranks = ctx, dist, nranks
        self.mine = ctx.peer_mailbox(nrhs)
        torch.cuda.synchronize(ctx.device)          # zeroed before anybody can see it
        boxes = [self.mine] * nranks
        if nranks > 1 and dist is not None:
            from torch.multiprocessing.reductions import reduce_tensor
            shared = [None] * nranks
            dist.all_gather_object(shared, reduce_tensor(self.mine))
            for r in range(nranks):
                if r == rank:
                    continue
                rebuild, args = shared[r]
                boxes[r] = rebuild(*args)
                if boxes[r].device != ctx.device:
                    # a first copy makes torch enable peer access from this GPU to the owner's (kernels need it too)
                    torch.empty(1, dtype=torch.uint8, device=ctx.device).copy_(boxes[r][:1])
        ctx.peer_attach(boxes, nrhs)
        self._barrier()

    def _barrier(self):
        torch.cuda.synchronize(self.ctx.device)
        if self.dist is not None and self.nranks > 1:
            self.dist.barrier()

    def send(self, field):
        self.ctx.halo_send(field)

    def recv(self, field):
        self.ctx.halo_recv(field)

    def allreduce(self, which: int, nrhs: int):
        """Sum over ranks of a CG state array (hisq_cgp_ptr numbering), in place, on the context's stream."""
        self.ctx.peer_reduce_send(which, nrhs)
        self.ctx.peer_reduce_recv(which, nrhs)

    def close(self):
        """Collective: nobody frees a mailbox a neighbour may still be writing to."""
        self._barrier()
        self.ctx._mailboxes = None
        self.mine = None


class PartitionedCG:
    """TEST SCAFFOLD, not the product path: one rank's side of the multi-RHS CG on a t-partitioned lattice sequenced from
    Python over the phase-wise calls (include/hisq.h, hisq_cgp_*), so that the phases can be checked one by one and ranks
    can be emulated in lockstep inside one process.  The product is hisq_cg on a partitioned context, which drives the
    same phases from C with every cross-rank step on the stream (hisq.cu, cgp_solve).  Every kernel is the library's;
    this class only sequences the phases and performs the two cross-rank steps between them -- halo exchange of a field
    and all-reduce of nrhs doubles -- through `dist` (torch.distributed: NCCL between GPUs).  t cut only."""

    def __init__(self, ctx, rank: int, nranks: int, dist=None, peer: "PeerHalo | None" = None):
        """peer: move the halos AND the all-reduces of the scalar products through peer-mapped mailboxes (PeerHalo)
        instead of `dist`: the iteration then runs without a communication-library call and without a host sync
        between status polls."""
        self.ctx, self.rank, self.nranks, self.dist, self.peer = ctx, rank, nranks, dist, peer

    def _halo_begin(self, field):
        if self.peer is not None:
            self.peer.send(field)
            return None
        n = field.shape[0]
        slo, shi = self.ctx.halo_buffers(n)
        rlo, rhi = self.ctx.halo_buffers(n)
        self.ctx.halo_pack(field, slo, shi)
        return begin_exchange(slo, shi, rlo, rhi, self.rank, self.nranks, self.dist), rlo, rhi

    def _halo_end(self, field, pending):
        if self.peer is not None:
            self.peer.recv(field)
            return
        ex, rlo, rhi = pending
        ex.finish()
        self.ctx.halo_unpack(field, rlo, rhi)

    def _allreduce(self, t, which=None):
        if self.peer is not None and which is not None:
            self.peer.allreduce(which, t.shape[0])
        elif self.dist is not None and self.nranks > 1:
            if t.is_cuda and self.dist.get_backend() != "nccl":
                h = t.cpu()
                self.dist.all_reduce(h, op=self.dist.ReduceOp.SUM)
                t.copy_(h)
            else:
                self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)

    def solve(self, b, mass: float, tol: float, x=None, check_every: int = 16, max_iter: int = 100000,
              overlap: bool = True):
        """overlap: each Dslash is split (phases 20/21, 30/31) so that the slices reading no halo run while the halo
        exchange is in flight; the iterates are bit-identical to the unsplit phases 2, 3."""
        c = self.ctx
        n = b.shape[0]
        if x is None:
            x = c.new_field(n)
        p, t = c.cgp_tensor(0, n), c.cgp_tensor(1, n)
        rho, pq, sums = c.cgp_tensor(2, n), c.cgp_tensor(3, n), c.cgp_tensor(4, n)
        c.cgp_begin(x, b, tol)
        self._allreduce(rho, 2)
        c.cgp_phase(0, mass)
        st = c.cgp_status(n)
        while not st["done"] and st["iterations"] < max_iter:
            for _ in range(check_every):
                c.cgp_phase(1, mass)
                pend = self._halo_begin(p)
                if overlap:
                    c.cgp_phase(20, mass)
                    self._halo_end(p, pend)
                    c.cgp_phase(21, mass)
                else:
                    self._halo_end(p, pend)
                    c.cgp_phase(2, mass)
                pend = self._halo_begin(t)
                if overlap:
                    c.cgp_phase(30, mass)
                    self._halo_end(t, pend)
                    c.cgp_phase(31, mass)
                else:
                    self._halo_end(t, pend)
                    c.cgp_phase(3, mass)
                self._allreduce(pq, 3)
                c.cgp_phase(4, mass)
                self._allreduce(sums, 4)
                c.cgp_phase(5, mass)
            st = c.cgp_status(n)
        return x, st
