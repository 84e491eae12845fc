// hisq.cu -- the C ABI of libhisq (include/hisq.h): context, workspace, link repack, Dslash dispatch,
// multi-RHS CG drivers (fp32 / fp64 / mixed with fp64 reliable updates).  sm_100a only; no CPU path.
#include "../../include/hisq.h"

#include <cuda.h>   // types of the stream memory operations only: the entry points are looked up at run time, libcuda is not linked

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "blas.cuh"
#include "dslash_launch.cuh"
#include "links.cuh"
#include "smear.cuh"

using namespace hisq;

struct hisq_ctx {
    Geom g;
    int prec;
    cudaStream_t stream;
    cudaStream_t cap_stream;   // private stream used only to CAPTURE graphs (the legacy stream cannot be captured)
    // workspace carve-up (all device pointers into the caller's buffer)
    char* ws;
    size_t ws_bytes;
    int ws_nrhs;           // RHS capacity of the CG / staging part
    double* links64;       // internal fp64 links (FP64, MIXED)
    float* links32;        // internal fp32 links (FP32, MIXED)
    CgState* state;
    double* partial;       // reduction partials [kMaxNrhs][partial_cols]
    double* true_rr;       // [kMaxNrhs] device
    size_t partial_cols;
    char* fields;          // CG temporaries
    char* stage;           // host-call staging (2 canonical + 2 native fields)
    bool have_links;
    bool naik_c14;         // Naik links currently stored compressed
    int naik_compress;     // option: try to compress at the next hisq_set_links
    int fused_blas;        // option: cooperative fused x/r/p update for small fields
    void* cgp_x; int cgp_nrhs; double cgp_tol;   // phase-wise CG on partitioned lattices
    int work_prec;         // precision the phase-wise / halo calls operate in: prec, except inside a HISQ_MIXED multi-rank
                           // solve, which switches between the fp32 iteration and the fp64 reliable update
    // peer-memory halo transport (hisq_peer_attach): mailboxes of this rank and of its t-neighbours, exchange counters
    int part_rank, part_nranks, part_nz, part_nt;
    char *mbox, *mbox_up, *mbox_down, *mbox_zup, *mbox_zdown;
    size_t mbox_zbuf;      // bytes of one z-halo buffer inside a mailbox
    PeerBoxes mbox_all;    // every rank's mailbox (all-reduce)
    PeerBoxes* d_boxes;    // the same table in device memory (kernels that push their sums themselves)
    // set by cgp_solve around the phases whose kernels push / read the cross-rank sums themselves; all null otherwise
    PeerPush fuse_push_pq, fuse_push_sums;
    const double *fuse_red_pq, *fuse_red_sums;
    size_t mbox_buf;       // bytes of one halo buffer inside a mailbox
    int mbox_nrhs;
    unsigned seq_send, seq_recv, red_send, red_recv;
    cudaStream_t abort_stream;   // the abort kernel must not queue behind a stream that is itself waiting for a peer
    int num_sms;
    unsigned long long* bad_count;  // device counter used by the compression check
    // options
    int max_iter, reliable_interval, check_interval, use_graph, nrhs_inner, tile_y, tile_z, overlap_opt, dot_fp64;
    double window_mb;
    // info of the last solve
    int info_iters, info_reliable;
    double info_relres[kMaxNrhs];
    LaunchStats stats;
    // instantiated CUDA graphs of a batch of CG iterations, kept across solves (capture + instantiate is a visible share of
    // a small solve: C1 is ~500 iterations of ~20 us).  A graph bakes in every kernel argument, so it is reused only if
    // they all match; `epoch` changes whenever the workspace, the links or an option change.
    struct GraphKey { const void* x; double m2; int nrhs, batch, keep, kind, wsize; unsigned long long epoch; };
    struct CachedGraph {
        cudaGraphExec_t exec; long long launches; GraphKey key;
        bool matches(const GraphKey& k) const
        {
            return exec && key.x == k.x && key.m2 == k.m2 && key.nrhs == k.nrhs && key.batch == k.batch && key.keep == k.keep &&
                   key.kind == k.kind && key.wsize == k.wsize && key.epoch == k.epoch;
        }
    };
    CachedGraph cg_graph[2], ms_graph;
    unsigned long long epoch;
    CgState* host_state;   // pinned: slot 0 (also the synchronous poll target) and slot 1, each followed by true_rr
    cudaEvent_t poll_ev[2];
    std::string last_error;
};

static constexpr size_t kPollSlot = (sizeof(CgState) + kMaxNrhs * sizeof(double) + 255) / 256 * 256;
static size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }
static size_t elem_size(int prec) { return prec == HISQ_FP32 ? 4 : 8; }

static int cuda_fail(hisq_ctx* h, cudaError_t e, const char* where)
{
    h->last_error = std::string(where) + ": " + cudaGetErrorString(e);
    return HISQ_ECUDA;
}
#define CK(call)                                                      \
    do {                                                              \
        cudaError_t e_ = (call);                                      \
        if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);        \
    } while (0)

// ---- CTA sweep order: (ty, tz) so that the 7 t-slices an in-flight output slice gathers from fit in L2 ----
static void choose_tiles(hisq_ctx* h, int nrhs, size_t w)
{
    Geom& g = h->g;
    const int Lz = g.z_cnt;   // the owned z planes (all of them unless the lattice is cut along z)
    int ty = g.L[1], tz = Lz;
    if (h->tile_y > 0 && g.L[1] % h->tile_y == 0) ty = h->tile_y;
    if (h->tile_z > 0 && Lz % h->tile_z == 0) tz = h->tile_z;
    if (h->tile_y <= 0 && h->tile_z <= 0) {
        const double target = h->window_mb * 1e6;
        const double per_site = 6.0 * nrhs * (double)w;
        double best_cost = 1e300;
        for (int cy = 4; cy <= g.L[1]; ++cy) {
            if (g.L[1] % cy) continue;
            for (int cz = 4; cz <= Lz; ++cz) {
                if (Lz % cz) continue;
                const double window = 7.0 * g.H * cy * cz * per_site;
                const double halo = (cy == g.L[1] ? 1.0 : (cy + 6.0) / cy) * (cz == Lz ? 1.0 : (cz + 6.0) / cz);
                double cost = halo + (window > target ? 100.0 * window / target : 0.0) - 1e-9 * cy * cz;
                if (cost < best_cost) { best_cost = cost; ty = cy; tz = cz; }
            }
        }
    }
    g.ty = ty; g.tz = tz; g.nty = g.L[1] / ty; g.ntz = Lz / tz;
}

extern "C" int hisq_create(hisq_ctx** out, int Lx, int Ly, int Lz, int Lt, int prec)
{
    if (!out) return HISQ_EINVAL;
    *out = nullptr;
    const int L[4] = { Lx, Ly, Lz, Lt };
    for (int i = 0; i < 4; ++i)
        if (L[i] < 4 || (L[i] & 1)) return HISQ_EINVAL;
    if (prec != HISQ_FP32 && prec != HISQ_FP64 && prec != HISQ_MIXED) return HISQ_EINVAL;
    const long long V = (long long)Lx * Ly * Lz * Lt;
    if (V / 2 > 0x3fffffffLL) return HISQ_EINVAL;  // half-index must fit comfortably in int
    hisq_ctx* h = new (std::nothrow) hisq_ctx();
    if (!h) return HISQ_EINVAL;
    for (int i = 0; i < 4; ++i) h->g.L[i] = L[i];
    h->g.H = Lx / 2;
    h->g.Vh = (int)(V / 2);
    h->g.sy = h->g.H; h->g.sz = h->g.H * Ly; h->g.st = h->g.H * Ly * Lz;
    h->g.stride[0] = 1; h->g.stride[1] = h->g.sy; h->g.stride[2] = h->g.sz; h->g.stride[3] = h->g.st;
    h->g.ty = Ly; h->g.tz = Lz; h->g.nty = 1; h->g.ntz = 1;
    h->g.part = 0; h->g.t_lo = 0; h->g.t_cnt = Lt; h->g.flip_lo = 1; h->g.flip_hi = 1;
    h->g.zpart = 0; h->g.z_lo = 0; h->g.z_cnt = Lz;
    h->prec = prec;
    h->stream = 0;
    h->cap_stream = nullptr;
    h->ws = nullptr; h->ws_bytes = 0; h->ws_nrhs = 0;
    h->links64 = nullptr; h->links32 = nullptr; h->have_links = false;
    h->max_iter = 100000;
    h->reliable_interval = prec == HISQ_MIXED ? 100 : 0;
    h->check_interval = 32;
    h->use_graph = 1;
    h->nrhs_inner = 0;
    h->naik_c14 = false; h->naik_compress = 0; h->bad_count = nullptr;
    h->fused_blas = 1; h->num_sms = 0; h->overlap_opt = -1; h->dot_fp64 = -1;
    h->cgp_x = nullptr; h->cgp_nrhs = 0; h->cgp_tol = 0.0;
    h->work_prec = prec == HISQ_MIXED ? HISQ_FP64 : prec;
    h->abort_stream = nullptr;
    { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev); }
    h->tile_y = 0; h->tile_z = 0;
    h->window_mb = 20.0;   // measured on C5 and C3: 10-20 MB windows are 2-3 % faster than 40, 10 % faster than none
    h->info_iters = 0; h->info_reliable = 0;
    for (int k = 0; k < kMaxNrhs; ++k) h->info_relres[k] = 0.0;
    h->cg_graph[0].exec = h->cg_graph[1].exec = h->ms_graph.exec = nullptr;
    h->epoch = 1;
    h->host_state = nullptr;
    if (cudaHostAlloc((void**)&h->host_state, 2 * kPollSlot, cudaHostAllocDefault) != cudaSuccess) {
        delete h;
        return HISQ_ECUDA;
    }
    h->poll_ev[0] = h->poll_ev[1] = nullptr;
    cudaEventCreateWithFlags(&h->poll_ev[0], cudaEventDisableTiming);
    cudaEventCreateWithFlags(&h->poll_ev[1], cudaEventDisableTiming);
    *out = h;
    return HISQ_OK;
}

// Row f3: one rank's share of a lattice partitioned along t (the paper's sub-lattice + halo scheme, PAPER.md:187-191,
// Eq. (6)/(7) :467-488).  The context lives on the EXTENDED local lattice Lx x Ly x Lz x (Lt/nranks + 2*kHaloT).
static const int kHopMax = 3;  // reach of the stencil in one direction (Naik term)
static const int kHaloT = 4;   // halo slices on each side: 3 are needed (Naik reach), 4 keeps site parity = global parity
// rank = rz + nz * rt on an nz x nt grid of ranks: the lattice is cut into nz parts along z and nt along t.  nz = 1 leaves z
// whole (periodic on every rank, no z halo); the t direction always carries halos (nt = 1: the ring closes on the rank).
extern "C" int hisq_create_part2(hisq_ctx** out, int Lx, int Ly, int Lz_global, int Lt_global, int prec, int rank, int nz, int nt)
{
    if (!out || nz < 1 || nt < 1 || nz * nt > kMaxRanks || rank < 0 || rank >= nz * nt || Lt_global % nt || Lz_global % nz) return HISQ_EINVAL;
    const int Lt_loc = Lt_global / nt, Lz_loc = Lz_global / nz;
    if (Lt_loc < 4 || (Lt_loc & 1)) return HISQ_EINVAL;   // even (parity) and >= 3 (halo comes from the nearest rank only)
    if (nz > 1 && (Lz_loc < 4 || (Lz_loc & 1))) return HISQ_EINVAL;
    int rc = hisq_create(out, Lx, Ly, Lz_loc + (nz > 1 ? 2 * kHaloT : 0), Lt_loc + 2 * kHaloT, prec);
    if (rc != HISQ_OK) return rc;
    Geom& g = (*out)->g;
    const int rz = rank % nz, rt = rank / nz;
    g.part = 1; g.t_lo = kHaloT; g.t_cnt = Lt_loc;
    g.flip_lo = rt == 0; g.flip_hi = rt == nt - 1;
    if (nz > 1) { g.zpart = 1; g.z_lo = kHaloT; g.z_cnt = Lz_loc; }
    (*out)->part_rank = rank; (*out)->part_nranks = nz * nt; (*out)->part_nz = nz; (*out)->part_nt = nt;
    return HISQ_OK;
}
extern "C" int hisq_create_part(hisq_ctx** out, int Lx, int Ly, int Lz, int Lt_global, int prec, int rank, int nranks)
{
    return hisq_create_part2(out, Lx, Ly, Lz, Lt_global, prec, rank, 1, nranks);
}

static void drop_graphs(hisq_ctx* h)
{
    hisq_ctx::CachedGraph* g[3] = { &h->cg_graph[0], &h->cg_graph[1], &h->ms_graph };
    for (int i = 0; i < 3; ++i)
        if (g[i]->exec) { cudaGraphExecDestroy(g[i]->exec); g[i]->exec = nullptr; }
    h->epoch++;
}

extern "C" int hisq_destroy(hisq_ctx* h)
{
    if (!h) return HISQ_EINVAL;
    drop_graphs(h);
    if (h->host_state) cudaFreeHost(h->host_state);
    if (h->d_boxes) cudaFree(h->d_boxes);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->abort_stream) cudaStreamDestroy(h->abort_stream);
    for (int i = 0; i < 2; ++i) if (h->poll_ev[i]) cudaEventDestroy(h->poll_ev[i]);
    delete h;
    return HISQ_OK;
}

extern "C" int hisq_set_stream(hisq_ctx* h, void* s)
{
    if (!h) return HISQ_EINVAL;
    drop_graphs(h);
    h->stream = (cudaStream_t)s;
    return HISQ_OK;
}

// ---- workspace layout ---------------------------------------------------------------------------
struct WsLayout {
    size_t links64, links32, state, true_rr, partial, fields, stage, total, partial_cols;
};

static size_t field_bytes(const hisq_ctx* h, int nrhs, size_t w) { return align_up((size_t)nrhs * 6 * h->g.Vh * w); }
// records per parity of the internal link layout (dslash.cuh): blocks of 32 half-indices, one spare block because a warp
// of a run that does not start on a multiple of 32 reads (and discards) the block's other lanes
static size_t link_blocks(const hisq_ctx* h) { return ((size_t)h->g.Vh + 31) / 32 + 1; }
static size_t link_bytes(const hisq_ctx* h, size_t w) { return align_up(2 * link_blocks(h) * 16 * 18 * 32 * w); }

static WsLayout ws_layout(const hisq_ctx* h, int nrhs)
{
    WsLayout l;
    size_t off = 0;
    l.links64 = off;
    if (h->prec != HISQ_FP32) off += link_bytes(h, 8);
    l.links32 = off;
    if (h->prec != HISQ_FP64) off += link_bytes(h, 4);
    l.state = off; off += align_up(sizeof(CgState));
    l.true_rr = off; off += align_up(kMaxNrhs * sizeof(double) + 64);   // + the compression check counter
    // columns: enough for the Dslash epilogue (one per CTA and chunk-slot) and the BLAS kernels
    size_t cols_d = ((size_t)h->g.Vh / 64 + (size_t)h->g.L[3] * h->g.L[1] * h->g.L[2] / 16 + 64);
    size_t cols_b = (size_t)blas_grid_x((size_t)6 * h->g.Vh, 2) + init_grid_x((size_t)6 * h->g.Vh) + 64 + 4096;
    l.partial_cols = cols_d > cols_b ? cols_d : cols_b;
    l.partial = off; off += align_up((size_t)kMaxNrhs * l.partial_cols * sizeof(double));
    l.fields = off;
    if (h->prec == HISQ_FP64) off += 4 * field_bytes(h, nrhs, 8);                            // r p q t
    else if (h->prec == HISQ_FP32) off += 4 * field_bytes(h, nrhs, 4);
    else off += 5 * field_bytes(h, nrhs, 4) + 2 * field_bytes(h, nrhs, 8);                   // r p q t xlo | rhi thi
    l.stage = off;
    off += 4 * field_bytes(h, nrhs, elem_size(h->prec));
    l.total = off;
    return l;
}

extern "C" size_t hisq_workspace_bytes(const hisq_ctx* h, int nrhs)
{
    if (!h || nrhs < 1 || nrhs > HISQ_MAX_NRHS) return 0;
    return ws_layout(h, nrhs).total;
}

extern "C" int hisq_set_workspace(hisq_ctx* h, void* p, size_t bytes)
{
    if (!h || !p || ((uintptr_t)p & 255)) return HISQ_EINVAL;
    int nrhs = 0;
    for (int n = HISQ_MAX_NRHS; n >= 1; --n)
        if (ws_layout(h, n).total <= bytes) { nrhs = n; break; }
    if (nrhs == 0) return HISQ_ENOWORKSPACE;
    WsLayout l = ws_layout(h, nrhs);
    h->ws = (char*)p; h->ws_bytes = bytes; h->ws_nrhs = nrhs;
    h->links64 = h->prec != HISQ_FP32 ? (double*)(h->ws + l.links64) : nullptr;
    h->links32 = h->prec != HISQ_FP64 ? (float*)(h->ws + l.links32) : nullptr;
    h->state = (CgState*)(h->ws + l.state);
    h->true_rr = (double*)(h->ws + l.true_rr);
    h->bad_count = (unsigned long long*)(h->ws + l.true_rr + kMaxNrhs * sizeof(double));
    h->partial = (double*)(h->ws + l.partial);
    h->partial_cols = l.partial_cols;
    h->fields = h->ws + l.fields;
    h->stage = h->ws + l.stage;
    h->have_links = false;
    drop_graphs(h);
    CK(cudaMemsetAsync(h->state, 0, sizeof(CgState), h->stream));
    return HISQ_OK;
}

template <typename TS, typename TD>
static void enqueue_link_records(hisq_ctx* h, const void* fat, const void* naik, TD* dst, bool c14)
{
    const size_t V = (size_t)2 * h->g.Vh;
    const unsigned grid = (unsigned)((4 * V + 255) / 256);
    if (c14) link_record_kernel<TS, TD, true><<<grid, 256, 0, h->stream>>>((const TS*)fat, (const TS*)naik, dst, h->g, link_blocks(h));
    else link_record_kernel<TS, TD, false><<<grid, 256, 0, h->stream>>>((const TS*)fat, (const TS*)naik, dst, h->g, link_blocks(h));
    h->stats.launches++;
}

extern "C" int hisq_set_links(hisq_ctx* h, const void* fat, const void* naik)
{
    if (!h || !fat || !naik || ((uintptr_t)fat & 15) || ((uintptr_t)naik & 15)) return HISQ_EINVAL;
    if (!h->ws) return HISQ_ENOWORKSPACE;
    const int Vh = h->g.Vh;
    const size_t V = (size_t)2 * Vh;
    h->naik_c14 = false;
    drop_graphs(h);
    if (h->naik_compress) {
        // row f2: the 14-real format for the Naik links is used only if EVERY link is reproduced from it
        // (|row2 - conj(row0 x row1) d| <= tol |row0|) in every precision the context keeps; otherwise all stay uncompressed
        const unsigned grid = (unsigned)((4 * V + 255) / 256);
        CK(cudaMemsetAsync(h->bad_count, 0, sizeof(unsigned long long), h->stream));
        if (h->prec == HISQ_FP32) naik_check_kernel<float><<<grid, 256, 0, h->stream>>>((const float*)naik, Vh, 1e-5, 0.0, h->bad_count);
        else naik_check_kernel<double><<<grid, 256, 0, h->stream>>>((const double*)naik, Vh, 1e-12, h->prec == HISQ_MIXED ? 1e-5 : 0.0, h->bad_count);
        h->stats.launches++;
        unsigned long long bad = 1;
        CK(cudaMemcpyAsync(&bad, h->bad_count, sizeof(bad), cudaMemcpyDeviceToHost, h->stream));
        CK(cudaStreamSynchronize(h->stream));
        if (bad == 0) h->naik_c14 = true;
        else h->last_error = "naik_compress: " + std::to_string(bad) + " Naik links are not a real multiple of a U(3) matrix; stored uncompressed";
    }
    if (h->prec == HISQ_FP32) {
        enqueue_link_records<float, float>(h, fat, naik, h->links32, h->naik_c14);
    } else {
        enqueue_link_records<double, double>(h, fat, naik, h->links64, h->naik_c14);
        if (h->prec == HISQ_MIXED) enqueue_link_records<double, float>(h, fat, naik, h->links32, h->naik_c14);
    }
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(h->stream));
    h->have_links = true;
    return HISQ_OK;
}

// ---- Dslash dispatch -----------------------------------------------------------------------------
static int default_inner_cap(int) { return 8; }  // measured: 8 RHS per thread beats 4 x 2 chunks in both precisions

template <typename T>
static int run_dslash(hisq_ctx* h, const T* links, T* out, const T* in, int parity, int nrhs, int mode, const T* u,
                      const T* v, double m2, double* result, const int* done, int ticket_slot, int t_first = 0,
                      int t_count = -1, int t_skip_at = 1 << 30, int t_skip = 0)
{
    choose_tiles(h, nrhs, sizeof(T));
    DslashArgs<T> a;
    a.g = h->g;
    a.links = links;
    a.nblk = link_blocks(h);
    a.in = in; a.out = out; a.u = u; a.v = v;
    a.partial = h->partial;
    a.ticket = &h->state->ticket[ticket_slot];
    a.result = result;
    a.done = done;
    a.m2 = m2;
    a.par = parity;
    a.k0 = 0; a.nrhs_total = nrhs; a.nchunks = 1; a.slab_blocks = 0; a.total_blocks = 0;
    a.nseg = a.seg_len = a.wps = a.merged = 0;
    a.wide_dot = h->dot_fp64;
    a.t0 = t_first; a.tn = t_count < 0 ? h->g.t_cnt - t_first : t_count;
    a.t_skip_at = t_skip_at; a.t_skip = t_skip;
    a.push = mode == MODE_APPLY_A ? h->fuse_push_pq : PeerPush();
    if (a.tn <= 0) return HISQ_OK;
    int cap = h->nrhs_inner > 0 ? h->nrhs_inner : default_inner_cap((int)sizeof(T));
    int e = launch_dslash<T>(a, mode, nrhs, cap, h->naik_c14, h->stream, &h->stats);
    if (e != 0) return cuda_fail(h, (cudaError_t)e, "dslash launch");
    return HISQ_OK;
}

static bool overlap(const void* a, const void* b, size_t bytes)
{
    const char* x = (const char*)a; const char* y = (const char*)b;
    return x < y + bytes && y < x + bytes;
}

extern "C" int hisq_dslash(hisq_ctx* h, void* out, const void* in, int parity, int nrhs)
{
    if (!h || !out || !in || nrhs < 1 || nrhs > HISQ_MAX_NRHS || (parity != 0 && parity != 1)) return HISQ_EINVAL;
    if (((uintptr_t)out & 15) || ((uintptr_t)in & 15)) return HISQ_EINVAL;
    if (!h->ws) return HISQ_ENOWORKSPACE;
    if (!h->have_links) return HISQ_ENOLINKS;
    const size_t bytes = (size_t)nrhs * 6 * h->g.Vh * elem_size(h->prec);
    if (overlap(out, in, bytes)) return HISQ_EINVAL;
    if (h->prec == HISQ_FP32)
        return run_dslash<float>(h, h->links32, (float*)out, (const float*)in, parity, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0,
                                 nullptr, nullptr, 2);
    return run_dslash<double>(h, h->links64, (double*)out, (const double*)in, parity, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0,
                              nullptr, nullptr, 2);
}

// hisq_dslash on some of the owned time slices only (the other slices of `out` are left untouched): `count` slices
// starting at `first`; with skip > 0 the slices from the skip_at-th on lie `skip` further up (two ranges, one launch).
static int dslash_some_slices(hisq_ctx* h, void* out, const void* in, int parity, int nrhs, int first, int count, int skip_at, int skip)
{
    if (!h || !out || !in || nrhs < 1 || nrhs > HISQ_MAX_NRHS || (parity != 0 && parity != 1)) return HISQ_EINVAL;
    if (first < 0 || count < 0 || skip < 0 || first + count + skip > h->g.t_cnt) return HISQ_EINVAL;
    if (((uintptr_t)out & 15) || ((uintptr_t)in & 15)) return HISQ_EINVAL;
    if (!h->ws) return HISQ_ENOWORKSPACE;
    if (!h->have_links) return HISQ_ENOLINKS;
    const size_t bytes = (size_t)nrhs * 6 * h->g.Vh * elem_size(h->prec);
    if (overlap(out, in, bytes)) return HISQ_EINVAL;
    if (count == 0) return HISQ_OK;
    if (h->prec == HISQ_FP32)
        return run_dslash<float>(h, h->links32, (float*)out, (const float*)in, parity, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0,
                                 nullptr, nullptr, 2, first, count, skip_at, skip);
    return run_dslash<double>(h, h->links64, (double*)out, (const double*)in, parity, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0,
                              nullptr, nullptr, 2, first, count, skip_at, skip);
}
extern "C" int hisq_dslash_slices(hisq_ctx* h, void* out, const void* in, int parity, int nrhs, int t_first, int t_count)
{
    return dslash_some_slices(h, out, in, parity, nrhs, t_first, t_count, 1 << 30, 0);
}
extern "C" int hisq_dslash_edges(hisq_ctx* h, void* out, const void* in, int parity, int nrhs, int width)
{
    if (!h || width < 0) return HISQ_EINVAL;
    const int n = h->g.t_cnt;
    if (2 * width >= n) return dslash_some_slices(h, out, in, parity, nrhs, 0, n, 1 << 30, 0);
    return dslash_some_slices(h, out, in, parity, nrhs, 0, 2 * width, width, n - 2 * width);
}

// out = (mass^2 - D_eo D_oe) in on even sites: the operator the solvers work on, as a call of its own (fused second
// Dslash: m^2 in - D_eo t and Re<in, out> in one kernel; the scalar products land in hisq_get_info-independent state).
extern "C" int hisq_apply_A(hisq_ctx* h, void* out, const void* in, double mass, int nrhs)
{
    if (!h || !out || !in || nrhs < 1 || nrhs > HISQ_MAX_NRHS || !std::isfinite(mass)) return HISQ_EINVAL;
    if (((uintptr_t)out & 15) || ((uintptr_t)in & 15)) return HISQ_EINVAL;
    if (!h->ws || nrhs > h->ws_nrhs) return HISQ_ENOWORKSPACE;
    if (!h->have_links) return HISQ_ENOLINKS;
    if (h->g.part) return HISQ_EINVAL;   // needs a halo exchange between the two hops: use the phase-wise calls
    const size_t bytes = (size_t)nrhs * 6 * h->g.Vh * elem_size(h->prec);
    if (overlap(out, in, bytes)) return HISQ_EINVAL;
    const size_t fb = field_bytes(h, h->ws_nrhs, elem_size(h->prec));
    void* t = h->fields + 3 * fb;
    int rc;
    if (h->prec == HISQ_FP32) {
        rc = run_dslash<float>(h, h->links32, (float*)t, (const float*)in, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, nullptr, 2);
        if (rc) return rc;
        return run_dslash<float>(h, h->links32, (float*)out, (const float*)t, HISQ_EVEN, nrhs, MODE_APPLY_A, (const float*)in, nullptr,
                                 mass * mass, h->state->sums, nullptr, 2);
    }
    rc = run_dslash<double>(h, h->links64, (double*)t, (const double*)in, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, nullptr, 2);
    if (rc) return rc;
    return run_dslash<double>(h, h->links64, (double*)out, (const double*)t, HISQ_EVEN, nrhs, MODE_APPLY_A, (const double*)in, nullptr,
                              mass * mass, h->state->sums, nullptr, 2);
}

// ---- CG --------------------------------------------------------------------------------------------
// One iteration (textbook Hestenes-Stiefel, independent scalars per RHS):
//   p = r + beta p ; t = D_oe p ; q = m^2 p - D_eo t , <p,q> ; x += alpha p , r -= alpha q , rho' = ||r||^2
static Span owned_span(const hisq_ctx* h, int vec_n)
{
    Span sp = { 0, 0, 0, 0, 0 };
    if (h->g.part) {   // vectors of vec_n reals; a plane is [Lt_ext][S] complex, the owned run starts at slice t_lo
        const size_t S = (size_t)h->g.Vh / h->g.L[3];
        sp.seg = 2 * S * h->g.t_cnt / vec_n; sp.plane = 2 * S * h->g.L[3] / vec_n; sp.off = 2 * S * h->g.t_lo / vec_n;
        if (h->g.zpart) {   // ... and inside every owned slice only the planes [z_lo, z_lo + z_cnt) are owned
            const size_t HLy = (size_t)h->g.H * h->g.L[1];
            sp.sub = 2 * HLy * h->g.z_cnt / vec_n; sp.sub_stride = 2 * S / vec_n;
            sp.seg = sp.sub * h->g.t_cnt;
            sp.off += 2 * HLy * h->g.z_lo / vec_n;
        }
    }
    return sp;
}
// x != nullptr: the pending x-update of the previous iteration rides in the same pass (blas.cuh); flush_only: only that
template <typename T>
static int enqueue_p_update(hisq_ctx* h, T* p, const T* r, int nrhs, T* x = nullptr, int flush_only = 0)
{
    const size_t nreal = (size_t)6 * h->g.Vh;
    const Span sp = owned_span(h, V16<T>::n);
    dim3 gb((unsigned)blas_grid_x(sp.seg ? 3 * sp.seg * V16<T>::n : nreal, V16<T>::n), (unsigned)nrhs);
    cg_update_p_kernel<T><<<gb, kBlasBlock, 0, h->stream>>>(p, r, nreal, h->state, sp, x, flush_only);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}

// Largest field for which the fused (cooperative) BLAS kernel applies: every thread keeps KEEP 16-byte vectors of
// r and p in registers across the grid barrier, and the whole grid must be co-resident.  Returns KEEP or 0.
template <typename T, int KEEP>
static int fused_blocks_per_sm()
{
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, cg_fused_update_kernel<T, KEEP>, kBlasBlock, 0) != cudaSuccess) return 0;
    return nb;
}
template <typename T>
static int fused_keep(hisq_ctx* h, int nrhs)
{
    if (!h->fused_blas) return 0;
    const size_t nvec = (size_t)6 * h->g.Vh / V16<T>::n;
    const int keeps[4] = { 1, 2, 4, 8 };
    for (int i = 0; i < 4; ++i) {
        const int keep = keeps[i];
        const size_t gx = (nvec + (size_t)kBlasBlock * keep - 1) / ((size_t)kBlasBlock * keep);
        int per_sm = keep == 1 ? fused_blocks_per_sm<T, 1>() : keep == 2 ? fused_blocks_per_sm<T, 2>()
                   : keep == 4 ? fused_blocks_per_sm<T, 4>() : fused_blocks_per_sm<T, 8>();
        if (gx * nrhs <= (size_t)per_sm * h->num_sms && gx <= h->partial_cols) return keep;
    }
    return 0;
}

template <typename T, int KEEP>
static cudaError_t launch_fused(hisq_ctx* h, T* x, T* r, T* p, const T* q, size_t nreal, int nrhs, int do_p)
{
    const size_t nvec = nreal / V16<T>::n;
    dim3 grid((unsigned)((nvec + (size_t)kBlasBlock * KEEP - 1) / ((size_t)kBlasBlock * KEEP)), (unsigned)nrhs);
    CgState* st = h->state;
    double* partial = h->partial;
    void* args[] = { &x, &r, &p, &q, &nreal, &st, &partial, &do_p };
    return cudaLaunchCooperativeKernel((void*)cg_fused_update_kernel<T, KEEP>, grid, dim3(kBlasBlock), args, 0, h->stream);
}

// keep = 0: the four-kernel iteration  [p = r + beta p] [D_oe] [D_eo + <p,Ap>] [x, r, rho'].
// keep > 0: the p-update of the NEXT iteration rides in the fused kernel: [D_oe] [D_eo + <p,Ap>] [x, r, rho' | p];
//           the caller launches one stand-alone p-update at the start and after every true-residual replacement.
template <typename T>
static int enqueue_iteration(hisq_ctx* h, const T* links, T* x, T* r, T* p, T* q, T* t, double m2, int nrhs, int keep = 0,
                             int do_p = 1)
{
    const size_t nreal = (size_t)6 * h->g.Vh;
    dim3 gb((unsigned)blas_grid_x(nreal, V16<T>::n), (unsigned)nrhs);
    int rc;
    if (keep == 0 && (rc = enqueue_p_update<T>(h, p, r, nrhs, x)) != HISQ_OK) return rc;
    rc = run_dslash<T>(h, links, t, p, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, &h->state->done, 2);
    if (rc) return rc;
    rc = run_dslash<T>(h, links, q, t, HISQ_EVEN, nrhs, MODE_APPLY_A, p, nullptr, m2, h->state->pq, &h->state->done, 2);
    if (rc) return rc;
    if (keep == 0) {
        // x is not touched here: its update is folded into the next iteration's p pass (or cg_solve's flush)
        // several chunks per CTA (blas.cuh: the dependent scalar loads at the head of a CTA and its reduction tail cost as
        // much as streaming one chunk), as long as >= 2 CTAs per SM remain; up to 8.  Measured on C4 (48^3 x 12, mixed,
        // n = 4): 57.8 us at one chunk per CTA, iteration 0.432 -> 0.412 ms with this rule (>= 16 CTAs per SM: no change there)
        int trips = (int)((size_t)gb.x * nrhs / ((size_t)h->num_sms * 2));
        trips = trips < 1 ? 1 : (trips > 8 ? 8 : trips);
        dim3 gt((gb.x + trips - 1) / trips, (unsigned)nrhs);
        cg_update_xr_kernel<T><<<gt, kBlasBlock, 0, h->stream>>>(x, r, p, q, nreal, h->state, h->partial, 0, PeerPush(), nullptr, Span(), 1, trips);
        CK(cudaGetLastError());
    } else {
        cudaError_t e = keep == 1 ? launch_fused<T, 1>(h, x, r, p, q, nreal, nrhs, do_p)
                      : keep == 2 ? launch_fused<T, 2>(h, x, r, p, q, nreal, nrhs, do_p)
                      : keep == 4 ? launch_fused<T, 4>(h, x, r, p, q, nreal, nrhs, do_p)
                                  : launch_fused<T, 8>(h, x, r, p, q, nreal, nrhs, do_p);
        if (e != cudaSuccess) return cuda_fail(h, e, "cudaLaunchCooperativeKernel");
    }
    h->stats.launches++;
    return HISQ_OK;
}

// r_out = b - A x in fp64-or-T, sums[k] = ||r_out_k||^2, then reliable-update bookkeeping.
template <typename T>
static int enqueue_true_residual(hisq_ctx* h, const T* links, T* r_out, const T* x, const T* b, T* t, double m2, int nrhs)
{
    int rc = run_dslash<T>(h, links, t, x, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, nullptr, 2);
    if (rc) return rc;
    rc = run_dslash<T>(h, links, r_out, t, HISQ_EVEN, nrhs, MODE_RESID, x, b, m2, h->state->sums, nullptr, 2);
    if (rc) return rc;
    cg_after_residual_kernel<<<1, 1, 0, h->stream>>>(h->state, h->true_rr);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}

static int poll_state(hisq_ctx* h)
{
    CK(cudaMemcpyAsync(h->host_state, h->state, sizeof(CgState), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaMemcpyAsync((char*)h->host_state + sizeof(CgState), h->true_rr, kMaxNrhs * sizeof(double), cudaMemcpyDeviceToHost,
                       h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return HISQ_OK;
}

// Asynchronous poll: copy the solver state into pinned slot `slot` and mark it with an event, so the host can
// enqueue the next batch before it looks at this one (a slow host then never idles the GPU).
static int poll_async(hisq_ctx* h, int slot)
{
    char* dst = (char*)h->host_state + (size_t)slot * kPollSlot;
    CK(cudaMemcpyAsync(dst, h->state, sizeof(CgState), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaEventRecord(h->poll_ev[slot], h->stream));
    return HISQ_OK;
}
static const CgState* poll_wait(hisq_ctx* h, int slot)
{
    if (cudaEventSynchronize(h->poll_ev[slot]) != cudaSuccess) return nullptr;
    return (const CgState*)((char*)h->host_state + (size_t)slot * kPollSlot);
}


template <typename T, typename TB>
static int cg_solve(hisq_ctx* h, const T* links, const double* links_hi, TB* x_user, const TB* b, double mass, double tol, int nrhs)
{
    constexpr bool MIXED = !std::is_same<T, TB>::value;
    const size_t nreal = (size_t)6 * h->g.Vh;
    const size_t total = nreal * nrhs;
    const double m2 = mass * mass;
    const size_t fb = field_bytes(h, h->ws_nrhs, sizeof(T));
    T* r = (T*)(h->fields);
    T* p = (T*)(h->fields + fb);
    T* q = (T*)(h->fields + 2 * fb);
    T* t = (T*)(h->fields + 3 * fb);
    T* x = MIXED ? (T*)(h->fields + 4 * fb) : (T*)x_user;
    TB* r_hi = MIXED ? (TB*)(h->fields + 5 * fb) : (TB*)r;
    TB* t_hi = MIXED ? (TB*)(h->fields + 5 * fb + field_bytes(h, h->ws_nrhs, sizeof(TB))) : (TB*)t;

    h->info_iters = 0; h->info_reliable = 0;
    // x = 0, p = 0, r = b, rho = ||b||^2
    CK(cudaMemsetAsync(x_user, 0, total * sizeof(TB), h->stream));
    if (MIXED) CK(cudaMemsetAsync(x, 0, total * sizeof(T), h->stream));
    CK(cudaMemsetAsync(p, 0, total * sizeof(T), h->stream));
    dim3 gi((unsigned)init_grid_x(nreal), (unsigned)nrhs);
    cg_init_kernel<TB, T><<<gi, kBlasBlock, 0, h->stream>>>(b, r, nreal, h->state, h->partial, tol, h->max_iter);
    h->stats.launches++;
    CK(cudaGetLastError());

    const int R = h->reliable_interval;
    int batch = h->check_interval > 0 ? h->check_interval : 32;
    if (R > 0) {
        int best = 1;
        for (int d = 1; d <= R && d <= batch; ++d)
            if (R % d == 0) best = d;
        batch = best;
    }
    const int keep = fused_keep<T>(h, nrhs);
    int rc = HISQ_OK;
    int status = HISQ_OK;
    int stagnation = 0;
    // enq_iter: iterations enqueued so far; rel_base: iteration count at the last true-residual replacement.  The
    // reliable-update schedule counts from rel_base, not from 0: when the recursion stops inside a batch (claimed
    // convergence not confirmed by the true residual) the solve resumes from an iteration count that is no multiple of
    // the batch, and a schedule tied to iter % R would never fire again.
    int enq_iter = 0, rel_base = 0, cur = 0;
    bool pending = false;
    double best_true[kMaxNrhs];
    for (int k = 0; k < kMaxNrhs; ++k) best_true[k] = 1e300;
    if (keep > 0 && (rc = enqueue_p_update<T>(h, p, r, nrhs)) != HISQ_OK) return rc;
    while (true) {
        // ---- a batch of iterations; the one that ends on a reliable-update boundary leaves p alone ----
        const int kind = (keep > 0 && R > 0 && (enq_iter - rel_base + batch) % R == 0) ? 1 : 0;
        if (h->use_graph) {
            hisq_ctx::CachedGraph& cg = h->cg_graph[kind];
            const hisq_ctx::GraphKey key = { (const void*)x, m2, nrhs, batch, keep, kind, (int)sizeof(T), h->epoch };
            if (!cg.matches(key)) {
                if (cg.exec) { cudaGraphExecDestroy(cg.exec); cg.exec = nullptr; }
                cudaGraph_t graph;
                const long long l0 = h->stats.launches;
                if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
                    rc = cuda_fail(h, cudaGetLastError(), "cudaStreamCreateWithFlags"); break;
                }
                cudaStream_t user_stream = h->stream;
                cudaError_t ce = cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal);
                if (ce != cudaSuccess) { rc = cuda_fail(h, ce, "cudaStreamBeginCapture"); break; }
                h->stream = h->cap_stream;
                for (int i = 0; i < batch && rc == HISQ_OK; ++i)
                    rc = enqueue_iteration<T>(h, links, x, r, p, q, t, m2, nrhs, keep, (kind == 1 && i == batch - 1) ? 0 : 1);
                h->stream = user_stream;
                ce = cudaStreamEndCapture(h->cap_stream, &graph);
                if (rc != HISQ_OK) { if (ce == cudaSuccess) cudaGraphDestroy(graph); break; }
                if (ce != cudaSuccess) { rc = cuda_fail(h, ce, "cudaStreamEndCapture"); break; }
                ce = cudaGraphInstantiate(&cg.exec, graph, 0);
                cudaGraphDestroy(graph);
                if (ce != cudaSuccess) { cg.exec = nullptr; rc = cuda_fail(h, ce, "cudaGraphInstantiate"); break; }
                cg.launches = h->stats.launches - l0;
                cg.key = key;
                h->stats.launches = l0;
            }
            cudaError_t ce = cudaGraphLaunch(cg.exec, h->stream);
            if (ce != cudaSuccess) { rc = cuda_fail(h, ce, "cudaGraphLaunch"); break; }
            h->stats.launches += cg.launches;
        } else {
            for (int i = 0; i < batch && rc == HISQ_OK; ++i)
                rc = enqueue_iteration<T>(h, links, x, r, p, q, t, m2, nrhs, keep, (kind == 1 && i == batch - 1) ? 0 : 1);
            if (rc != HISQ_OK) break;
        }
        // ---- look at the state, staying one batch ahead of the GPU whenever no reliable update is due ----
        enq_iter += batch;
        if ((rc = poll_async(h, cur)) != HISQ_OK) break;
        const bool boundary = R > 0 && (enq_iter - rel_base) % R == 0;
        const CgState* sp;
        if (!boundary && !pending) { pending = true; cur ^= 1; continue; }      // first batch of a run: just get ahead
        if (pending) {
            sp = poll_wait(h, cur ^ 1);                                             // the older batch
            if (sp && !sp->done && !sp->breakdown && !boundary) { cur ^= 1; continue; }   // newer poll stays in flight
            pending = false;
        }
        sp = poll_wait(h, cur);                                                    // newest state (stream drained up to it)
        if (!sp) { rc = cuda_fail(h, cudaGetLastError(), "cudaEventSynchronize"); break; }
        const CgState s = *sp;
        enq_iter = s.iter;
        h->info_iters = s.iter;
        if (s.breakdown) { status = HISQ_EBREAKDOWN; }
        const bool at_reliable = R > 0 && s.iter > rel_base && (s.iter - rel_base) % R == 0;
        if (!s.done && !at_reliable) continue;
        // ---- reliable update / final check: true residual in the high precision ----
        if (keep == 0 && (rc = enqueue_p_update<T>(h, p, r, nrhs, x, 1)) != HISQ_OK) break;   // the pending x += alpha p
        if (MIXED) {
            acc_xhi_kernel<<<(unsigned)((total / 4 + kBlasBlock - 1) / kBlasBlock + 1), kBlasBlock, 0, h->stream>>>(
                (double*)x_user, (float*)x, total);
            h->stats.launches++;
            rc = enqueue_true_residual<TB>(h, (const TB*)links_hi, r_hi, x_user, b, t_hi, m2, nrhs);
            if (rc) break;
            convert_kernel<TB, T><<<1184, kBlasBlock, 0, h->stream>>>(r_hi, r, total);
            h->stats.launches++;
        } else {
            rc = enqueue_true_residual<TB>(h, (const TB*)links, (TB*)r, x_user, b, (TB*)t, m2, nrhs);
            if (rc) break;
        }
        h->info_reliable++;
        rel_base = s.iter;
        if ((rc = poll_state(h)) != HISQ_OK) break;
        const CgState& s2 = *h->host_state;
        const double* trr = (const double*)((const char*)h->host_state + sizeof(CgState));
        for (int k = 0; k < nrhs; ++k)
            h->info_relres[k] = s2.bnorm2[k] > 0.0 ? std::sqrt(trr[k] / s2.bnorm2[k]) : 0.0;
        if (status == HISQ_EBREAKDOWN) break;
        if (s.done && !s2.done) {
            // the recursion said "converged", the true residual says no: resume, unless this keeps happening
            // without progress (tol below what this precision can reach)
            bool improved = false;
            for (int k = 0; k < nrhs; ++k)
                if (s2.active[k] && h->info_relres[k] < 0.9 * best_true[k]) { best_true[k] = h->info_relres[k]; improved = true; }
            stagnation = improved ? 0 : stagnation + 1;
            if (stagnation >= 3) { status = HISQ_ENOCONV; break; }
        }
        if (s2.done) {
            bool all = true;
            for (int k = 0; k < nrhs; ++k) all = all && !s2.active[k];
            if (!all) status = HISQ_ENOCONV;
            break;
        }
        if (keep > 0 && (rc = enqueue_p_update<T>(h, p, r, nrhs)) != HISQ_OK) break;   // p = r_true + beta p
    }
    if (rc != HISQ_OK) return rc;
    return status;
}

// ---- multi-shift CG (row f1): (A + sigma_k) x_k = b, one operator application per iteration -----------------
template <typename T>
static int ms_enqueue_iteration(hisq_ctx* h, const T* links, T* x, T* r, T* p, T* q, T* t, double m2_base, int kmin, int nshift)
{
    const size_t nreal = (size_t)6 * h->g.Vh;
    const unsigned gx = (unsigned)blas_grid_x(nreal, V16<T>::n);
    ms_update_p_kernel<T><<<dim3(gx, (unsigned)nshift), kBlasBlock, 0, h->stream>>>(p, r, nreal, h->state);
    h->stats.launches++;
    T* pb = p + (size_t)kmin * nreal;   // the base direction: the smallest shift has zeta = 1
    int rc = run_dslash<T>(h, links, t, pb, HISQ_ODD, 1, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, &h->state->done, 2);
    if (rc) return rc;
    rc = run_dslash<T>(h, links, q, t, HISQ_EVEN, 1, MODE_APPLY_A, pb, nullptr, m2_base, h->state->pq, &h->state->done, 2);
    if (rc) return rc;
    ms_update_xr_kernel<T><<<dim3(gx, (unsigned)nshift + 1), kBlasBlock, 0, h->stream>>>(x, r, p, q, nreal, h->state, h->partial);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}

template <typename T>
static int ms_solve(hisq_ctx* h, const T* links, T* x, const T* b, double mass, const double* shifts, int nshift, double tol)
{
    const size_t nreal = (size_t)6 * h->g.Vh;
    const size_t fb = field_bytes(h, h->ws_nrhs, sizeof(T));
    T* r = (T*)(h->fields);
    T* p = (T*)(h->fields + fb);
    T* q = (T*)(h->fields + 2 * fb);
    T* t = (T*)(h->fields + 3 * fb);
    int kmin = 0;
    for (int k = 1; k < nshift; ++k)
        if (shifts[k] < shifts[kmin]) kmin = k;
    const double m2_base = mass * mass + shifts[kmin];
    h->info_iters = 0; h->info_reliable = 0;
    CK(cudaMemsetAsync(x, 0, nreal * nshift * sizeof(T), h->stream));
    CK(cudaMemsetAsync(p, 0, nreal * nshift * sizeof(T), h->stream));
    ms_init_kernel<T><<<(unsigned)init_grid_x(nreal), kBlasBlock, 0, h->stream>>>(b, r, nreal, h->state, h->partial, tol,
                                                                                   h->max_iter, nshift);
    h->stats.launches++;
    double delta[kMaxNrhs];
    for (int k = 0; k < nshift; ++k) delta[k] = shifts[k] - shifts[kmin];
    CK(cudaMemcpyAsync(h->state->ms_delta, delta, nshift * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));   // `delta` is a stack array

    const int batch = h->check_interval > 0 ? h->check_interval : 32;
    int rc = HISQ_OK, status = HISQ_OK, cur = 0;
    bool pending = false;
    while (true) {
        if (h->use_graph) {
            hisq_ctx::CachedGraph& cg = h->ms_graph;
            // kind carries kmin, keep the number of shifts: both are baked into the captured launches
            const hisq_ctx::GraphKey key = { (const void*)x, m2_base, nshift, batch, nshift, kmin, (int)sizeof(T), h->epoch };
            if (!cg.matches(key)) {
                if (cg.exec) { cudaGraphExecDestroy(cg.exec); cg.exec = nullptr; }
                cudaGraph_t graph;
                const long long l0 = h->stats.launches;
                if (!h->cap_stream && cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
                    rc = cuda_fail(h, cudaGetLastError(), "cudaStreamCreateWithFlags"); break;
                }
                cudaStream_t user_stream = h->stream;
                cudaError_t ce = cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal);
                if (ce != cudaSuccess) { rc = cuda_fail(h, ce, "cudaStreamBeginCapture"); break; }
                h->stream = h->cap_stream;
                for (int i = 0; i < batch && rc == HISQ_OK; ++i) rc = ms_enqueue_iteration<T>(h, links, x, r, p, q, t, m2_base, kmin, nshift);
                h->stream = user_stream;
                ce = cudaStreamEndCapture(h->cap_stream, &graph);
                if (rc != HISQ_OK) { if (ce == cudaSuccess) cudaGraphDestroy(graph); break; }
                if (ce != cudaSuccess) { rc = cuda_fail(h, ce, "cudaStreamEndCapture"); break; }
                ce = cudaGraphInstantiate(&cg.exec, graph, 0);
                cudaGraphDestroy(graph);
                if (ce != cudaSuccess) { cg.exec = nullptr; rc = cuda_fail(h, ce, "cudaGraphInstantiate"); break; }
                cg.launches = h->stats.launches - l0;
                cg.key = key;
                h->stats.launches = l0;
            }
            cudaError_t ce = cudaGraphLaunch(cg.exec, h->stream);
            if (ce != cudaSuccess) { rc = cuda_fail(h, ce, "cudaGraphLaunch"); break; }
            h->stats.launches += cg.launches;
        } else {
            for (int i = 0; i < batch && rc == HISQ_OK; ++i) rc = ms_enqueue_iteration<T>(h, links, x, r, p, q, t, m2_base, kmin, nshift);
            if (rc != HISQ_OK) break;
        }
        if ((rc = poll_async(h, cur)) != HISQ_OK) break;
        if (!pending) { pending = true; cur ^= 1; continue; }
        const CgState* sp = poll_wait(h, cur ^ 1);
        if (!sp) { rc = cuda_fail(h, cudaGetLastError(), "cudaEventSynchronize"); break; }
        if (!sp->done) { cur ^= 1; continue; }
        sp = poll_wait(h, cur);
        if (!sp) { rc = cuda_fail(h, cudaGetLastError(), "cudaEventSynchronize"); break; }
        h->info_iters = sp->iter;
        if (sp->breakdown) status = HISQ_EBREAKDOWN;
        else {
            for (int k = 0; k < nshift; ++k)
                if (sp->active[k]) status = HISQ_ENOCONV;
        }
        break;
    }
    if (rc != HISQ_OK) return rc;
    // true residuals ||b - (A + sigma_k) x_k|| / ||b|| per shift (q and t are free now)
    for (int k = 0; k < nshift; ++k) {
        const double m2k = mass * mass + shifts[k];
        T* xk = x + (size_t)k * nreal;
        rc = run_dslash<T>(h, links, t, xk, HISQ_ODD, 1, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, nullptr, 2);
        if (rc) return rc;
        rc = run_dslash<T>(h, links, q, t, HISQ_EVEN, 1, MODE_RESID, xk, b, m2k, h->state->sums + k, nullptr, 2);
        if (rc) return rc;
    }
    if ((rc = poll_state(h)) != HISQ_OK) return rc;
    const CgState& s = *h->host_state;
    for (int k = 0; k < nshift; ++k) {
        h->info_relres[k] = s.bnorm2[0] > 0.0 ? std::sqrt(s.sums[k] / s.bnorm2[0]) : 0.0;
        if (status == HISQ_OK && !(h->info_relres[k] <= tol)) status = HISQ_ENOCONV;
    }
    return status;
}

static int cgp_ms_solve(hisq_ctx* h, void* x, const void* b, double mass, const double* shifts, int nshift, double tol);

extern "C" int hisq_cg_multishift(hisq_ctx* h, void* x, const void* b, double mass, const double* shifts, int nshift, double tol)
{
    if (!h || !x || !b || !shifts || nshift < 1 || nshift > HISQ_MAX_NRHS || !(tol > 0.0) || !std::isfinite(mass)) return HISQ_EINVAL;
    if (((uintptr_t)x & 15) || ((uintptr_t)b & 15)) return HISQ_EINVAL;
    for (int k = 0; k < nshift; ++k)
        if (!(shifts[k] >= 0.0) || !std::isfinite(shifts[k])) return HISQ_EINVAL;
    if (h->prec == HISQ_MIXED) return HISQ_EINVAL;   // fp64 or fp32 contexts only
    if (!h->ws) return HISQ_ENOWORKSPACE;
    if (nshift > h->ws_nrhs) return HISQ_ENOWORKSPACE;
    if (!h->have_links) return HISQ_ENOLINKS;
    const size_t bytes = (size_t)6 * h->g.Vh * elem_size(h->prec);
    if ((const char*)x < (const char*)b + bytes && (const char*)b < (const char*)x + bytes * nshift) return HISQ_EINVAL;
    if (h->g.part) return cgp_ms_solve(h, x, b, mass, shifts, nshift, tol);   // across ranks: needs the peer mailboxes
    if (h->prec == HISQ_FP32) return ms_solve<float>(h, h->links32, (float*)x, (const float*)b, mass, shifts, nshift, tol);
    return ms_solve<double>(h, h->links64, (double*)x, (const double*)b, mass, shifts, nshift, tol);
}

static int cgp_solve(hisq_ctx* h, void* x, const void* b, double mass, double tol, int nrhs);
extern "C" int hisq_cg(hisq_ctx* h, void* x, const void* b, double mass, double tol, int nrhs)
{
    if (!h || !x || !b || nrhs < 1 || nrhs > HISQ_MAX_NRHS || !(tol > 0.0) || !std::isfinite(mass)) return HISQ_EINVAL;
    if (((uintptr_t)x & 15) || ((uintptr_t)b & 15)) return HISQ_EINVAL;
    if (!h->ws) return HISQ_ENOWORKSPACE;
    if (nrhs > h->ws_nrhs) return HISQ_ENOWORKSPACE;
    if (!h->have_links) return HISQ_ENOLINKS;
    const size_t bytes = (size_t)nrhs * 6 * h->g.Vh * elem_size(h->prec);
    if (overlap(x, b, bytes)) return HISQ_EINVAL;
    if (h->g.part) return cgp_solve(h, x, b, mass, tol, nrhs);   // across ranks: needs the peer mailboxes
    if (h->prec == HISQ_FP32) return cg_solve<float, float>(h, h->links32, nullptr, (float*)x, (const float*)b, mass, tol, nrhs);
    if (h->prec == HISQ_FP64) return cg_solve<double, double>(h, h->links64, nullptr, (double*)x, (const double*)b, mass, tol, nrhs);
    return cg_solve<float, double>(h, h->links32, h->links64, (double*)x, (const double*)b, mass, tol, nrhs);
}

// ---- full-lattice solve M x = b, M = D + m (Eq. (1)) by even-odd preconditioning ----------------------
template <typename T>
static int solve_M_impl(hisq_ctx* h, const T* links, T* xe, T* xo, const T* be, const T* bo, double mass, double tol, int nrhs)
{
    const size_t nreal = (size_t)6 * h->g.Vh;
    double* dsum = h->state->sums;
    double bb[kMaxNrhs], ss[kMaxNrhs];
    const dim3 gn((unsigned)init_grid_x(nreal), (unsigned)nrhs);
    norm2_kernel<T><<<gn, kBlasBlock, 0, h->stream>>>(be, bo, nreal, h->state, h->partial, dsum);
    h->stats.launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(bb, dsum, nrhs * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    // s_e = m b_e - D_eo b_o, kept in the caller's x_odd until the even system is solved
    T* s = xo;
    int rc = run_dslash<T>(h, links, s, bo, HISQ_EVEN, nrhs, MODE_APPLY_A, be, nullptr, mass, h->state->pq, nullptr, 2);
    if (rc) return rc;
    norm2_kernel<T><<<gn, kBlasBlock, 0, h->stream>>>(s, nullptr, nreal, h->state, h->partial, dsum);
    h->stats.launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(ss, dsum, nrhs * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    double scale = 1e300;   // tol of the even system: ||r_e|| <= tol m ||b|| for every RHS
    for (int k = 0; k < nrhs; ++k)
        if (ss[k] > 0.0 && bb[k] > 0.0) scale = std::fmin(scale, mass * std::sqrt(bb[k] / ss[k]));
    if (scale == 1e300) scale = 1.0;   // b = 0 (or s_e = 0: the even system is solved by x_e = 0)
    const int rc_cg = hisq_cg(h, xe, s, mass, tol * scale, nrhs);
    if (rc_cg != HISQ_OK && rc_cg != HISQ_ENOCONV) return rc_cg;
    // x_o = (b_o - D_oe x_e) / m ; t in the solver's (now idle) temporary
    const size_t fb = field_bytes(h, h->ws_nrhs, elem_size(h->prec));
    T* t = (T*)(h->fields + 3 * fb);
    rc = run_dslash<T>(h, links, t, xe, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, nullptr, 2);
    if (rc) return rc;
    const size_t n = nreal * nrhs;
    unsigned grid = (unsigned)std::min<size_t>((n + kBlasBlock - 1) / kBlasBlock, (size_t)h->num_sms * 16);
    recon_odd_kernel<T><<<grid, kBlasBlock, 0, h->stream>>>(xo, bo, t, n, (T)(1.0 / mass));
    h->stats.launches++;
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(h->stream));
    // hisq_cg left ||s_e - A x_e|| / ||s_e||; the full-lattice residual is ||r_e|| / (m ||b||)
    for (int k = 0; k < nrhs; ++k)
        h->info_relres[k] = bb[k] > 0.0 ? h->info_relres[k] * std::sqrt(ss[k] / bb[k]) / mass : 0.0;
    return rc_cg;
}

extern "C" int hisq_solve_M(hisq_ctx* h, void* x_even, void* x_odd, const void* b_even, const void* b_odd, double mass, double tol,
                            int nrhs)
{
    if (!h || !x_even || !x_odd || !b_even || !b_odd || nrhs < 1 || nrhs > HISQ_MAX_NRHS || !(tol > 0.0) || !std::isfinite(mass) ||
        !(mass > 0.0))
        return HISQ_EINVAL;
    const void* ptr[4] = { x_even, x_odd, b_even, b_odd };
    const size_t bytes = (size_t)nrhs * 6 * h->g.Vh * elem_size(h->prec);
    for (int i = 0; i < 4; ++i) {
        if ((uintptr_t)ptr[i] & 15) return HISQ_EINVAL;
        for (int j = i + 1; j < 4; ++j)
            if (overlap(ptr[i], ptr[j], bytes)) return HISQ_EINVAL;
    }
    if (!h->ws || nrhs > h->ws_nrhs) return HISQ_ENOWORKSPACE;
    if (!h->have_links) return HISQ_ENOLINKS;
    if (h->g.part) return HISQ_EINVAL;
    if (h->prec == HISQ_FP32)
        return solve_M_impl<float>(h, h->links32, (float*)x_even, (float*)x_odd, (const float*)b_even, (const float*)b_odd, mass, tol, nrhs);
    return solve_M_impl<double>(h, h->links64, (double*)x_even, (double*)x_odd, (const double*)b_even, (const double*)b_odd, mass, tol, nrhs);
}

// ---- HISQ link smearing (row f4): thin links -> fat and Naik links, canonical layout in and out ----------------------
struct SmearCoeff { double c1, c3, c5, c7, cL; };

template <typename T>
static cudaError_t launch_staple(hisq_ctx* h, unsigned grid, const T* U, const T* a_up, const T* a_dn, const T* b, T* out_up, T* out_dn, T* acc,
                          int mu, int nu, T coef)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = 0; cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    h->stats.launches++;
    return cudaLaunchKernelEx(&cfg, staple_kernel<T>, h->g, U, a_up, a_dn, b, out_up, out_dn, acc, mu, nu, coef);
}

// out (4V matrices) = smeared `in` (4V); A, B, C: V matrices of scratch each
template <typename T>
static int smear_level(hisq_ctx* h, const T* in, T* out, T* A, T* B, T* C, const SmearCoeff& k)
{
    const Geom& g = h->g;
    const size_t V = (size_t)2 * g.Vh, mat = 18;
    const unsigned grid = (unsigned)((V + 127) / 128);
    for (int mu = 0; mu < 4; ++mu) {
        const T* Umu = in + (size_t)mu * V * mat;
        T* acc = out + (size_t)mu * V * mat;
        smear_init_kernel<T><<<(unsigned)std::min<size_t>((V * mat + 127) / 128, (size_t)h->num_sms * 32), 128, 0, h->stream>>>(acc, Umu, V * mat, (T)k.c1);
        h->stats.launches++;
        for (int nu = 0; nu < 4; ++nu) {
            if (nu == mu) continue;
            // S3_nu: up part -> A, down part -> B
            CK(launch_staple<T>(h, grid, in, Umu, Umu, nullptr, A, B, acc, mu, nu, (T)k.c3));
            if (k.cL != 0.0) {   // Lepage: the straight two-step staples only (up of up, down of down)
                CK(launch_staple<T>(h, grid, in, A, B, nullptr, nullptr, nullptr, acc, mu, nu, (T)k.cL));
            }
            for (int rho = 0; rho < 4; ++rho) {
                if (rho == mu || rho == nu) continue;
                // S5_nu,rho = G_rho[A + B] -> C
                CK(launch_staple<T>(h, grid, in, A, A, B, C, C, acc, mu, rho, (T)k.c5));
                const int sig = 6 - mu - nu - rho;
                CK(launch_staple<T>(h, grid, in, C, C, nullptr, nullptr, nullptr, acc, mu, sig, (T)k.c7));
            }
        }
    }
    CK(cudaGetLastError());
    return HISQ_OK;
}

template <typename T>
static int smear_impl(hisq_ctx* h, const T* thin, T* fat, T* naik, T* scratch, double fat_scale, double naik_scale, int fold)
{
    const Geom& g = h->g;
    const size_t V = (size_t)2 * g.Vh, field = 4 * V * 18;
    // all intermediate fields are structure-of-arrays (smear.cuh); the outputs double as scratch until they are written:
    //   fat  <- thin links transposed          (dead after level 1)
    //   naik <- the three staple fields A, B, C (dead after level 2)
    //   scratch[0] <- level 1 -> W             scratch[1] <- level 2 (X), later W in the canonical layout
    T* Usoa = fat;
    T* W = scratch;
    T* X = scratch + field;
    T* A = naik; T* B = naik + V * 18; T* C = naik + 2 * V * 18;
    const dim3 gl((unsigned)((V + 127) / 128), 4);
    link_layout_kernel<T, true><<<gl, 128, 0, h->stream>>>(g, thin, Usoa, T(1), 0);
    h->stats.launches++;
    const SmearCoeff fat7 = { 1.0 / 8.0, 1.0 / 16.0, 1.0 / 64.0, 1.0 / 384.0, 0.0 };
    const SmearCoeff fat7L = { 1.0, 1.0 / 16.0, 1.0 / 64.0, 1.0 / 384.0, -1.0 / 8.0 };
    int rc = smear_level<T>(h, Usoa, W, A, B, C, fat7);
    if (rc) return rc;
    unsigned long long* bad = h->bad_count;
    CK(cudaMemsetAsync(bad, 0, sizeof(unsigned long long), h->stream));
    project_u3_kernel<T><<<(unsigned)((4 * V + 127) / 128), 128, 0, h->stream>>>(W, V, bad);
    h->stats.launches++;
    rc = smear_level<T>(h, W, X, A, B, C, fat7L);
    if (rc) return rc;
    link_layout_kernel<T, false><<<gl, 128, 0, h->stream>>>(g, X, fat, (T)fat_scale, fold);
    naik_kernel<T><<<gl, 128, 0, h->stream>>>(g, W, naik, (T)naik_scale, fold);
    link_layout_kernel<T, false><<<gl, 128, 0, h->stream>>>(g, W, X, T(1), 0);   // W for the caller, canonical, in scratch[1]
    h->stats.launches += 3;
    CK(cudaGetLastError());
    unsigned long long nbad = 0;
    CK(cudaMemcpyAsync(&nbad, bad, sizeof(nbad), cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    if (nbad) {
        h->last_error = "hisq_smear: " + std::to_string(nbad) + " level-1 links are singular or not finite (no unitary projection)";
        return HISQ_EBREAKDOWN;
    }
    return HISQ_OK;
}

extern "C" size_t hisq_smear_bytes(const hisq_ctx* h)
{
    if (!h) return 0;
    return 2 * (size_t)4 * 2 * h->g.Vh * 18 * elem_size(h->prec);   // two link fields (see smear_impl)
}

extern "C" int hisq_smear(hisq_ctx* h, const void* thin, void* fat, void* naik, void* scratch, double fat_scale, double naik_scale,
                          int fold_phases)
{
    if (!h || !thin || !fat || !naik || !scratch || !std::isfinite(fat_scale) || !std::isfinite(naik_scale)) return HISQ_EINVAL;
    const size_t bytes = (size_t)4 * 2 * h->g.Vh * 18 * elem_size(h->prec);
    const void* ptr[5] = { thin, fat, naik, scratch, (const char*)scratch + bytes };
    for (int i = 0; i < 5; ++i) {
        if ((uintptr_t)ptr[i] & 15) return HISQ_EINVAL;
        for (int j = i + 1; j < 5; ++j)
            if (overlap(ptr[i], ptr[j], bytes)) return HISQ_EINVAL;
    }
    if (h->g.part) return HISQ_EINVAL;
    if (!h->ws) return HISQ_ENOWORKSPACE;   // the non-convergence counter lives there
    if (h->prec == HISQ_FP32)
        return smear_impl<float>(h, (const float*)thin, (float*)fat, (float*)naik, (float*)scratch, fat_scale, naik_scale, fold_phases);
    return smear_impl<double>(h, (const double*)thin, (double*)fat, (double*)naik, (double*)scratch, fat_scale, naik_scale, fold_phases);
}

// ---- options / info ----------------------------------------------------------------------------------
extern "C" int hisq_set_option(hisq_ctx* h, const char* key, double value)
{
    if (!h || !key) return HISQ_EINVAL;
    const int v = (int)value;
    drop_graphs(h);
    if (!strcmp(key, "max_iter")) { if (v < 1) return HISQ_EINVAL; h->max_iter = v; }
    else if (!strcmp(key, "reliable_interval")) { if (v < 0) return HISQ_EINVAL; h->reliable_interval = v; }
    else if (!strcmp(key, "check_interval")) { if (v < 1 || v > 1024) return HISQ_EINVAL; h->check_interval = v; }
    else if (!strcmp(key, "use_graph")) h->use_graph = v != 0;
    else if (!strcmp(key, "nrhs_inner")) { if (v < 0 || v > 8) return HISQ_EINVAL; h->nrhs_inner = v; }
    else if (!strcmp(key, "naik_compress")) h->naik_compress = v != 0;
    else if (!strcmp(key, "fused_blas")) h->fused_blas = v != 0;
    else if (!strcmp(key, "dot_fp64")) { if (v < -1 || v > 1) return HISQ_EINVAL; h->dot_fp64 = v; }
    else if (!strcmp(key, "overlap")) { if (v < -1 || v > 1) return HISQ_EINVAL; h->overlap_opt = v; }
    else if (!strcmp(key, "tile_y")) { if (v < 0 || (v > 0 && (v < 4 || h->g.L[1] % v))) return HISQ_EINVAL; h->tile_y = v; }
    else if (!strcmp(key, "tile_z")) { if (v < 0 || (v > 0 && (v < 4 || h->g.z_cnt % v))) return HISQ_EINVAL; h->tile_z = v; }
    else if (!strcmp(key, "window_mb")) { if (!(value > 0)) return HISQ_EINVAL; h->window_mb = value; }
    else return HISQ_EINVAL;
    return HISQ_OK;
}

extern "C" int hisq_get_info(const hisq_ctx* h, int* iterations, int* reliable_updates, double* true_rel_resid)
{
    if (!h) return HISQ_EINVAL;
    if (iterations) *iterations = h->info_iters;
    if (reliable_updates) *reliable_updates = h->info_reliable;
    if (true_rel_resid)
        for (int k = 0; k < kMaxNrhs && k < h->host_state->nrhs; ++k) true_rel_resid[k] = h->info_relres[k];
    return HISQ_OK;
}

// ---- layout conversion ---------------------------------------------------------------------------------
template <bool TO_NATIVE>
static int convert_layout(hisq_ctx* h, void* dst, const void* src, int nrhs)
{
    if (!h || !dst || !src || nrhs < 1 || nrhs > HISQ_MAX_NRHS) return HISQ_EINVAL;
    if (((uintptr_t)dst & 15) || ((uintptr_t)src & 15)) return HISQ_EINVAL;
    const size_t total = (size_t)nrhs * 3 * h->g.Vh;
    unsigned grid = (unsigned)((total + 255) / 256);
    if (grid > 148 * 16) grid = 148 * 16;
    if (h->prec == HISQ_FP32)
        spinor_layout_kernel<float, TO_NATIVE><<<grid, 256, 0, h->stream>>>((float*)dst, (const float*)src, h->g.Vh, nrhs);
    else
        spinor_layout_kernel<double, TO_NATIVE><<<grid, 256, 0, h->stream>>>((double*)dst, (const double*)src, h->g.Vh, nrhs);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}

extern "C" int hisq_spinor_pack(hisq_ctx* h, void* native, const void* canonical, int nrhs)
{
    return convert_layout<true>(h, native, canonical, nrhs);
}
extern "C" int hisq_spinor_unpack(hisq_ctx* h, void* canonical, const void* native, int nrhs)
{
    return convert_layout<false>(h, canonical, native, nrhs);
}

// ---- host-buffer entry points (end-to-end path: H2D, pack, run, unpack, D2H) ------------------------------
extern "C" int hisq_dslash_host(hisq_ctx* h, void* out_host, const void* in_host, int parity, int nrhs)
{
    if (!h || !out_host || !in_host || nrhs < 1 || nrhs > HISQ_MAX_NRHS) return HISQ_EINVAL;
    if (!h->ws || nrhs > h->ws_nrhs) return HISQ_ENOWORKSPACE;
    const size_t fb = field_bytes(h, h->ws_nrhs, elem_size(h->prec));
    const size_t bytes = (size_t)nrhs * 6 * h->g.Vh * elem_size(h->prec);
    char *c_in = h->stage, *n_in = h->stage + fb, *n_out = h->stage + 2 * fb, *c_out = h->stage + 3 * fb;
    CK(cudaMemcpyAsync(c_in, in_host, bytes, cudaMemcpyHostToDevice, h->stream));
    int rc = hisq_spinor_pack(h, n_in, c_in, nrhs);
    if (rc) return rc;
    rc = hisq_dslash(h, n_out, n_in, parity, nrhs);
    if (rc) return rc;
    rc = hisq_spinor_unpack(h, c_out, n_out, nrhs);
    if (rc) return rc;
    CK(cudaMemcpyAsync(out_host, c_out, bytes, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return HISQ_OK;
}

extern "C" int hisq_cg_host(hisq_ctx* h, void* x_host, const void* b_host, double mass, double tol, int nrhs)
{
    if (!h || !x_host || !b_host || nrhs < 1 || nrhs > HISQ_MAX_NRHS) return HISQ_EINVAL;
    if (!h->ws || nrhs > h->ws_nrhs) return HISQ_ENOWORKSPACE;
    const size_t fb = field_bytes(h, h->ws_nrhs, elem_size(h->prec));
    const size_t bytes = (size_t)nrhs * 6 * h->g.Vh * elem_size(h->prec);
    char *c_in = h->stage, *n_in = h->stage + fb, *n_out = h->stage + 2 * fb, *c_out = h->stage + 3 * fb;
    CK(cudaMemcpyAsync(c_in, b_host, bytes, cudaMemcpyHostToDevice, h->stream));
    int rc = hisq_spinor_pack(h, n_in, c_in, nrhs);
    if (rc) return rc;
    const int solve_rc = hisq_cg(h, n_out, n_in, mass, tol, nrhs);
    if (solve_rc != HISQ_OK && solve_rc != HISQ_ENOCONV && solve_rc != HISQ_EBREAKDOWN) return solve_rc;
    rc = hisq_spinor_unpack(h, c_out, n_out, nrhs);
    if (rc) return rc;
    CK(cudaMemcpyAsync(x_host, c_out, bytes, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return solve_rc;
}

// ---- partitioned-lattice CG (row f3): the iteration is cut into phases; between phases the CALLER exchanges halos
// and all-reduces the per-RHS sums across ranks (torch.distributed / NCCL), see partition.PartitionedCG. -----------------
struct CgpFields { void *r, *p, *q, *t; };
static CgpFields cgp_fields(hisq_ctx* h)
{
    if (h->prec == HISQ_MIXED && h->work_prec == HISQ_FP64) {   // the fp64 pair of the reliable update: r_hi, t_hi
        char* hi = h->fields + 5 * field_bytes(h, h->ws_nrhs, 4);
        return { hi, nullptr, nullptr, hi + field_bytes(h, h->ws_nrhs, 8) };
    }
    const size_t fb = field_bytes(h, h->ws_nrhs, elem_size(h->work_prec));
    return { h->fields, h->fields + fb, h->fields + 2 * fb, h->fields + 3 * fb };
}

template <typename T>
static int cgp_begin(hisq_ctx* h, T* x, const T* b, double tol, int nrhs)
{
    const size_t nreal = (size_t)6 * h->g.Vh, total = nreal * nrhs;
    CgpFields f = cgp_fields(h);
    CK(cudaMemsetAsync(x, 0, total * sizeof(T), h->stream));
    CK(cudaMemsetAsync(f.p, 0, total * sizeof(T), h->stream));
    CK(cudaMemsetAsync(f.q, 0, total * sizeof(T), h->stream));
    CK(cudaMemsetAsync(f.t, 0, total * sizeof(T), h->stream));
    const int S = h->g.Vh / h->g.L[3];
    // r = b, then r's halo := 0 so that ||r||^2 over the extended array is the interior sum; LOCAL ||b||^2 -> state.rho
    cudaMemcpyAsync(f.r, b, total * sizeof(T), cudaMemcpyDeviceToDevice, h->stream);
    zero_halo_kernel<T><<<148 * 4, 256, 0, h->stream>>>((T*)f.r, S, h->g.L[3], h->g.t_lo, h->g.t_cnt, nrhs, h->g.zpart ? h->g.H * h->g.L[1] : 0, h->g.z_lo, h->g.z_cnt);
    dim3 gi((unsigned)init_grid_x(nreal), (unsigned)nrhs);
    cg_init_kernel<T, T><<<gi, kBlasBlock, 0, h->stream>>>((const T*)f.r, (T*)f.r, nreal, h->state, h->partial, tol, h->max_iter);
    h->stats.launches += 2;
    CK(cudaGetLastError());
    h->cgp_x = x; h->cgp_nrhs = nrhs; h->cgp_tol = tol;
    return HISQ_OK;
}

template <typename T>
static int cgp_phase(hisq_ctx* h, const T* links, int phase, double mass)
{
    const int nrhs = h->cgp_nrhs;
    if (nrhs < 1 || !h->cgp_x) return HISQ_EINVAL;
    const size_t nreal = (size_t)6 * h->g.Vh;
    CgpFields f = cgp_fields(h);
    T *r = (T*)f.r, *p = (T*)f.p, *q = (T*)f.q, *t = (T*)f.t, *x = (T*)h->cgp_x;
    const Span sp = owned_span(h, V16<T>::n);
    dim3 gb((unsigned)blas_grid_x(sp.seg ? 3 * sp.seg * V16<T>::n : nreal, V16<T>::n), (unsigned)nrhs);
    switch (phase) {
    case 0:  // after the all-reduce of rho (= ||b||^2)
        cgp_finalize_init_kernel<<<1, 1, 0, h->stream>>>(h->state, nrhs, h->cgp_tol, h->max_iter);
        h->stats.launches++;
        break;
    case 1: return enqueue_p_update<T>(h, p, r, nrhs);
    case 2: return run_dslash<T>(h, links, t, p, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, &h->state->done, 2);
    case 3: return run_dslash<T>(h, links, q, t, HISQ_EVEN, nrhs, MODE_APPLY_A, p, nullptr, mass * mass, h->state->pq, &h->state->done, 2);
    // Phases 2 and 3 split so that the halo exchange overlaps the slices that do not read the halo: 20 / 30 compute the
    // owned slices [3, n-3) (no t-hop leaves the owned range), 21 / 31 the first and last 3.  The launches of 30 + 31 share
    // one ticket and one table of partial sums, so pq is the same sum, in the same order, as phase 3 gives.
    case 20: case 21: case 30: case 31: {
        const int n = h->g.t_cnt, w = kHopMax;
        const bool second = phase >= 30, boundary = (phase % 10) == 1;
        // interior: [w, n-w); boundary: [0, w) and [n-w, n) in ONE launch (blockIdx.y >= w skips the interior)
        int first = 0, count = 0, skip_at = 1 << 30, skip = 0;
        if (n > 2 * w) {
            if (!boundary) { first = w; count = n - 2 * w; }
            else { count = 2 * w; skip_at = w; skip = n - 2 * w; }
        } else if (boundary) count = n;
        if (count > 0) {
            int rc = second ? run_dslash<T>(h, links, q, t, HISQ_EVEN, nrhs, MODE_APPLY_A, p, nullptr, mass * mass, h->state->pq,
                                            &h->state->done, 2, first, count, skip_at, skip)
                            : run_dslash<T>(h, links, t, p, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr,
                                            &h->state->done, 2, first, count, skip_at, skip);
            if (rc) return rc;
        }
        return HISQ_OK;
    }
    case 4:
        cg_update_xr_kernel<T><<<gb, kBlasBlock, 0, h->stream>>>(x, r, p, q, nreal, h->state, h->partial, 1, h->fuse_push_sums, h->fuse_red_pq, sp);
        h->stats.launches++;
        break;
    case 5:  // after the all-reduce of sums (= ||r||^2)
        cgp_finalize_xr_kernel<<<1, 1, 0, h->stream>>>(h->state, nrhs, h->fuse_red_sums, h->part_nranks);
        h->stats.launches++;
        break;
    default: return HISQ_EINVAL;
    }
    CK(cudaGetLastError());
    return HISQ_OK;
}

extern "C" int hisq_cgp_begin(hisq_ctx* h, void* x, const void* b, double tol, int nrhs)
{
    if (!h || !x || !b || nrhs < 1 || nrhs > HISQ_MAX_NRHS || !(tol > 0.0)) return HISQ_EINVAL;
    if (!h->ws || nrhs > h->ws_nrhs) return HISQ_ENOWORKSPACE;
    if (!h->have_links) return HISQ_ENOLINKS;
    if (h->prec == HISQ_MIXED) return HISQ_EINVAL;
    return h->prec == HISQ_FP32 ? cgp_begin<float>(h, (float*)x, (const float*)b, tol, nrhs)
                                : cgp_begin<double>(h, (double*)x, (const double*)b, tol, nrhs);
}
static int cgp_phase_any(hisq_ctx* h, int phase, double mass)
{
    return h->work_prec == HISQ_FP32 ? cgp_phase<float>(h, h->links32, phase, mass) : cgp_phase<double>(h, h->links64, phase, mass);
}
extern "C" int hisq_cgp_phase(hisq_ctx* h, int phase, double mass)
{
    if (!h || h->prec == HISQ_MIXED) return HISQ_EINVAL;
    return cgp_phase_any(h, phase, mass);
}
// which: 0 = p field, 1 = t field (halo exchange); 2 = rho, 3 = pq, 4 = sums (kMaxNrhs doubles each; all-reduce the first nrhs)
extern "C" void* hisq_cgp_ptr(hisq_ctx* h, int which)
{
    if (!h || !h->ws) return nullptr;
    CgpFields f = cgp_fields(h);
    switch (which) {
    case 0: return f.p;
    case 1: return f.t;
    case 2: return h->state->rho;
    case 3: return h->state->pq;
    case 4: return h->state->sums;
    default: return nullptr;
    }
}
extern "C" int hisq_cgp_status(hisq_ctx* h, int* iterations, int* done, int* breakdown, double* rel_resid)
{
    if (!h || !h->ws) return HISQ_EINVAL;
    int rc = poll_state(h);
    if (rc) return rc;
    const CgState& s = *h->host_state;
    if (iterations) *iterations = s.iter;
    if (done) *done = s.done;
    if (breakdown) *breakdown = s.breakdown;
    if (rel_resid)
        for (int k = 0; k < s.nrhs && k < kMaxNrhs; ++k) rel_resid[k] = s.bnorm2[k] > 0.0 ? std::sqrt(s.rho[k] / s.bnorm2[k]) : 0.0;
    return HISQ_OK;
}

extern "C" size_t hisq_halo_bytes(const hisq_ctx* h, int nrhs)
{
    if (!h || !h->g.part || nrhs < 1 || nrhs > HISQ_MAX_NRHS) return 0;
    return (size_t)nrhs * 3 * kHopMax * (h->g.Vh / h->g.L[3]) * 2 * elem_size(h->prec);   // only 3 of the 4 halo slices are ever read
}

template <bool PACK>
static int halo_move(hisq_ctx* h, void* field, void* lo, void* hi, int nrhs, unsigned* sig_a = nullptr, unsigned* sig_b = nullptr)
{
    if (!h || !field || !lo || !hi || nrhs < 1 || nrhs > HISQ_MAX_NRHS || !h->g.part) return HISQ_EINVAL;
    if (!h->ws) return HISQ_ENOWORKSPACE;
    const int S = h->g.Vh / h->g.L[3];
    const size_t total = (size_t)nrhs * 3 * kHopMax * S;
    unsigned grid = (unsigned)((total + 255) / 256);
    if (grid > 148 * 4) grid = 148 * 4;
    unsigned* ticket = &h->state->ticket[3];
    if (h->work_prec == HISQ_FP32)
        halo_kernel<float, PACK><<<grid, 256, 0, h->stream>>>((float*)field, (float*)lo, (float*)hi, S, h->g.L[3], h->g.t_lo, h->g.t_cnt, kHopMax, nrhs, ticket, sig_a, sig_b);
    else
        halo_kernel<double, PACK><<<grid, 256, 0, h->stream>>>((double*)field, (double*)lo, (double*)hi, S, h->g.L[3], h->g.t_lo, h->g.t_cnt, kHopMax, nrhs, ticket, sig_a, sig_b);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}
extern "C" int hisq_halo_pack(hisq_ctx* h, void* send_lo, void* send_hi, const void* field, int nrhs)
{
    return halo_move<true>(h, const_cast<void*>(field), send_lo, send_hi, nrhs);
}
extern "C" int hisq_halo_unpack(hisq_ctx* h, void* field, const void* recv_lo, const void* recv_hi, int nrhs)
{
    return halo_move<false>(h, field, const_cast<void*>(recv_lo), const_cast<void*>(recv_hi), nrhs);
}

// the same for the z cut: 3 planes on each side of the owned z range, owned time slices only
extern "C" size_t hisq_zhalo_bytes(const hisq_ctx* h, int nrhs)
{
    if (!h || !h->g.zpart || nrhs < 1 || nrhs > HISQ_MAX_NRHS) return 0;
    return (size_t)nrhs * 3 * h->g.t_cnt * kHopMax * h->g.H * h->g.L[1] * 2 * elem_size(h->prec);
}
template <bool PACK>
static int zhalo_move(hisq_ctx* h, void* field, void* lo, void* hi, int nrhs, unsigned* sig_a = nullptr, unsigned* sig_b = nullptr)
{
    if (!h || !field || !lo || !hi || nrhs < 1 || nrhs > HISQ_MAX_NRHS || !h->g.zpart) return HISQ_EINVAL;
    if (!h->ws) return HISQ_ENOWORKSPACE;
    const Geom& g = h->g;
    const int S = g.Vh / g.L[3], HLy = g.H * g.L[1];
    const size_t total = (size_t)nrhs * 3 * g.t_cnt * kHopMax * HLy;
    unsigned grid = (unsigned)((total + 255) / 256);
    if (grid > 148 * 4) grid = 148 * 4;
    unsigned* ticket = &h->state->ticket[3];
    if (h->work_prec == HISQ_FP32)
        zhalo_kernel<float, PACK><<<grid, 256, 0, h->stream>>>((float*)field, (float*)lo, (float*)hi, HLy, S, g.L[3], g.t_lo, g.t_cnt, g.z_lo, g.z_cnt, kHopMax, nrhs, ticket, sig_a, sig_b);
    else
        zhalo_kernel<double, PACK><<<grid, 256, 0, h->stream>>>((double*)field, (double*)lo, (double*)hi, HLy, S, g.L[3], g.t_lo, g.t_cnt, g.z_lo, g.z_cnt, kHopMax, nrhs, ticket, sig_a, sig_b);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}
extern "C" int hisq_zhalo_pack(hisq_ctx* h, void* send_lo, void* send_hi, const void* field, int nrhs)
{
    return zhalo_move<true>(h, const_cast<void*>(field), send_lo, send_hi, nrhs);
}
extern "C" int hisq_zhalo_unpack(hisq_ctx* h, void* field, const void* recv_lo, const void* recv_hi, int nrhs)
{
    return zhalo_move<false>(h, field, const_cast<void*>(recv_lo), const_cast<void*>(recv_hi), nrhs);
}

// ---- halo transport through peer-mapped memory (no library collective) ----------------------------------------
// Mailbox = [16 counters (u32), 256 B][reduce data: [2 slots][16 ranks][16] doubles][slot 0: lo, hi][slot 1: lo, hi].
// Counters 0, 1: halo arrivals of the two slots (each exchange adds 2: one per neighbour); 8, 9: reduce arrivals (each
// reduce adds nranks).  The SENDING kernels bump them with system-scope atomics after fencing their stores; the receiver
// waits with a stream memory operation (cuStreamWaitValue32): no kernel spins.
// Why two slots and no "free" credits: every rank alternates send e, recv e, send e+1, ...  A rank's send e+2 follows
// its recv e+1 in stream order, which completes only after BOTH neighbours' send e+1, each of which follows that
// neighbour's recv e (unpack finished) in its own stream order: the slot of exchange e has been read before it is
// written again.
static const size_t kMboxFlags = 256;
static const size_t kMboxReduce = (size_t)2 * kMaxRanks * kMaxNrhs * sizeof(double);
typedef CUresult (*StreamMemOp32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
static StreamMemOp32 g_wait32 = nullptr;
static bool load_memops()
{
    if (g_wait32) return true;
    void* w = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &w, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) return false;
    g_wait32 = (StreamMemOp32)w;
    return true;
}
static CUresult stream_wait_geq(hisq_ctx* h, const void* counter, unsigned value)
{
    return g_wait32((CUstream)h->stream, (CUdeviceptr)(uintptr_t)counter, value, CU_STREAM_WAIT_VALUE_GEQ);
}
static char* mbox_buffer(char* box, size_t buf, int slot, int hi) { return box + kMboxFlags + kMboxReduce + (size_t)(2 * slot + hi) * buf; }
static unsigned* mbox_counter(char* box, int slot) { return reinterpret_cast<unsigned*>(box) + slot; }
// the z-halo buffers follow the four t-halo buffers; their arrival counters are 2, 3
static char* mbox_zbuffer(char* box, size_t tbuf, size_t zbuf, int slot, int hi) { return box + kMboxFlags + kMboxReduce + 4 * tbuf + (size_t)(2 * slot + hi) * zbuf; }
static unsigned* mbox_zcounter(char* box, int slot) { return reinterpret_cast<unsigned*>(box) + 2 + slot; }

extern "C" size_t hisq_peer_bytes(const hisq_ctx* h, int nrhs)
{
    const size_t b = hisq_halo_bytes(h, nrhs);
    return b ? kMboxFlags + kMboxReduce + 4 * align_up(b) + 4 * align_up(hisq_zhalo_bytes(h, nrhs)) : 0;
}
extern "C" int hisq_peer_attach(hisq_ctx* h, void* const* boxes, int nboxes, int nrhs)
{
    if (!h || !h->g.part || !boxes || nrhs < 1 || nrhs > HISQ_MAX_NRHS) return HISQ_EINVAL;
    if (nboxes != h->part_nranks || nboxes > kMaxRanks) return HISQ_EINVAL;
    for (int r = 0; r < nboxes; ++r)
        if (!boxes[r] || ((uintptr_t)boxes[r] & 255)) return HISQ_EINVAL;
    if (!load_memops()) { h->last_error = "stream memory operations (cuStreamWaitValue32) are not available"; return HISQ_ECUDA; }
    for (int r = 0; r < kMaxRanks; ++r) h->mbox_all.box[r] = r < nboxes ? (char*)boxes[r] : nullptr;
    h->mbox = (char*)boxes[h->part_rank];
    {   // neighbours on the nz x nt grid of ranks (rank = rz + nz * rt), periodic in both directions
        const int nz = h->part_nz, nt = h->part_nt, rz = h->part_rank % nz, rt = h->part_rank / nz;
        h->mbox_up = (char*)boxes[rz + nz * ((rt + 1) % nt)];
        h->mbox_down = (char*)boxes[rz + nz * ((rt + nt - 1) % nt)];
        h->mbox_zup = (char*)boxes[(rz + 1) % nz + nz * rt];
        h->mbox_zdown = (char*)boxes[(rz + nz - 1) % nz + nz * rt];
    }
    h->mbox_buf = align_up(hisq_halo_bytes(h, nrhs));
    h->mbox_zbuf = align_up(hisq_zhalo_bytes(h, nrhs));
    h->mbox_nrhs = nrhs;
    h->seq_send = h->seq_recv = h->red_send = h->red_recv = 0;
    {   // the protocol counts arrivals from zero: a mailbox that has been used (or poisoned by an abort) is refused
        unsigned counters[16];
        CK(cudaMemcpyAsync(counters, h->mbox, sizeof counters, cudaMemcpyDeviceToHost, h->stream));
        CK(cudaStreamSynchronize(h->stream));
        for (int i = 0; i < 16; ++i)
            if (counters[i] != 0) {
                h->mbox = nullptr;
                h->last_error = "hisq_peer_attach: this rank's mailbox is not zeroed (used before, or aborted)";
                return HISQ_EINVAL;
            }
    }
    if (!h->d_boxes) CK(cudaMalloc(&h->d_boxes, sizeof(PeerBoxes)));
    CK(cudaMemcpyAsync(h->d_boxes, &h->mbox_all, sizeof(PeerBoxes), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    return HISQ_OK;
}
#define CKU(call)                                                                                         \
    do {                                                                                                  \
        CUresult r_ = (call);                                                                             \
        if (r_ != CUDA_SUCCESS) { h->last_error = std::string(#call) + ": CUresult " + std::to_string((int)r_); return HISQ_ECUDA; } \
    } while (0)
extern "C" int hisq_halo_send(hisq_ctx* h, const void* field, int nrhs)
{
    if (!h || !field || !h->mbox || nrhs < 1 || nrhs > h->mbox_nrhs) return HISQ_EINVAL;
    if (h->seq_send != h->seq_recv) return HISQ_EINVAL;   // strict alternation send / recv (see the slot argument above)
    const unsigned e = h->seq_send + 1;
    const int s = (int)(e & 1u);
    // my lowest slices -> the previous rank's UPPER halo buffer, my highest -> the next rank's LOWER halo buffer
    int rc = halo_move<true>(h, const_cast<void*>(field), mbox_buffer(h->mbox_down, h->mbox_buf, s, 1),
                             mbox_buffer(h->mbox_up, h->mbox_buf, s, 0), nrhs, mbox_counter(h->mbox_down, s),
                             mbox_counter(h->mbox_up, s));
    if (rc) return rc;
    if (h->g.zpart) {   // my lowest planes -> the z-previous rank's UPPER z-halo buffer, my highest -> the z-next rank's LOWER
        rc = zhalo_move<true>(h, const_cast<void*>(field), mbox_zbuffer(h->mbox_zdown, h->mbox_buf, h->mbox_zbuf, s, 1),
                              mbox_zbuffer(h->mbox_zup, h->mbox_buf, h->mbox_zbuf, s, 0), nrhs, mbox_zcounter(h->mbox_zdown, s),
                              mbox_zcounter(h->mbox_zup, s));
        if (rc) return rc;
    }
    h->seq_send = e;
    return HISQ_OK;
}
extern "C" int hisq_halo_recv(hisq_ctx* h, void* field, int nrhs)
{
    if (!h || !field || !h->mbox || nrhs < 1 || nrhs > h->mbox_nrhs) return HISQ_EINVAL;
    if (h->seq_recv + 1 != h->seq_send) return HISQ_EINVAL;   // nothing sent for this exchange: the neighbours would wait for ever
    const unsigned e = h->seq_recv + 1;
    const int s = (int)(e & 1u);
    const unsigned uses = (e + 1) >> 1;   // how often this slot has been used, this exchange included
    CKU(stream_wait_geq(h, mbox_counter(h->mbox, s), 2u * uses));
    int rc = halo_move<false>(h, field, mbox_buffer(h->mbox, h->mbox_buf, s, 0), mbox_buffer(h->mbox, h->mbox_buf, s, 1), nrhs);
    if (rc) return rc;
    if (h->g.zpart) {
        CKU(stream_wait_geq(h, mbox_zcounter(h->mbox, s), 2u * uses));
        rc = zhalo_move<false>(h, field, mbox_zbuffer(h->mbox, h->mbox_buf, h->mbox_zbuf, s, 0),
                               mbox_zbuffer(h->mbox, h->mbox_buf, h->mbox_zbuf, s, 1), nrhs);
        if (rc) return rc;
    }
    h->seq_recv = e;
    return HISQ_OK;
}

static double* state_array(hisq_ctx* h, int which)
{
    switch (which) {
    case 2: return h->state->rho;
    case 3: return h->state->pq;
    case 4: return h->state->sums;
    default: return nullptr;
    }
}
// Reduce number e uses slot e & 1.  A slot is written again two reduces later; by then every rank has finished reduce
// e + 1, which needed every rank's contribution, sent after that rank had summed reduce e: no credit flags are needed.
extern "C" int hisq_peer_reduce_send(hisq_ctx* h, int which, int nrhs)
{
    if (!h || !h->mbox || !h->ws || nrhs < 1 || nrhs > kMaxNrhs || !state_array(h, which)) return HISQ_EINVAL;
    if (h->red_send != h->red_recv) return HISQ_EINVAL;   // one reduce in flight at a time (the slot argument above)
    const unsigned e = ++h->red_send;
    peer_reduce_send_kernel<<<h->part_nranks, 32, 0, h->stream>>>(state_array(h, which), h->mbox_all, h->part_rank, (int)(e & 1u), nrhs,
                                                                  kMboxFlags, kMboxCounterOff);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}
extern "C" int hisq_peer_reduce_recv(hisq_ctx* h, int which, int nrhs)
{
    if (!h || !h->mbox || !h->ws || nrhs < 1 || nrhs > kMaxNrhs || !state_array(h, which)) return HISQ_EINVAL;
    if (h->red_recv + 1 != h->red_send) return HISQ_EINVAL;
    const unsigned e = ++h->red_recv;
    const int s = (int)(e & 1u);
    const unsigned uses = (e + 1) >> 1;   // how often this slot has been used, this reduce included
    CKU(stream_wait_geq(h, h->mbox + kMboxCounterOff + 4 * s, uses * (unsigned)h->part_nranks));
    peer_reduce_sum_kernel<<<1, 32, 0, h->stream>>>(state_array(h, which), h->mbox, h->part_nranks, s, nrhs, kMboxFlags);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}

// Fused form of hisq_peer_reduce_send / recv: the producing kernel's last block pushes (PeerPush), the stream waits,
// the consuming kernels read the slot.  Same counters and slots as the stand-alone calls.
static PeerPush reduce_next_push(hisq_ctx* h)
{
    const unsigned e = ++h->red_send;
    PeerPush pp;
    pp.boxes = h->d_boxes; pp.nranks = h->part_nranks; pp.rank = h->part_rank; pp.slot = (int)(e & 1u);
    return pp;
}
static const double* reduce_wait(hisq_ctx* h, int& rc)
{
    const unsigned e = ++h->red_recv;
    const int s = (int)(e & 1u);
    const unsigned uses = (e + 1) >> 1;
    CUresult r = stream_wait_geq(h, h->mbox + kMboxCounterOff + 4 * s, uses * (unsigned)h->part_nranks);
    rc = HISQ_OK;
    if (r != CUDA_SUCCESS) { h->last_error = "cuStreamWaitValue32: CUresult " + std::to_string((int)r); rc = HISQ_ECUDA; }
    return reinterpret_cast<const double*>(h->mbox + kMboxFlags) + (size_t)s * kMaxRanks * kMaxNrhs;
}
struct FuseGuard {   // the fused pointers never outlive the solve
    hisq_ctx* h;
    ~FuseGuard() { h->fuse_push_pq = h->fuse_push_sums = PeerPush(); h->fuse_red_pq = h->fuse_red_sums = nullptr; }
};

// r := b - A x over all ranks, sums := global ||r_k||^2, then the reliable-update bookkeeping (rho := true value, systems
// above tol become active again, done re-evaluated).  Stand-alone reduce kernels: this runs once or twice per solve.
template <typename T>
static int cgp_true_residual_t(hisq_ctx* h, const T* links, T* x, const T* b, double mass, int nrhs)
{
    CgpFields f = cgp_fields(h);
    int rc;
    if ((rc = hisq_halo_send(h, x, nrhs)) || (rc = hisq_halo_recv(h, x, nrhs))) return rc;
    if ((rc = run_dslash<T>(h, links, (T*)f.t, x, HISQ_ODD, nrhs, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, nullptr, 2))) return rc;
    if ((rc = hisq_halo_send(h, f.t, nrhs)) || (rc = hisq_halo_recv(h, f.t, nrhs))) return rc;
    if ((rc = run_dslash<T>(h, links, (T*)f.r, (const T*)f.t, HISQ_EVEN, nrhs, MODE_RESID, x, b, mass * mass, h->state->sums, nullptr, 2))) return rc;
    if ((rc = hisq_peer_reduce_send(h, 4, nrhs)) || (rc = hisq_peer_reduce_recv(h, 4, nrhs))) return rc;
    cg_after_residual_kernel<<<1, 1, 0, h->stream>>>(h->state, h->true_rr);
    h->stats.launches++;
    CK(cudaGetLastError());
    return HISQ_OK;
}
static int cgp_true_residual(hisq_ctx* h, void* x, const void* b, double mass, int nrhs)
{
    return h->work_prec == HISQ_FP32 ? cgp_true_residual_t<float>(h, h->links32, (float*)x, (const float*)b, mass, nrhs)
                                : cgp_true_residual_t<double>(h, h->links64, (double*)x, (const double*)b, mass, nrhs);
}

// hisq_cg on a partitioned context: the phase-wise iteration with every cross-rank step done through the mailboxes, all
// on the stream -- the host only polls the state every check_interval iterations.  The all-reduce gives every rank the
// same bits, so all ranks take the same decisions (stop, breakdown, iteration count) and issue the same calls.
// Tell every rank that this one is leaving the solve with an error (peer_abort_kernel): on a stream of its own, because
// the context's stream may itself be waiting for a peer.
static void peer_abort(hisq_ctx* h)
{
    if (!h->mbox) return;
    if (!h->abort_stream && cudaStreamCreateWithFlags(&h->abort_stream, cudaStreamNonBlocking) != cudaSuccess) return;
    peer_abort_kernel<<<1, 96, 0, h->abort_stream>>>(h->mbox_all, h->part_nranks);
    cudaStreamSynchronize(h->abort_stream);
    cudaStreamSynchronize(h->stream);   // poisoned counters release this rank's own waits too
}
// state + this rank's abort word; HISQ_EPEER if a peer has aborted
static int poll_state_peer(hisq_ctx* h)
{
    int rc = poll_state(h);
    if (rc) return rc;
    unsigned flag = 0;
    CK(cudaMemcpyAsync(&flag, h->mbox + kMboxAbortWord * sizeof(unsigned), sizeof flag, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    if (flag) { h->last_error = "a peer rank aborted the solve"; return HISQ_EPEER; }
    return HISQ_OK;
}
// All ranks must run the same sequence of exchanges: compare what decides it (nrhs, max_iter, check_interval, overlap, tol,
// mass) across the ranks before the first iteration, through one round of the reduce mailbox.
static int cgp_check_options(hisq_ctx* h, double mass, double tol, int nrhs, bool split)
{
    double mine[6] = { (double)nrhs, (double)h->max_iter, (double)h->check_interval, split ? 1.0 : 0.0, tol, mass };
    CK(cudaMemcpyAsync(h->state->sums, mine, sizeof mine, cudaMemcpyHostToDevice, h->stream));
    int rc = hisq_peer_reduce_send(h, 4, 6);
    if (rc) return rc;
    const double* slot = reduce_wait(h, rc);
    if (rc) return rc;
    double all[kMaxRanks * kMaxNrhs];
    unsigned flag = 0;
    CK(cudaMemcpyAsync(all, slot, sizeof all, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaMemcpyAsync(&flag, h->mbox + kMboxAbortWord * sizeof(unsigned), sizeof flag, cudaMemcpyDeviceToHost, h->stream));
    CK(cudaStreamSynchronize(h->stream));
    if (flag) { h->last_error = "a peer rank aborted the solve"; return HISQ_EPEER; }   // the wait was released by its poison
    for (int r = 0; r < h->part_nranks; ++r)
        for (int i = 0; i < 6; ++i)
            if (all[r * kMaxNrhs + i] != mine[i]) {
                h->last_error = "hisq_cg on a partitioned lattice: rank " + std::to_string(r) + " was called with different arguments or options";
                return HISQ_EINVAL;
            }
    return HISQ_OK;
}

static int cgp_solve_impl(hisq_ctx* h, void* x, const void* b, double mass, double tol, int nrhs);
static int cgp_solve(hisq_ctx* h, void* x, const void* b, double mass, double tol, int nrhs)
{
    const int rc = cgp_solve_impl(h, x, b, mass, tol, nrhs);
    // HISQ_ENOCONV / HISQ_EBREAKDOWN are decided from all-reduced numbers: every rank returns them together.  Anything else
    // is this rank's own failure: release the others (they return HISQ_EPEER at their next poll)
    if (rc != HISQ_OK && rc != HISQ_ENOCONV && rc != HISQ_EBREAKDOWN && rc != HISQ_EPEER) peer_abort(h);
    return rc;
}
// start of a HISQ_MIXED multi-rank solve: fp64 interface (x, b), fp32 iteration fields r p q t x_lo, fp64 pair r_hi t_hi
static int cgp_begin_mixed(hisq_ctx* h, double* x, const double* b, double tol, int nrhs)
{
    const size_t nreal = (size_t)6 * h->g.Vh, total = nreal * nrhs;
    const size_t fb32 = field_bytes(h, h->ws_nrhs, 4), fb64 = field_bytes(h, h->ws_nrhs, 8);
    float* r = (float*)h->fields;
    float* xlo = (float*)(h->fields + 4 * fb32);
    double* rhi = (double*)(h->fields + 5 * fb32);
    double* thi = (double*)(h->fields + 5 * fb32 + fb64);
    CK(cudaMemsetAsync(x, 0, total * 8, h->stream));
    CK(cudaMemsetAsync(h->fields + fb32, 0, 4 * fb32, h->stream));   // p, q, t, x_lo
    CK(cudaMemsetAsync(thi, 0, total * 8, h->stream));
    // r_hi = b with zeroed halo slices (sums over the extended arrays are then interior sums); r = (float) r_hi;
    // LOCAL ||b||^2 in fp64 -> state.rho
    CK(cudaMemcpyAsync(rhi, b, total * 8, cudaMemcpyDeviceToDevice, h->stream));
    const int S = h->g.Vh / h->g.L[3];
    zero_halo_kernel<double><<<148 * 4, 256, 0, h->stream>>>(rhi, S, h->g.L[3], h->g.t_lo, h->g.t_cnt, nrhs, h->g.zpart ? h->g.H * h->g.L[1] : 0, h->g.z_lo, h->g.z_cnt);
    dim3 gi((unsigned)init_grid_x(nreal), (unsigned)nrhs);
    cg_init_kernel<double, float><<<gi, kBlasBlock, 0, h->stream>>>(rhi, r, nreal, h->state, h->partial, tol, h->max_iter);
    h->stats.launches += 2;
    CK(cudaGetLastError());
    h->cgp_x = xlo; h->cgp_nrhs = nrhs; h->cgp_tol = tol;
    return HISQ_OK;
}

struct WorkPrecGuard {   // the working precision never outlives the solve
    hisq_ctx* h;
    ~WorkPrecGuard() { h->work_prec = h->prec == HISQ_MIXED ? HISQ_FP64 : h->prec; }
};

static int cgp_solve_impl(hisq_ctx* h, void* x, const void* b, double mass, double tol, int nrhs)
{
    if (!h->mbox || nrhs > h->mbox_nrhs) return HISQ_EINVAL;
    const bool mixed = h->prec == HISQ_MIXED;
    // with a z cut every time slice reads the z halo: the interior / edge split by time slices does not apply
    const bool split_opt = !h->g.zpart && (h->overlap_opt < 0 ? h->g.t_cnt >= 4 * kHopMax : h->overlap_opt != 0);
    int rc = cgp_check_options(h, mass, tol, nrhs, split_opt);
    if (rc) return rc;
    WorkPrecGuard wguard{ h };
    h->work_prec = mixed ? HISQ_FP32 : h->prec;     // the iteration's precision (phases, halos, fields)
    rc = mixed ? cgp_begin_mixed(h, (double*)x, (const double*)b, tol, nrhs) : hisq_cgp_begin(h, x, b, tol, nrhs);
    if (rc) return rc;
    if ((rc = hisq_peer_reduce_send(h, 2, nrhs)) || (rc = hisq_peer_reduce_recv(h, 2, nrhs)) || (rc = cgp_phase_any(h, 0, mass))) return rc;
    const CgpFields fl = cgp_fields(h);
    void* p = fl.p;
    void* t = fl.t;
    const size_t total = (size_t)6 * h->g.Vh * nrhs;
    h->info_reliable = 0;
    FuseGuard guard{ h };
    // splitting a Dslash costs a launch tail and some L2 reuse: do it when at least half of the owned
    // slices can run under the transfer, or when asked to (option "overlap": -1 auto, 0 never, 1 always)
    const bool split = split_opt;
    // HISQ_MIXED: every R iterations (counted from the last one) x_hi += x_lo and r is replaced by the fp64 true residual
    // over all ranks, as on one GPU (a8); batches divide R so that a poll falls on every boundary
    const int R = mixed ? h->reliable_interval : 0;
    int batch = h->check_interval > 0 ? h->check_interval : 32;
    if (R > 0) {
        int best = 1;
        for (int d = 1; d <= R && d <= batch; ++d)
            if (R % d == 0) best = d;
        batch = best;
    }
    int confirms = 0, rel_base = 0;
    bool have_true = false;
    for (;;) {
        if ((rc = poll_state_peer(h))) return rc;
        CgState s = *h->host_state;
        const bool claimed = s.done && !s.breakdown && s.iter < h->max_iter;
        const bool due = R > 0 && !s.done && s.iter > rel_base && (s.iter - rel_base) % R == 0;
        if (claimed || due) {
            if (claimed && confirms >= 8) {   // the recursive residual keeps converging, the true one does not: below the attainable accuracy
                h->info_iters = s.iter;
                for (int k = 0; k < nrhs; ++k) h->info_relres[k] = s.bnorm2[k] > 0.0 ? std::sqrt(((const double*)((const char*)h->host_state + sizeof(CgState)))[k] / s.bnorm2[k]) : 0.0;
                return HISQ_ENOCONV;
            }
            // converged by the recursive residual (or a reliable update is due): r = b - A x across the ranks (halo of x,
            // of D_oe x, one all-reduce); the bookkeeping kernel re-activates the systems whose true residual is above tol
            // and the iteration resumes from the true residual (the single-GPU rule, a7 / a8)
            if (claimed) ++confirms;
            h->fuse_push_pq = h->fuse_push_sums = PeerPush(); h->fuse_red_pq = h->fuse_red_sums = nullptr;
            if (mixed) {
                acc_xhi_kernel<<<(unsigned)((total / 4 + kBlasBlock - 1) / kBlasBlock + 1), kBlasBlock, 0, h->stream>>>((double*)x, (float*)h->cgp_x, total);
                h->stats.launches++;
                h->work_prec = HISQ_FP64;
                rc = cgp_true_residual_t<double>(h, h->links64, (double*)x, (const double*)b, mass, nrhs);
                const CgpFields hi = cgp_fields(h);
                h->work_prec = HISQ_FP32;
                if (rc) return rc;
                convert_kernel<double, float><<<1184, kBlasBlock, 0, h->stream>>>((const double*)hi.r, (float*)fl.r, total);
                h->stats.launches++;
                CK(cudaGetLastError());
            } else if ((rc = cgp_true_residual(h, x, b, mass, nrhs))) return rc;
            if ((rc = poll_state_peer(h))) return rc;
            s = *h->host_state;
            rel_base = s.iter;
            have_true = true;
            h->info_reliable++;
        }
        if (s.done || s.breakdown || s.iter >= h->max_iter) {
            if (mixed && !(claimed || due)) {   // stopped by max_iter or a breakdown: hand out what has been accumulated
                acc_xhi_kernel<<<(unsigned)((total / 4 + kBlasBlock - 1) / kBlasBlock + 1), kBlasBlock, 0, h->stream>>>((double*)x, (float*)h->cgp_x, total);
                h->stats.launches++;
                CK(cudaStreamSynchronize(h->stream));
            }
            h->info_iters = s.iter;
            (void)have_true;
            for (int k = 0; k < nrhs; ++k) h->info_relres[k] = s.bnorm2[k] > 0.0 ? std::sqrt(s.rho[k] / s.bnorm2[k]) : 0.0;
            if (s.breakdown) return HISQ_EBREAKDOWN;
            int any = 0;      // done is also raised at max_iter: converged = no system left active
            for (int k = 0; k < nrhs; ++k) any |= s.active[k];
            return any ? HISQ_ENOCONV : HISQ_OK;
        }
        for (int i = 0; i < batch; ++i) {
            if ((rc = cgp_phase_any(h, 1, mass))) return rc;
            // the kernels that produce <p,q> and ||r||^2 push them to all ranks themselves, those that consume them add up
            // the mailbox entries themselves: no reduction kernel, one stream wait per all-reduce
            h->fuse_push_pq = reduce_next_push(h);
            if (split) {   // interior slices while the halo is in flight, edge slices once it has arrived
                if ((rc = hisq_halo_send(h, p, nrhs)) || (rc = cgp_phase_any(h, 20, mass))) return rc;
                if ((rc = hisq_halo_recv(h, p, nrhs)) || (rc = cgp_phase_any(h, 21, mass))) return rc;
                if ((rc = hisq_halo_send(h, t, nrhs)) || (rc = cgp_phase_any(h, 30, mass))) return rc;
                if ((rc = hisq_halo_recv(h, t, nrhs)) || (rc = cgp_phase_any(h, 31, mass))) return rc;
            } else {
                if ((rc = hisq_halo_send(h, p, nrhs)) || (rc = hisq_halo_recv(h, p, nrhs)) || (rc = cgp_phase_any(h, 2, mass))) return rc;
                if ((rc = hisq_halo_send(h, t, nrhs)) || (rc = hisq_halo_recv(h, t, nrhs)) || (rc = cgp_phase_any(h, 3, mass))) return rc;
            }
            h->fuse_red_pq = reduce_wait(h, rc);            // <p,q> of all ranks have arrived
            if (rc) return rc;
            h->fuse_push_sums = reduce_next_push(h);
            if ((rc = cgp_phase_any(h, 4, mass))) return rc;
            h->fuse_red_sums = reduce_wait(h, rc);          // ||r||^2 of all ranks have arrived
            if (rc) return rc;
            if ((rc = cgp_phase_any(h, 5, mass))) return rc;
        }
    }
}

// Multi-shift CG across the ranks of a partitioned lattice (PAPER.md:141 on top of :187-191): the single-GPU iteration
// (ms_solve) with the two halo exchanges of the base direction and the two all-reduces (<p,q>, ||r||^2: one double each)
// put where the cross-rank steps are due; the other shifts cost AXPYs only, as on one GPU.
template <typename T>
static int cgp_ms_solve_t(hisq_ctx* h, const T* links, T* x, const T* b, double mass, const double* shifts, int nshift, double tol)
{
    if (!h->mbox || h->mbox_nrhs < 1) return HISQ_EINVAL;
    double shift_sum = 0.0;
    for (int k = 0; k < nshift; ++k) shift_sum += shifts[k] * (k + 1);
    int rc = cgp_check_options(h, mass + shift_sum, tol, nshift, false);
    if (rc) return rc;
    const size_t nreal = (size_t)6 * h->g.Vh;
    const size_t fb = field_bytes(h, h->ws_nrhs, sizeof(T));
    T* r = (T*)(h->fields);
    T* p = (T*)(h->fields + fb);
    T* q = (T*)(h->fields + 2 * fb);
    T* t = (T*)(h->fields + 3 * fb);
    int kmin = 0;
    for (int k = 1; k < nshift; ++k)
        if (shifts[k] < shifts[kmin]) kmin = k;
    const double m2_base = mass * mass + shifts[kmin];
    h->info_iters = 0; h->info_reliable = 0;
    CK(cudaMemsetAsync(x, 0, nreal * nshift * sizeof(T), h->stream));
    CK(cudaMemsetAsync(p, 0, nreal * nshift * sizeof(T), h->stream));
    CK(cudaMemsetAsync(q, 0, nreal * sizeof(T), h->stream));
    CK(cudaMemsetAsync(t, 0, nreal * sizeof(T), h->stream));
    // r = b with zeroed halo slices, LOCAL ||b||^2 -> rho, all-reduce, then the state from the global value
    CK(cudaMemcpyAsync(r, b, nreal * sizeof(T), cudaMemcpyDeviceToDevice, h->stream));
    const int S = h->g.Vh / h->g.L[3];
    zero_halo_kernel<T><<<148 * 4, 256, 0, h->stream>>>(r, S, h->g.L[3], h->g.t_lo, h->g.t_cnt, 1, h->g.zpart ? h->g.H * h->g.L[1] : 0, h->g.z_lo, h->g.z_cnt);
    ms_init_kernel<T><<<(unsigned)init_grid_x(nreal), kBlasBlock, 0, h->stream>>>(r, r, nreal, h->state, h->partial, tol, h->max_iter, nshift);
    h->stats.launches += 2;
    double delta[kMaxNrhs];
    for (int k = 0; k < nshift; ++k) delta[k] = shifts[k] - shifts[kmin];
    CK(cudaMemcpyAsync(h->state->ms_delta, delta, nshift * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CK(cudaStreamSynchronize(h->stream));   // `delta` is a stack array
    if ((rc = hisq_peer_reduce_send(h, 2, 1)) || (rc = hisq_peer_reduce_recv(h, 2, 1))) return rc;
    ms_finalize_init_kernel<<<1, 1, 0, h->stream>>>(h->state, nshift);
    h->stats.launches++;
    const unsigned gx = (unsigned)blas_grid_x(nreal, V16<T>::n);
    T* pb = p + (size_t)kmin * nreal;   // the base direction: the smallest shift has zeta = 1
    int status = HISQ_OK;
    for (;;) {
        if ((rc = poll_state_peer(h))) return rc;
        const CgState s = *h->host_state;
        if (s.done || s.breakdown || s.iter >= h->max_iter) {
            h->info_iters = s.iter;
            if (s.breakdown) status = HISQ_EBREAKDOWN;
            else
                for (int k = 0; k < nshift; ++k)
                    if (s.active[k]) status = HISQ_ENOCONV;
            break;
        }
        for (int i = 0; i < h->check_interval; ++i) {
            ms_update_p_kernel<T><<<dim3(gx, (unsigned)nshift), kBlasBlock, 0, h->stream>>>(p, r, nreal, h->state);
            h->stats.launches++;
            if ((rc = hisq_halo_send(h, pb, 1)) || (rc = hisq_halo_recv(h, pb, 1))) return rc;
            if ((rc = run_dslash<T>(h, links, t, pb, HISQ_ODD, 1, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, &h->state->done, 2))) return rc;
            if ((rc = hisq_halo_send(h, t, 1)) || (rc = hisq_halo_recv(h, t, 1))) return rc;
            if ((rc = run_dslash<T>(h, links, q, t, HISQ_EVEN, 1, MODE_APPLY_A, pb, nullptr, m2_base, h->state->pq, &h->state->done, 2))) return rc;
            if ((rc = hisq_peer_reduce_send(h, 3, 1)) || (rc = hisq_peer_reduce_recv(h, 3, 1))) return rc;
            ms_update_xr_kernel<T><<<dim3(gx, (unsigned)nshift + 1), kBlasBlock, 0, h->stream>>>(x, r, p, q, nreal, h->state, h->partial, 1);
            h->stats.launches++;
            if ((rc = hisq_peer_reduce_send(h, 4, 1)) || (rc = hisq_peer_reduce_recv(h, 4, 1))) return rc;
            ms_finalize_kernel<<<1, 1, 0, h->stream>>>(h->state, nshift);
            h->stats.launches++;
            CK(cudaGetLastError());
        }
    }
    // true residuals ||b - (A + sigma_k) x_k|| / ||b|| per shift over all ranks (q and t are free now)
    for (int k = 0; k < nshift; ++k) {
        const double m2k = mass * mass + shifts[k];
        T* xk = x + (size_t)k * nreal;
        if ((rc = hisq_halo_send(h, xk, 1)) || (rc = hisq_halo_recv(h, xk, 1))) return rc;
        if ((rc = run_dslash<T>(h, links, t, xk, HISQ_ODD, 1, MODE_PLAIN, nullptr, nullptr, 0.0, nullptr, nullptr, 2))) return rc;
        if ((rc = hisq_halo_send(h, t, 1)) || (rc = hisq_halo_recv(h, t, 1))) return rc;
        if ((rc = run_dslash<T>(h, links, q, t, HISQ_EVEN, 1, MODE_RESID, xk, b, m2k, h->state->sums + k, nullptr, 2))) return rc;
    }
    if ((rc = hisq_peer_reduce_send(h, 4, nshift)) || (rc = hisq_peer_reduce_recv(h, 4, nshift))) return rc;
    if ((rc = poll_state_peer(h)) != HISQ_OK) return rc;
    const CgState& s = *h->host_state;
    for (int k = 0; k < nshift; ++k) {
        h->info_relres[k] = s.bnorm2[0] > 0.0 ? std::sqrt(s.sums[k] / s.bnorm2[0]) : 0.0;
        if (status == HISQ_OK && !(h->info_relres[k] <= tol)) status = HISQ_ENOCONV;
    }
    return status;
}

static int cgp_ms_solve(hisq_ctx* h, void* x, const void* b, double mass, const double* shifts, int nshift, double tol)
{
    const int rc = h->prec == HISQ_FP32 ? cgp_ms_solve_t<float>(h, h->links32, (float*)x, (const float*)b, mass, shifts, nshift, tol)
                                        : cgp_ms_solve_t<double>(h, h->links64, (double*)x, (const double*)b, mass, shifts, nshift, tol);
    if (rc != HISQ_OK && rc != HISQ_ENOCONV && rc != HISQ_EBREAKDOWN && rc != HISQ_EPEER) peer_abort(h);
    return rc;
}

extern "C" int hisq_naik_compressed(const hisq_ctx* h) { return h && h->naik_c14 ? 1 : 0; }

extern "C" long long hisq_launch_count(const hisq_ctx* h) { return h ? h->stats.launches : 0; }

extern "C" const char* hisq_strerror(int code)
{
    switch (code) {
    case HISQ_OK: return "success";
    case HISQ_EINVAL: return "invalid argument";
    case HISQ_ENOLINKS: return "links not set";
    case HISQ_ENOWORKSPACE: return "workspace missing or too small";
    case HISQ_ECUDA: return "CUDA error (see hisq_last_error)";
    case HISQ_ENOCONV: return "CG did not converge within max_iter";
    case HISQ_EBREAKDOWN: return "breakdown (CG: <p,Ap> <= 0 or non-finite scalar; smearing: singular link)";
    case HISQ_EIO: return "file cannot be read / written or fails its checksum";
    case HISQ_EPEER: return "multi-rank solve aborted by another rank (its error, or options that differ between ranks)";
    case HISQ_ETOOBIG: return "hisq_norm2_noalloc: beyond its static scratch (at most 16 right-hand sides of 67108864 reals each)";
    default: return "unknown error code";
    }
}

extern "C" const char* hisq_last_error(const hisq_ctx* h) { return h ? h->last_error.c_str() : ""; }

// introspection for tests / DESIGN.md tables: registers per thread of a Dslash instantiation
extern "C" int hisq_debug_dslash_regs(int prec, int nr, int mode)
{
    return prec == HISQ_FP32 ? dslash_regs<float>(nr, mode) : dslash_regs<double>(nr, mode);
}
// the CTA sweep tiling the next Dslash launch with `nrhs` would use: out[0]=tile_y, out[1]=tile_z
extern "C" int hisq_debug_tiles(hisq_ctx* h, int nrhs, int* out)
{
    if (!h || !out) return HISQ_EINVAL;
    choose_tiles(h, nrhs, h->prec == HISQ_FP32 ? 4 : 8);
    out[0] = h->g.ty; out[1] = h->g.tz;
    return HISQ_OK;
}
