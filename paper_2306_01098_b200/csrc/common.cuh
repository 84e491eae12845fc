// common.cuh -- shared device helpers of libhisq (sm_100a).  Product code; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace hisq {

constexpr int kMaxNrhs = 16;

// ---- 16-byte / 8-byte vector types per precision -------------------------------------------------
template <typename T> struct Vec;
template <> struct Vec<double> { using c1 = double2; using c16 = double2; };   // one complex; one 16-byte chunk
template <> struct Vec<float>  { using c1 = float2; using c16 = float4; };

// ---- global loads with cache hints ---------------------------------------------------------------
// Links are read exactly once per Dslash application (every link is used forward by its
// own site and backward by the site it points to), so they stream: no L1 allocation, evict-first.
// (measured neutral and dropped: ld.global.nc.L1::no_allocate for the links, L1::evict_last on the gathers; a plain
// read-only load for the links is 3-6 % slower: DESIGN.md section 6)
__device__ __forceinline__ double2 ld_stream(const double2* p) { return __ldcs(p); }
__device__ __forceinline__ float4 ld_stream(const float4* p) { return __ldcs(p); }
__device__ __forceinline__ float2 ld_stream(const float2* p) { return __ldcs(p); }
// Colour vectors are gathered by 16 different output sites: keep them in L1/L2.
__device__ __forceinline__ double2 ld_keep(const double2* p) { return __ldg(p); }
__device__ __forceinline__ float2 ld_keep(const float2* p) { return __ldg(p); }
__device__ __forceinline__ float4 ld_keep(const float4* p) { return __ldg(p); }

// ---- lattice geometry handed to kernels ----------------------------------------------------------
struct Geom {
    int L[4];       // Lx, Ly, Lz, Lt
    int H;          // Lx / 2 : sites of one parity in an x-row
    int Vh;         // sites of one parity
    int sy, sz, st; // half-index strides of a unit step in y, z, t: H, H*Ly, H*Ly*Lz
    int stride[4];  // {1, sy, sz, st}: half-index step per unit of (x/2, y, z, t)
    // CTA sweep order: the lattice is cut into (tile_y x tile_z) columns in
    // (y,z); inside a column work runs x fastest, then y, then z, then t; columns are swept last.
    int ty, tz;     // tile extents in y and z (divide Ly, Lz)
    int nty, ntz;   // number of tiles
    // t-partitioned lattice (row f3): this context holds t_cnt time slices of a larger lattice at local slices
    // [t_lo, t_lo + t_cnt) of an array of L[3] = t_cnt + 2*t_lo slices; the rest are halo slices filled by the
    // neighbouring ranks.  t-hops never wrap locally; the antiperiodic sign applies where the GLOBAL boundary is.
    int part;       // 0: ordinary periodic lattice (t_lo = 0, t_cnt = L[3])
    int t_lo, t_cnt;
    int flip_lo, flip_hi;  // this rank owns the lower / upper global t boundary
    // second cut, along z (a rank grid nz x nt): the context holds z_cnt planes of the global lattice at local planes
    // [z_lo, z_lo + z_cnt) of L[2] = z_cnt + 2*z_lo; z-hops never wrap locally (z is periodic: no sign).  zpart = 0: z whole.
    int zpart, z_lo, z_cnt;
};

// ---- device-side state of one CG solve (all scalars stay on the GPU) -------------
struct CgState {
    double rho[kMaxNrhs];      // ||r_k||^2 (recursive)
    double rho_prev[kMaxNrhs]; // rho before the last update (for beta after a reliable update)
    double pq[kMaxNrhs];       // Re<p_k, A p_k>
    double beta[kMaxNrhs];
    double bnorm2[kMaxNrhs];   // ||b_k||^2
    double sums[kMaxNrhs];     // scratch result of stand-alone reductions
    double alpha[kMaxNrhs];    // alpha_k of the last iteration (x += alpha p is applied by the NEXT p-update pass)
    int xpend[kMaxNrhs];       // iteration number whose x-update of RHS k is still pending, -1: none
    double tol2;               // tol^2
    int active[kMaxNrhs];      // 1 while RHS k still iterates
    int iter;
    int max_iter;
    int done;                  // 1: every RHS converged (tentatively) or max_iter hit -> kernels return at once
    int breakdown;
    int nrhs;
    unsigned ticket[4];        // last-block tickets of the reducing kernels
    // multi-shift CG: shifted residuals stay collinear, r_k = zeta_k r
    double ms_delta[kMaxNrhs];     // sigma_k - sigma_min
    double ms_zeta[kMaxNrhs];      // zeta_k^n
    double ms_zeta_prev[kMaxNrhs]; // zeta_k^{n-1}
    double ms_beta_k[kMaxNrhs];    // beta_k^n = beta_n (zeta^{n+1}/zeta^n)^2
    double ms_alpha_old, ms_beta_old;
    int ms_nshift;
};

// ---- all-reduce through peer-mapped mailboxes (row f3; layout and protocol: hisq.cu, "halo transport") ----------
constexpr int kMaxRanks = 16;
constexpr size_t kMboxCounterOff = 8 * sizeof(unsigned);   // reduce arrival counters (one per slot)
constexpr size_t kMboxDataOff = 256;                        // reduce data [2 slots][kMaxRanks][kMaxNrhs] doubles
struct PeerBoxes { char* box[kMaxRanks]; };                 // every rank's mailbox as addressable from this device
struct PeerPush {                                           // boxes == nullptr: off
    const PeerBoxes* boxes;
    int nranks, rank, slot;
};

// The LAST block of a reducing kernel hands its n local sums (vals: shared memory, written before a barrier) to every
// rank: stores into each mailbox [slot][my rank][k], barrier, then one thread per destination fences at system scope
// (cumulative over the CTA's stores, the grid.sync idiom) and bumps that mailbox's counter.  Call block-uniformly.
__device__ __forceinline__ void peer_push(const PeerPush& pp, const double* vals, int n)
{
    for (int idx = threadIdx.x; idx < pp.nranks * n; idx += blockDim.x) {
        const int r = idx / n, k = idx - r * n;
        double* dst = reinterpret_cast<double*>(pp.boxes->box[r] + kMboxDataOff) + ((size_t)pp.slot * kMaxRanks + pp.rank) * kMaxNrhs;
        dst[k] = vals[k];
    }
    __syncthreads();
    if ((int)threadIdx.x < pp.nranks) {
        __threadfence_system();
        atomicAdd_system(reinterpret_cast<unsigned*>(pp.boxes->box[threadIdx.x] + kMboxCounterOff) + pp.slot, 1u);
    }
}
// Sum over ranks, in rank order (the same bits on every rank), of entry k of one slot of this rank's own mailbox.
__device__ __forceinline__ double peer_sum(const double* slot_data, int nranks, int k)
{
    const volatile double* d = slot_data;
    double s = 0.0;
    for (int r = 0; r < nranks; ++r) s += d[(size_t)r * kMaxNrhs + k];
    return s;
}

// ---- deterministic two-stage reduction: block partials, then the last block to finish sums them ---
// vals[NR] are this thread's contributions to right-hand sides k0 .. k0+NR-1.  partial is
// [nrhs_total][ncols]; this block owns column `col` of rows k0..k0+NR-1.  Returns true in the LAST of
// `total_blocks` blocks to arrive, where totals[k], k < nrhs_total (shared memory) then hold the grid
// sums.  Fixed summation order: run-to-run reproducible (no floating-point atomics).
template <int NR, int BLOCK>
__device__ __forceinline__ bool grid_reduce(const double (&vals)[NR], int k0, double* __restrict__ partial, int ncols,
                                            int col, unsigned* ticket, unsigned total_blocks, int nrhs_total,
                                            double* totals /* shared, kMaxNrhs */)
{
    constexpr int NW = BLOCK / 32;
    __shared__ double s_warp[NW * (NR > 1 ? NR : 1)];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NR; ++k) {
        double v = vals[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) s_warp[k * NW + warp] = v;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < NR; ++k) {
            double s = 0.0;
            for (int w = 0; w < NW; ++w) s += s_warp[k * NW + w];
            partial[(size_t)(k0 + k) * ncols + col] = s;
        }
        __threadfence();
        unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == total_blocks - 1u);
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
    for (int k = 0; k < nrhs_total; ++k) {
        // 8 loads in flight per thread (the partials sit in L2: ~1 us each if serialised); fixed order: deterministic
        double acc8[8] = { 0, 0, 0, 0, 0, 0, 0, 0 };
        const double* row = partial + (size_t)k * ncols;
        for (int i0 = threadIdx.x; i0 < ncols; i0 += BLOCK * 8) {
            double v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int i = i0 + j * BLOCK;
                v[j] = i < ncols ? __ldcg(row + i) : 0.0;
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) acc8[j] += v[j];
        }
        double s = ((acc8[0] + acc8[1]) + (acc8[2] + acc8[3])) + ((acc8[4] + acc8[5]) + (acc8[6] + acc8[7]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        __syncthreads();
        if (lane == 0) s_warp[warp] = s;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < NW; ++w) tot += s_warp[w];
            totals[k] = tot;
        }
    }
    if (threadIdx.x == 0) *ticket = 0u;
    __syncthreads();
    return true;
}

}  // namespace hisq
