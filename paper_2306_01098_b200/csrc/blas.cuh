// blas.cuh -- fused BLAS-1 kernels of the multi-RHS CG (rows a6-a8 of SURVEY.md section 8).
// Per right-hand side k the scalars alpha_k, beta_k are independent ("solves A x_k = b_k
// with multiple input vectors b_k"); they live in CgState on the device and are derived in each
// kernel's prologue, so the host never sits between two kernels of an iteration.
// Sums are accumulated in fp64 whatever the field precision and reduced in a fixed order.
//
// Fields are NATIVE half-lattice arrays: RHS k is the contiguous block [k*nreal, (k+1)*nreal) of reals,
// nreal = 6*Vh.  Grid: blockIdx.y = k, blockIdx.x over 16-byte vectors of that block.
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"

namespace hisq {

constexpr int kBlasBlock = 256;
constexpr int kBlasItems = 4;  // 16-byte vectors per thread

template <typename T> struct V16;
template <> struct V16<double> { using type = double2; static constexpr int n = 2; };
template <> struct V16<float> { using type = float4; static constexpr int n = 4; };

template <typename T> __device__ __forceinline__ void unpack16(const typename V16<T>::type& w, T* e);
template <> __device__ __forceinline__ void unpack16<double>(const double2& w, double* e) { e[0] = w.x; e[1] = w.y; }
template <> __device__ __forceinline__ void unpack16<float>(const float4& w, float* e) { e[0] = w.x; e[1] = w.y; e[2] = w.z; e[3] = w.w; }
template <typename T> __device__ __forceinline__ typename V16<T>::type pack16(const T* e);
template <> __device__ __forceinline__ double2 pack16<double>(const double* e) { return make_double2(e[0], e[1]); }
template <> __device__ __forceinline__ float4 pack16<float>(const float* e) { return make_float4(e[0], e[1], e[2], e[3]); }

// Partitioned lattices: the per-iteration updates touch the OWNED slices only.  A field is 3 planes (colour) per RHS,
// the owned part of a plane is one contiguous run: vector i' of the 3*seg owned vectors is vector
// (i'/seg)*plane + off + i'%seg of the field.  seg == 0: the whole field, i' = i.
// With a z cut as well the owned part of a time slice is itself a run (sub vectors) inside the slice (sub_stride vectors):
// seg = t_cnt * sub.
struct Span { size_t seg, plane, off, sub, sub_stride; };
__device__ __forceinline__ size_t span_map(const Span& sp, size_t i)
{
    if (sp.seg == 0) return i;
    const size_t c = i / sp.seg;
    size_t j = i - c * sp.seg;
    if (sp.sub) {
        const size_t tt = j / sp.sub;
        j = tt * sp.sub_stride + (j - tt * sp.sub);
    }
    return c * sp.plane + sp.off + j;
}

inline int blas_grid_x(size_t nreal, int vec_n) {
    size_t nvec = nreal / vec_n;
    return (int)((nvec + (size_t)kBlasBlock * kBlasItems - 1) / ((size_t)kBlasBlock * kBlasItems));
}

// ---- start of a solve: r = b (rounded to T), rho = ||b||^2 in fp64, state reset ---------------------
template <typename TB, typename T>
__global__ void __launch_bounds__(kBlasBlock) cg_init_kernel(const TB* b, T* r /* may alias b (phase-wise CG) */, size_t nreal,
                                                             CgState* st, double* partial, double tol, int max_iter)
{
    const int k = blockIdx.y;
    const size_t base = (size_t)k * nreal;
    double sum[1] = { 0.0 };
    for (int it = 0; it < kBlasItems * 4; ++it) {
        size_t i = ((size_t)blockIdx.x * kBlasItems * 4 + it) * kBlasBlock + threadIdx.x;
        if (i < nreal) {
            TB v = b[base + i];
            r[base + i] = (T)v;
            sum[0] += (double)v * (double)v;
        }
    }
    __shared__ double totals[kMaxNrhs];
    const int ncols = gridDim.x;
    if (grid_reduce<1, kBlasBlock>(sum, k, partial, ncols, blockIdx.x, &st->ticket[0], gridDim.x * gridDim.y, gridDim.y, totals)) {
        const int n = gridDim.y;
        if (threadIdx.x < n) {
            const int kk = threadIdx.x;
            const double bb = totals[kk];
            st->rho[kk] = bb; st->rho_prev[kk] = bb; st->bnorm2[kk] = bb;
            st->pq[kk] = 1.0; st->beta[kk] = 0.0; st->sums[kk] = 0.0;
            st->alpha[kk] = 0.0; st->xpend[kk] = -1;
            st->active[kk] = bb > 0.0 ? 1 : 0;
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int any = 0;
            for (int kk = 0; kk < n; ++kk) any |= st->active[kk];
            st->tol2 = tol * tol; st->iter = 0; st->max_iter = max_iter; st->breakdown = 0; st->nrhs = n;
            st->done = any ? 0 : 1;
        }
    }
}
inline int init_grid_x(size_t nreal) { return (int)((nreal + (size_t)kBlasBlock * kBlasItems * 4 - 1) / ((size_t)kBlasBlock * kBlasItems * 4)); }

// ---- [x_k += alpha_k p_k of the PREVIOUS iteration] ; p_k = r_k + beta_k p_k  (first kernel of an iteration; beta = 0 at
// the start gives p = r).  Folding the x-update into this pass (x is touched nowhere else inside an iteration) saves one
// read of p per iteration: 48 n instead of 54 n words per site for the BLAS part.  The update of iteration i is
// pending (st->xpend[k] == i) from the r-update of iteration i until this kernel of iteration i+1, or until
// cg_flush_x_kernel when the loop is left (true-residual check, reliable update, end of the solve).
// x == nullptr: plain p-update (partitioned lattices, start of a solve).
template <typename T>
__global__ void __launch_bounds__(kBlasBlock) cg_update_p_kernel(T* __restrict__ p, const T* __restrict__ r, size_t nreal,
                                                                 const CgState* st, Span sp = Span(), T* __restrict__ x = nullptr,
                                                                 int flush_only = 0)
{
    if (st->done && !flush_only) return;
    using V = typename V16<T>::type;
    constexpr int N = V16<T>::n;
    const int k = blockIdx.y;
    const bool do_x = x != nullptr && st->xpend[k] == st->iter;
    const bool do_p = !flush_only && st->active[k] != 0;  // frozen RHS keep their search direction (needed if they are resumed)
    if (!do_x && !do_p) return;
    const T beta = (T)st->beta[k], alpha = (T)st->alpha[k];
    const size_t nvec = sp.seg ? 3 * sp.seg : nreal / N;
    V* pv = reinterpret_cast<V*>(p + (size_t)k * nreal);
    V* xv = reinterpret_cast<V*>(x + (size_t)k * nreal);
    const V* rv = reinterpret_cast<const V*>(r + (size_t)k * nreal);
    V rr[kBlasItems], pp[kBlasItems], xx[kBlasItems];
#pragma unroll
    for (int it = 0; it < kBlasItems; ++it) {
        size_t i = ((size_t)blockIdx.x * kBlasItems + it) * kBlasBlock + threadIdx.x;
        if (i < nvec) {
            const size_t j = span_map(sp, i);
            pp[it] = pv[j];
            if (do_p) rr[it] = rv[j];
            if (do_x) xx[it] = xv[j];
        }
    }
#pragma unroll
    for (int it = 0; it < kBlasItems; ++it) {
        size_t i = ((size_t)blockIdx.x * kBlasItems + it) * kBlasBlock + threadIdx.x;
        if (i < nvec) {
            const size_t j = span_map(sp, i);
            T b[N];
            unpack16<T>(pp[it], b);
            if (do_x) {
                T c[N];
                unpack16<T>(xx[it], c);
#pragma unroll
                for (int e = 0; e < N; ++e) c[e] = fma(alpha, b[e], c[e]);
                xv[j] = pack16<T>(c);
            }
            if (do_p) {
                T a[N];
                unpack16<T>(rr[it], a);
#pragma unroll
                for (int e = 0; e < N; ++e) b[e] = fma(beta, b[e], a[e]);
                pv[j] = pack16<T>(b);
            }
        }
    }
}

// ---- x_k += alpha_k p_k ; r_k -= alpha_k q_k ; rho'_k = ||r_k||^2 ; last block: beta, convergence ----
template <typename T>
__global__ void __launch_bounds__(kBlasBlock) cg_update_xr_kernel(T* __restrict__ x, T* __restrict__ r, const T* __restrict__ p,
                                                                  const T* __restrict__ q, size_t nreal, CgState* st,
                                                                  double* partial, int defer = 0, PeerPush push = PeerPush(),
                                                                  const double* red_pq = nullptr, Span sp = Span(), int fold_x = 0,
                                                                  int trips = 1)
{
    // trips: consecutive 4 KB-per-array chunks one CTA works through (large fields: the reduction tail and the dependent
    // loads of the scalars at the head of a CTA cost as much as streaming one chunk; measured 4.7 -> see DESIGN.md 7)
    // fold_x = 1: x is left alone here; alpha_k is handed to the next cg_update_p_kernel pass (st->alpha, st->xpend)
    // defer = 1 (partitioned lattice).  red_pq: <p,q> is not in st->pq yet but, rank by rank, in this slot of the
    // mailbox (every block adds them up itself); push: the last block hands the local ||r||^2 to all ranks.
    if (st->done) {   // finished: keep the other ranks' arrival count right (see dslash_kernel)
        if (push.boxes != nullptr && blockIdx.x == 0 && blockIdx.y == 0) peer_push(push, st->sums, gridDim.y);
        return;
    }
    using V = typename V16<T>::type;
    constexpr int N = V16<T>::n;
    const int k = blockIdx.y;
    double alpha_d = 0.0;
    if (st->active[k]) {
        const double pq = red_pq ? peer_sum(red_pq, push.nranks, k) : st->pq[k];
        alpha_d = (pq > 0.0 && isfinite(pq)) ? st->rho[k] / pq : 0.0;
    }
    const T alpha = (T)alpha_d;
    const size_t nvec = sp.seg ? 3 * sp.seg : nreal / N;
    const size_t base = (size_t)k * nreal;
    V* xv = reinterpret_cast<V*>(x + base);
    V* rv = reinterpret_cast<V*>(r + base);
    const V* pv = reinterpret_cast<const V*>(p + base);
    const V* qv = reinterpret_cast<const V*>(q + base);
    const bool live = st->active[k] != 0;  // frozen RHS: no traffic, but the block still joins the reduction
    double sum[1] = { 0.0 };
    for (int tr = 0; tr < trips; ++tr) {
        const size_t bx = (size_t)blockIdx.x * trips + tr;
        V xx[kBlasItems], rr[kBlasItems], pp[kBlasItems], qq[kBlasItems];
#pragma unroll
        for (int it = 0; it < kBlasItems; ++it) {
            size_t i = (bx * kBlasItems + it) * kBlasBlock + threadIdx.x;
            if (live && i < nvec) {
                const size_t j = span_map(sp, i);
                rr[it] = rv[j]; qq[it] = qv[j];
                if (!fold_x) { xx[it] = xv[j]; pp[it] = pv[j]; }
            }
        }
#pragma unroll
        for (int it = 0; it < kBlasItems; ++it) {
            size_t i = (bx * kBlasItems + it) * kBlasBlock + threadIdx.x;
            if (live && i < nvec) {
                T b[N], d[N];
                unpack16<T>(rr[it], b); unpack16<T>(qq[it], d);
#pragma unroll
                for (int e = 0; e < N; ++e) {
                    b[e] = fma(-alpha, d[e], b[e]);
                    sum[0] += (double)b[e] * (double)b[e];
                }
                const size_t j = span_map(sp, i);
                if (!fold_x) {
                    T a[N], c[N];
                    unpack16<T>(xx[it], a); unpack16<T>(pp[it], c);
#pragma unroll
                    for (int e = 0; e < N; ++e) a[e] = fma(alpha, c[e], a[e]);
                    xv[j] = pack16<T>(a);
                }
                rv[j] = pack16<T>(b);
            }
        }
    }
    __shared__ double totals[kMaxNrhs];
    if (grid_reduce<1, kBlasBlock>(sum, k, partial, gridDim.x, blockIdx.x, &st->ticket[1], gridDim.x * gridDim.y, gridDim.y,
                                   totals)) {
        const int n = gridDim.y;
        if (defer) {   // partitioned lattice: only the LOCAL sums; the scalar update runs after the cross-rank all-reduce
            if (threadIdx.x < n) {
                st->sums[threadIdx.x] = totals[threadIdx.x];
                if (red_pq) st->pq[threadIdx.x] = peer_sum(red_pq, push.nranks, threadIdx.x);   // for the scalar update
            }
            if (push.boxes) peer_push(push, totals, n);
            return;
        }
        if (threadIdx.x < n) {
            const int kk = threadIdx.x;
            if (st->active[kk]) {
                const double rn = totals[kk], pq = st->pq[kk];
                if (!(pq > 0.0) || !isfinite(pq) || !isfinite(rn)) st->breakdown = 1;
                if (fold_x) {   // the same alpha every block used above; applied to x by the next p-update pass
                    st->alpha[kk] = (pq > 0.0 && isfinite(pq)) ? st->rho[kk] / pq : 0.0;
                    st->xpend[kk] = st->iter + 1;
                }
                st->rho_prev[kk] = st->rho[kk];
                st->beta[kk] = rn / st->rho[kk];
                st->rho[kk] = rn;
                if (rn <= st->tol2 * st->bnorm2[kk]) st->active[kk] = 0;
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int any = 0;
            for (int kk = 0; kk < n; ++kk) any |= st->active[kk];
            const int it = st->iter + 1;
            st->iter = it;
            if (!any || it >= st->max_iter || st->breakdown) st->done = 1;
        }
    }
}

// ---- fused update for fields small enough to stay in registers across a grid barrier (cooperative launch) ----
// = cg_update_xr_kernel of iteration i followed by cg_update_p_kernel of iteration i+1 in ONE kernel: the new r and the
// old p stay in registers over the barrier, so r is not re-read and one launch per iteration disappears (C1/C2-size
// lattices are launch- and L2-latency-bound in their BLAS part).  Same arithmetic, same summation order per block
// column as the two-kernel path.  `do_p = 0` (last iteration before a reliable update) leaves p untouched.
template <typename T, int KEEP>
__global__ void __launch_bounds__(kBlasBlock) cg_fused_update_kernel(T* __restrict__ x, T* __restrict__ r, T* __restrict__ p,
                                                                     const T* __restrict__ q, size_t nreal, CgState* st,
                                                                     double* partial, int do_p)
{
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    if (st->done) return;   // grid-uniform: written only by earlier kernels
    using V = typename V16<T>::type;
    constexpr int N = V16<T>::n;
    constexpr int NW = kBlasBlock / 32;
    const int k = blockIdx.y, n = gridDim.y, gx = gridDim.x;
    __shared__ double s_rho[kMaxNrhs], s_pq[kMaxNrhs], s_bn2[kMaxNrhs], s_rn[kMaxNrhs], s_warp[NW];
    __shared__ int s_active[kMaxNrhs], s_misc[3];
    if (threadIdx.x < n) {
        s_rho[threadIdx.x] = st->rho[threadIdx.x]; s_pq[threadIdx.x] = st->pq[threadIdx.x];
        s_bn2[threadIdx.x] = st->bnorm2[threadIdx.x]; s_active[threadIdx.x] = st->active[threadIdx.x];
    }
    if (threadIdx.x == 0) { s_misc[0] = st->iter; s_misc[1] = st->max_iter; s_misc[2] = st->breakdown; }
    const double tol2 = st->tol2;
    __syncthreads();
    const bool live = s_active[k] != 0;
    double alpha_d = 0.0;
    if (live) alpha_d = (s_pq[k] > 0.0 && isfinite(s_pq[k])) ? s_rho[k] / s_pq[k] : 0.0;
    const T alpha = (T)alpha_d;
    const size_t nvec = nreal / N, base = (size_t)k * nreal;
    V* xv = reinterpret_cast<V*>(x + base);
    V* rv = reinterpret_cast<V*>(r + base);
    V* pv = reinterpret_cast<V*>(p + base);
    const V* qv = reinterpret_cast<const V*>(q + base);
    T rk[KEEP][N], pk[KEEP][N];
    double sum = 0.0;
#pragma unroll
    for (int j = 0; j < KEEP; ++j) {
        const size_t i = ((size_t)blockIdx.x * KEEP + j) * kBlasBlock + threadIdx.x;
        if (live && i < nvec) {
            T a[N], d[N];
            unpack16<T>(xv[i], a); unpack16<T>(rv[i], rk[j]); unpack16<T>(pv[i], pk[j]); unpack16<T>(qv[i], d);
#pragma unroll
            for (int e = 0; e < N; ++e) {
                a[e] = fma(alpha, pk[j][e], a[e]);
                rk[j][e] = fma(-alpha, d[e], rk[j][e]);
                sum += (double)rk[j][e] * (double)rk[j][e];
            }
            xv[i] = pack16<T>(a);
            rv[i] = pack16<T>(rk[j]);
        }
    }
    // block partial (same two-stage order as grid_reduce)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if (lane == 0) s_warp[warp] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < NW; ++w) s += s_warp[w];
        partial[(size_t)k * gx + blockIdx.x] = s;
        __threadfence();
    }
    grid.sync();
    // every block rebuilds all rho'_k identically (fixed order), so no second barrier is needed
    for (int kk = warp; kk < n; kk += NW) {
        double s = 0.0;
        for (int i = lane; i < gx; i += 32) s += __ldcg(partial + (size_t)kk * gx + i);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) s_rn[kk] = s;
    }
    __syncthreads();
    int any = 0, brk = s_misc[2];
    double beta_k = 0.0;
    bool my_active = false;
    for (int kk = 0; kk < n; ++kk) {
        if (!s_active[kk]) continue;
        const double rn = s_rn[kk], pq = s_pq[kk];
        if (!(pq > 0.0) || !isfinite(pq) || !isfinite(rn)) brk = 1;
        const bool still = !(rn <= tol2 * s_bn2[kk]);
        any |= still ? 1 : 0;
        if (kk == k) { beta_k = rn / s_rho[kk]; my_active = still; }
    }
    const int it = s_misc[0] + 1;
    const bool done = !any || it >= s_misc[1] || brk;
    if (blockIdx.x == 0 && blockIdx.y == 0) {
        if (threadIdx.x < n && s_active[threadIdx.x]) {
            const int kk = threadIdx.x;
            const double rn = s_rn[kk];
            st->rho_prev[kk] = s_rho[kk];
            st->beta[kk] = rn / s_rho[kk];
            st->rho[kk] = rn;
            if (rn <= tol2 * s_bn2[kk]) st->active[kk] = 0;
        }
        if (threadIdx.x == 0) {
            st->iter = it;
            if (brk) st->breakdown = 1;
            if (done) st->done = 1;
        }
    }
    if (!do_p || done || !my_active) return;
    const T beta = (T)beta_k;
#pragma unroll
    for (int j = 0; j < KEEP; ++j) {
        const size_t i = ((size_t)blockIdx.x * KEEP + j) * kBlasBlock + threadIdx.x;
        if (i < nvec) {
#pragma unroll
            for (int e = 0; e < N; ++e) pk[j][e] = fma(beta, pk[j][e], rk[j][e]);
            pv[i] = pack16<T>(pk[j]);
        }
    }
}

// ---- full-lattice solve M x = b (hisq_solve_M): norms and the odd-site reconstruction ------------------------------
// out[k] = ||a_k||^2 (+ ||b_k||^2 if b != nullptr), k = blockIdx.y, summed in fp64 in the fixed two-stage order
template <typename T>
__global__ void __launch_bounds__(kBlasBlock) norm2_kernel(const T* __restrict__ a, const T* __restrict__ b, size_t nreal, CgState* st,
                                                           double* partial, double* out)
{
    const int k = blockIdx.y;
    const size_t base = (size_t)k * nreal;
    double sum[1] = { 0.0 };
    for (int it = 0; it < kBlasItems * 4; ++it) {
        size_t i = ((size_t)blockIdx.x * kBlasItems * 4 + it) * kBlasBlock + threadIdx.x;
        if (i < nreal) {
            const double v = (double)a[base + i];
            sum[0] += v * v;
            if (b != nullptr) {
                const double w = (double)b[base + i];
                sum[0] += w * w;
            }
        }
    }
    __shared__ double totals[kMaxNrhs];
    if (grid_reduce<1, kBlasBlock>(sum, k, partial, gridDim.x, blockIdx.x, &st->ticket[0], gridDim.x * gridDim.y, gridDim.y, totals)) {
        if (threadIdx.x < gridDim.y) out[threadIdx.x] = totals[threadIdx.x];
    }
}

// x_o = (b_o - t) * inv_m   with t = D_oe x_e
template <typename T>
__global__ void __launch_bounds__(kBlasBlock) recon_odd_kernel(T* __restrict__ x, const T* __restrict__ b, const T* __restrict__ t,
                                                               size_t n, T inv_m)
{
    for (size_t i = (size_t)blockIdx.x * kBlasBlock + threadIdx.x; i < n; i += (size_t)gridDim.x * kBlasBlock)
        x[i] = (b[i] - t[i]) * inv_m;
}

// ---- partitioned-lattice CG (row f3): scalar updates that consume GLOBAL (all-reduced) sums ------------------------
__global__ void cgp_finalize_init_kernel(CgState* st, int n, double tol, int max_iter, const double* red = nullptr, int nranks = 0)
{
    int any = 0;
    for (int k = 0; k < n; ++k) {
        const double bb = red ? peer_sum(red, nranks, k) : st->rho[k];       // all-reduced ||b_k||^2
        st->rho[k] = bb;
        st->rho_prev[k] = bb; st->bnorm2[k] = bb; st->pq[k] = 1.0; st->beta[k] = 0.0; st->sums[k] = 0.0;
        st->active[k] = bb > 0.0 ? 1 : 0;
        any |= st->active[k];
    }
    st->tol2 = tol * tol; st->iter = 0; st->max_iter = max_iter; st->breakdown = 0; st->nrhs = n;
    st->done = any ? 0 : 1;
}

__global__ void cgp_finalize_xr_kernel(CgState* st, int n, const double* red_sums = nullptr, int nranks = 0)
{
    if (st->done) return;
    int any = 0;
    for (int k = 0; k < n; ++k) {
        if (st->active[k]) {
            const double rn = red_sums ? peer_sum(red_sums, nranks, k) : st->sums[k], pq = st->pq[k];   // both all-reduced
            if (!(pq > 0.0) || !isfinite(pq) || !isfinite(rn)) st->breakdown = 1;
            st->rho_prev[k] = st->rho[k];
            st->beta[k] = rn / st->rho[k];
            st->rho[k] = rn;
            if (rn <= st->tol2 * st->bnorm2[k]) st->active[k] = 0;
        }
        any |= st->active[k];
    }
    const int it = st->iter + 1;
    st->iter = it;
    if (!any || it >= st->max_iter || st->breakdown) st->done = 1;
}

// zero everything outside the owned box (t and, with a z cut, z) of a native field, so that sums over the whole extended
// array are sums over the owned sites.  S = complex per time slice, HLy = complex per z plane.
template <typename T>
__global__ void __launch_bounds__(256) zero_halo_kernel(T* __restrict__ field, int S, int Lt_ext, int t_lo, int t_cnt, int nrhs,
                                                        int HLy = 0, int z_lo = 0, int z_cnt = 0)
{
    using C = typename Vec<T>::c1;
    C* f = reinterpret_cast<C*>(field);
    const size_t total = (size_t)nrhs * 3 * Lt_ext * S;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
        const int t = (int)((i / S) % Lt_ext);
        bool out = t < t_lo || t >= t_lo + t_cnt;
        if (HLy > 0) {
            const int z = (int)((i % S) / HLy);
            out = out || z < z_lo || z >= z_lo + z_cnt;
        }
        if (out) { C zero; zero.x = 0; zero.y = 0; f[i] = zero; }
    }
}

// ---- after a true-residual recomputation (sums[k] = ||b_k - A x_k||^2): reliable-update bookkeeping ---
// rho_k = rho_true; beta_k = rho_true / rho_prev (search direction kept; frozen RHS kept
// theirs too, see cg_update_p_kernel); `done` is re-evaluated.
__global__ void cg_after_residual_kernel(CgState* st, double* true_rr_out)
{
    const int n = st->nrhs;
    int any = 0;
    for (int k = 0; k < n; ++k) {
        const double rt = st->sums[k];
        true_rr_out[k] = rt;
        const bool conv = rt <= st->tol2 * st->bnorm2[k];
        // keep the search direction while the recomputed residual is consistent with the recursive one;
        // if it drifted far (rt > 4 rho: the recursion was below the attainable accuracy) restart with p = r
        const bool consistent = rt <= 4.0 * st->rho[k];
        st->beta[k] = (!conv && consistent && st->rho_prev[k] > 0.0) ? rt / st->rho_prev[k] : 0.0;
        st->rho[k] = rt;
        st->active[k] = (!conv && st->bnorm2[k] > 0.0) ? 1 : 0;
        st->xpend[k] = -1;   // the caller flushed the pending x-update before recomputing the residual
        any |= st->active[k];
    }
    st->done = (!any || st->iter >= st->max_iter || st->breakdown) ? 1 : 0;
}

// ---- mixed precision helpers ------------------------------------------------------------------------
// x_hi += x_lo ; x_lo = 0
__global__ void __launch_bounds__(kBlasBlock) acc_xhi_kernel(double* __restrict__ xhi, float* __restrict__ xlo, size_t n)
{
    size_t i = ((size_t)blockIdx.x * kBlasBlock + threadIdx.x) * 4;
    if (i + 3 < n) {
        float4 lo = *reinterpret_cast<float4*>(xlo + i);
        double2 a = *reinterpret_cast<double2*>(xhi + i), b = *reinterpret_cast<double2*>(xhi + i + 2);
        a.x += (double)lo.x; a.y += (double)lo.y; b.x += (double)lo.z; b.y += (double)lo.w;
        *reinterpret_cast<double2*>(xhi + i) = a;
        *reinterpret_cast<double2*>(xhi + i + 2) = b;
        *reinterpret_cast<float4*>(xlo + i) = make_float4(0.f, 0.f, 0.f, 0.f);
    } else {
        for (; i < n; ++i) { xhi[i] += (double)xlo[i]; xlo[i] = 0.f; }
    }
}

template <typename TS, typename TD>
__global__ void __launch_bounds__(kBlasBlock) convert_kernel(const TS* __restrict__ src, TD* __restrict__ dst, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * kBlasBlock + threadIdx.x; i < n; i += (size_t)gridDim.x * kBlasBlock)
        dst[i] = (TD)src[i];
}

// ---- layout conversion: canonical (k,h,c) <-> native (k,c,h) -----------------------------------------
template <typename T, bool TO_NATIVE>
__global__ void __launch_bounds__(256) spinor_layout_kernel(T* __restrict__ dst, const T* __restrict__ src, int Vh, int nrhs)
{
    using C = typename Vec<T>::c1;
    const C* s = reinterpret_cast<const C*>(src);
    C* d = reinterpret_cast<C*>(dst);
    const size_t total = (size_t)nrhs * 3 * Vh;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
        // i enumerates the NATIVE order (k, c, h): coalesced on the native side
        const int h = (int)(i % Vh);
        const size_t kc = i / Vh;
        const int c = (int)(kc % 3);
        const size_t k = kc / 3;
        const size_t j = (k * Vh + h) * 3 + c;  // canonical
        if (TO_NATIVE) d[i] = s[j];
        else d[j] = s[i];
    }
}

// ---- t-halo pack / unpack (row f3): native field [k][c][slice][S] complex, S = sites of one parity per time slice.
// H = 3 slices move (the reach of the stencil); the 4th halo slice on each side only keeps parities aligned, never read.
// PACK:   lo <- interior slices [t_lo, t_lo+H)            (goes to the previous rank's UPPER halo)
//         hi <- interior slices [t_lo+t_cnt-H, t_lo+t_cnt) (goes to the next rank's LOWER halo)
// UNPACK: lower halo [t_lo-H, t_lo) <- lo (received from the previous rank), upper halo [t_lo+t_cnt, +H) <- hi.
// Buffers are [k][c][H*S] complex.
// sig_a / sig_b (PACK into peer mailboxes only, else null): arrival counters in the two neighbours' mailboxes, bumped
// once by the last CTA after every CTA's stores have been fenced at system scope -- the kernel signals, nothing waits.
template <typename T, bool PACK>
__global__ void __launch_bounds__(256) halo_kernel(T* __restrict__ field, T* __restrict__ lo, T* __restrict__ hi, int S, int Lt_ext,
                                                   int t_lo, int t_cnt, int H, int nrhs, unsigned* ticket, unsigned* sig_a,
                                                   unsigned* sig_b)
{
    using C = typename Vec<T>::c1;
    C* f = reinterpret_cast<C*>(field);
    C* l = reinterpret_cast<C*>(lo);
    C* u = reinterpret_cast<C*>(hi);
    const size_t chunk = (size_t)H * S, total = (size_t)nrhs * 3 * chunk;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
        const size_t kc = i / chunk, j = i % chunk;
        const size_t plane = kc * (size_t)Lt_ext * S;
        if (PACK) {
            l[i] = f[plane + (size_t)t_lo * S + j];
            u[i] = f[plane + (size_t)(t_lo + t_cnt - H) * S + j];
        } else {
            f[plane + (size_t)(t_lo - H) * S + j] = l[i];
            f[plane + (size_t)(t_lo + t_cnt) * S + j] = u[i];
        }
    }
    if (PACK && sig_a != nullptr) {
        // the barrier orders the CTA's stores before thread 0's fence, which is cumulative (the grid.sync idiom):
        // one system-scope fence per CTA instead of one per thread
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence_system();
            const unsigned done = atomicAdd(ticket, 1u);
            if (done == gridDim.x - 1) {
                *ticket = 0;
                __threadfence_system();
                atomicAdd_system(sig_a, 1u);
                atomicAdd_system(sig_b, 1u);
            }
        }
    }
}

// ---- z-halo pack / unpack (second cut): H = 3 planes of HLy complex on each side, for the OWNED time slices only (the
// stencil is axis-aligned: a site reads its z-neighbours at its own t).  Buffers are [k][c][t_cnt][H*HLy] complex; the H
// planes of one slice are one contiguous run.  Signalling as in halo_kernel.
template <typename T, bool PACK>
__global__ void __launch_bounds__(256) zhalo_kernel(T* __restrict__ field, T* __restrict__ lo, T* __restrict__ hi, int HLy, int S,
                                                    int Lt_ext, int t_lo, int t_cnt, int z_lo, int z_cnt, int H, int nrhs,
                                                    unsigned* ticket, unsigned* sig_a, unsigned* sig_b)
{
    using C = typename Vec<T>::c1;
    C* f = reinterpret_cast<C*>(field);
    C* l = reinterpret_cast<C*>(lo);
    C* u = reinterpret_cast<C*>(hi);
    const size_t chunk = (size_t)H * HLy, per_kc = (size_t)t_cnt * chunk, total = (size_t)nrhs * 3 * per_kc;
    for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
        const size_t kc = i / per_kc, rem = i % per_kc;
        const size_t tt = rem / chunk, j = rem % chunk;
        const size_t base = (kc * Lt_ext + t_lo + tt) * (size_t)S;
        if (PACK) {
            l[i] = f[base + (size_t)z_lo * HLy + j];
            u[i] = f[base + (size_t)(z_lo + z_cnt - H) * HLy + j];
        } else {
            f[base + (size_t)(z_lo - H) * HLy + j] = l[i];
            f[base + (size_t)(z_lo + z_cnt) * HLy + j] = u[i];
        }
    }
    if (PACK && sig_a != nullptr) {
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence_system();
            const unsigned done = atomicAdd(ticket, 1u);
            if (done == gridDim.x - 1) {
                *ticket = 0;
                __threadfence_system();
                atomicAdd_system(sig_a, 1u);
                atomicAdd_system(sig_b, 1u);
            }
        }
    }
}

// ---- all-reduce of nrhs doubles through peer-mapped mailboxes (row f3): every rank stores its local sums into EVERY
// rank's mailbox (slot, source rank) and bumps that mailbox's arrival counter; after a stream wait on its own counter
// each rank adds the contributions in rank order -- the same order everywhere, so all ranks hold the same bits.
__global__ void __launch_bounds__(32) peer_reduce_send_kernel(const double* __restrict__ src, PeerBoxes pb, int rank, int slot, int n,
                                                               size_t data_off, size_t counter_off)
{
    char* box = pb.box[blockIdx.x];       // one CTA per destination rank (my own mailbox included)
    double* dst = reinterpret_cast<double*>(box + data_off) + ((size_t)slot * kMaxRanks + rank) * kMaxNrhs;
    if (threadIdx.x < n) {
        dst[threadIdx.x] = src[threadIdx.x];
        __threadfence_system();
    }
    __syncwarp();
    if (threadIdx.x == 0) atomicAdd_system(reinterpret_cast<unsigned*>(box + counter_off) + slot, 1u);
}

// Abort path of the mailbox protocol: a rank that leaves a multi-rank solve with an error raises every rank's abort word and
// adds a poison value to all four arrival counters of every mailbox, so that every stream wait (">= expected") anywhere
// passes at once and no peer's stream stays parked on a counter that will never arrive; the peers see the abort word at
// their next status poll.  One thread per (mailbox, counter).
constexpr unsigned kMboxPoison = 0x40000000u;
constexpr int kMboxAbortWord = 15;
__global__ void __launch_bounds__(96) peer_abort_kernel(PeerBoxes pb, int nranks)
{
    const int r = threadIdx.x / 6, c = threadIdx.x % 6;
    if (r >= nranks || pb.box[r] == nullptr) return;
    unsigned* counters = reinterpret_cast<unsigned*>(pb.box[r]);
    const int idx[6] = { 0, 1, 8, 9, 2, 3 };   // t-halo slots 0, 1; reduce slots 0, 1; z-halo slots 0, 1
    if (c == 0) atomicExch_system(counters + kMboxAbortWord, 1u);
    __threadfence_system();
    atomicAdd_system(counters + idx[c], kMboxPoison);
}

__global__ void __launch_bounds__(32) peer_reduce_sum_kernel(double* __restrict__ dst, const char* __restrict__ mybox, int nranks, int slot,
                                                              int n, size_t data_off)
{
    const volatile double* d = reinterpret_cast<const volatile double*>(mybox + data_off) + (size_t)slot * kMaxRanks * kMaxNrhs;
    if (threadIdx.x < n) {
        double s = 0.0;
        for (int r = 0; r < nranks; ++r) s += d[(size_t)r * kMaxNrhs + threadIdx.x];
        dst[threadIdx.x] = s;
    }
}

}  // namespace hisq

// ===== multi-shift CG (row f1; PAPER.md:141 AdvancedMultiShiftCG): (A + sigma_k) x_k = b for all k with ONE
// operator application per iteration, on the smallest shift; the other shifts cost only these AXPYs. ==========
namespace hisq {

// zeta_k^{n+1} from the three-term recurrences of the base and the shifted system (derivation in DESIGN.md):
//   zeta' = zeta zeta_prev alpha_old / ( alpha_old zeta_prev (1 + delta alpha) + alpha beta_old (zeta_prev - zeta) )
__device__ __forceinline__ double ms_zeta_next(double zeta, double zeta_prev, double alpha, double alpha_old, double beta_old,
                                               double delta)
{
    const double den = alpha_old * zeta_prev * (1.0 + delta * alpha) + alpha * beta_old * (zeta_prev - zeta);
    return zeta * zeta_prev * alpha_old / den;
}

// One thread: with rn = ||r||^2 of the new residual, advance every scalar recurrence of the multi-shift iteration
// (alpha from the state as ms_update_xr_kernel formed it: rho and pq are still those of this iteration).
__device__ __forceinline__ void ms_advance(CgState* st, double rn, int nshift)
{
    const double pq = st->pq[0];
    const bool ok = pq > 0.0 && isfinite(pq);
    const double alpha = ok ? st->rho[0] / pq : 0.0;
    const double alpha_old = st->ms_alpha_old, beta_old = st->ms_beta_old;
    if (!ok || !isfinite(rn)) st->breakdown = 1;
    const double beta = rn / st->rho[0];
    int any = 0;
    for (int s = 0; s < nshift; ++s) {
        if (!st->active[s]) continue;
        const double z = st->ms_zeta[s];
        const double zn = ms_zeta_next(z, st->ms_zeta_prev[s], alpha, alpha_old, beta_old, st->ms_delta[s]);
        st->ms_beta_k[s] = beta * (zn / z) * (zn / z);
        st->ms_zeta_prev[s] = z;
        st->ms_zeta[s] = zn;
        if (!isfinite(zn)) st->breakdown = 1;
        // ||r_s|| = |zeta_s| ||r||; stop at half the requested tolerance (recursion drift margin)
        if (zn * zn * rn <= 0.25 * st->tol2 * st->bnorm2[0]) st->active[s] = 0;
        any |= st->active[s];
    }
    st->rho_prev[0] = st->rho[0];
    st->rho[0] = rn;
    st->ms_alpha_old = alpha;
    st->ms_beta_old = beta;
    const int it = st->iter + 1;
    st->iter = it;
    if (!any || it >= st->max_iter || st->breakdown) st->done = 1;
}

// start: r = b, x_k = 0 and p_k = 0 are memset by the host; rho = ||b||^2
template <typename T>
__global__ void __launch_bounds__(kBlasBlock) ms_init_kernel(const T* __restrict__ b, T* __restrict__ r, size_t nreal, CgState* st,
                                                             double* partial, double tol, int max_iter, int nshift)
{
    double sum[1] = { 0.0 };
    for (int it = 0; it < kBlasItems * 4; ++it) {
        size_t i = ((size_t)blockIdx.x * kBlasItems * 4 + it) * kBlasBlock + threadIdx.x;
        if (i < nreal) {
            T v = b[i];
            r[i] = v;
            sum[0] += (double)v * (double)v;
        }
    }
    __shared__ double totals[kMaxNrhs];
    if (grid_reduce<1, kBlasBlock>(sum, 0, partial, gridDim.x, blockIdx.x, &st->ticket[0], gridDim.x, 1, totals)) {
        if (threadIdx.x == 0) {
            const double bb = totals[0];
            st->rho[0] = bb; st->rho_prev[0] = bb; st->bnorm2[0] = bb; st->pq[0] = 1.0; st->beta[0] = 0.0;
            for (int k = 0; k < nshift; ++k) {
                st->ms_zeta[k] = 1.0; st->ms_zeta_prev[k] = 1.0; st->ms_beta_k[k] = 0.0;
                st->active[k] = bb > 0.0 ? 1 : 0;
                st->bnorm2[k] = bb;
            }
            st->ms_alpha_old = 1.0; st->ms_beta_old = 0.0; st->ms_nshift = nshift;
            st->tol2 = tol * tol; st->iter = 0; st->max_iter = max_iter; st->breakdown = 0; st->nrhs = nshift;
            st->done = bb > 0.0 ? 0 : 1;
        }
    }
}

// p_k = zeta_k r + beta_k p_k   (blockIdx.y = shift k)
template <typename T>
__global__ void __launch_bounds__(kBlasBlock) ms_update_p_kernel(T* __restrict__ p, const T* __restrict__ r, size_t nreal,
                                                                 const CgState* st)
{
    if (st->done) return;
    using V = typename V16<T>::type;
    constexpr int N = V16<T>::n;
    const int k = blockIdx.y;
    if (!st->active[k]) return;
    const T zeta = (T)st->ms_zeta[k], beta = (T)st->ms_beta_k[k];
    const size_t nvec = nreal / N;
    V* pv = reinterpret_cast<V*>(p + (size_t)k * nreal);
    const V* rv = reinterpret_cast<const V*>(r);
#pragma unroll
    for (int it = 0; it < kBlasItems; ++it) {
        size_t i = ((size_t)blockIdx.x * kBlasItems + it) * kBlasBlock + threadIdx.x;
        if (i < nvec) {
            T a[N], b[N];
            unpack16<T>(rv[i], a); unpack16<T>(pv[i], b);
#pragma unroll
            for (int e = 0; e < N; ++e) b[e] = fma(beta, b[e], zeta * a[e]);
            pv[i] = pack16<T>(b);
        }
    }
}

// blockIdx.y < nshift: x_k += alpha_k p_k with alpha_k = alpha zeta_k^{n+1} / zeta_k^n
// blockIdx.y == nshift: r -= alpha q, rho' = ||r||^2; the last block advances every scalar recurrence
template <typename T>
__global__ void __launch_bounds__(kBlasBlock) ms_update_xr_kernel(T* __restrict__ x, T* __restrict__ r, const T* __restrict__ p,
                                                                  const T* __restrict__ q, size_t nreal, CgState* st, double* partial,
                                                                  int defer = 0)
{
    if (st->done) return;
    using V = typename V16<T>::type;
    constexpr int N = V16<T>::n;
    const int nshift = gridDim.y - 1;
    const int k = blockIdx.y;
    const double pq = st->pq[0];
    const bool ok = pq > 0.0 && isfinite(pq);
    const double alpha = ok ? st->rho[0] / pq : 0.0;
    const double alpha_old = st->ms_alpha_old, beta_old = st->ms_beta_old;
    const size_t nvec = nreal / N;
    double sum[1] = { 0.0 };
    if (k < nshift) {
        if (st->active[k]) {
            const double z = st->ms_zeta[k];
            const double zn = ms_zeta_next(z, st->ms_zeta_prev[k], alpha, alpha_old, beta_old, st->ms_delta[k]);
            const T ak = (T)(alpha * zn / z);
            V* xv = reinterpret_cast<V*>(x + (size_t)k * nreal);
            const V* pv = reinterpret_cast<const V*>(p + (size_t)k * nreal);
#pragma unroll
            for (int it = 0; it < kBlasItems; ++it) {
                size_t i = ((size_t)blockIdx.x * kBlasItems + it) * kBlasBlock + threadIdx.x;
                if (i < nvec) {
                    T a[N], b[N];
                    unpack16<T>(xv[i], a); unpack16<T>(pv[i], b);
#pragma unroll
                    for (int e = 0; e < N; ++e) a[e] = fma(ak, b[e], a[e]);
                    xv[i] = pack16<T>(a);
                }
            }
        }
    } else {
        const T al = (T)alpha;
        V* rv = reinterpret_cast<V*>(r);
        const V* qv = reinterpret_cast<const V*>(q);
#pragma unroll
        for (int it = 0; it < kBlasItems; ++it) {
            size_t i = ((size_t)blockIdx.x * kBlasItems + it) * kBlasBlock + threadIdx.x;
            if (i < nvec) {
                T a[N], b[N];
                unpack16<T>(rv[i], a); unpack16<T>(qv[i], b);
#pragma unroll
                for (int e = 0; e < N; ++e) {
                    a[e] = fma(-al, b[e], a[e]);
                    sum[0] += (double)a[e] * (double)a[e];
                }
                rv[i] = pack16<T>(a);
            }
        }
    }
    __shared__ double totals[kMaxNrhs];
    // row 0 of `partial` collects the residual norm; x-blocks contribute zeros to their own rows (never summed)
    if (grid_reduce<1, kBlasBlock>(sum, k < nshift ? 1 : 0, partial, gridDim.x, blockIdx.x, &st->ticket[1], gridDim.x * gridDim.y,
                                   1, totals)) {
        if (threadIdx.x == 0) {
            if (defer) st->sums[0] = totals[0];   // partitioned lattice: the LOCAL sum; ms_finalize_kernel after the all-reduce
            else ms_advance(st, totals[0], nshift);
        }
    }
}

// partitioned lattice: the scalar recurrences once ||r||^2 (st->sums[0]) has been all-reduced
__global__ void ms_finalize_kernel(CgState* st, int nshift)
{
    if (st->done) return;
    ms_advance(st, st->sums[0], nshift);
}

// partitioned lattice: state from the all-reduced ||b||^2 (st->rho[0]) after ms_init_kernel ran on the local part
__global__ void ms_finalize_init_kernel(CgState* st, int nshift)
{
    const double bb = st->rho[0];
    st->rho_prev[0] = bb; st->bnorm2[0] = bb;
    for (int k = 0; k < nshift; ++k) { st->active[k] = bb > 0.0 ? 1 : 0; st->bnorm2[k] = bb; }
    st->done = bb > 0.0 ? 0 : 1;
}

}  // namespace hisq
