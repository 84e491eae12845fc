// dslash_launch_impl.cuh -- included by exactly one .cu per precision (explicit instantiation).
#pragma once
#include "dslash_launch.cuh"

namespace hisq {

template <typename T, int NR, int MODE, bool NC>
static cudaError_t launch_kernel(const DslashArgs<T>& a, dim3 grid, cudaStream_t s)
{
    // programmatic dependent launch: the CTAs of this launch may become resident while the previous kernel of the
    // stream drains its last wave; they wait in griddepcontrol.wait (top of dslash_kernel) until it has completed
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(kDslashBlock); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, dslash_kernel<T, NR, MODE, NC>, a);
}

template <typename T, int NR, int MODE>
static cudaError_t launch_one(const DslashArgs<T>& a, bool c14, dim3 grid, cudaStream_t s)
{
    return c14 ? launch_kernel<T, NR, MODE, true>(a, grid, s) : launch_kernel<T, NR, MODE, false>(a, grid, s);
}

template <typename T, int NR>
static cudaError_t launch_mode(const DslashArgs<T>& a, int mode, bool c14, dim3 grid, cudaStream_t s)
{
    switch (mode) {
    case MODE_PLAIN: return launch_one<T, NR, MODE_PLAIN>(a, c14, grid, s);
    case MODE_APPLY_A: return launch_one<T, NR, MODE_APPLY_A>(a, c14, grid, s);
    default: return launch_one<T, NR, MODE_RESID>(a, c14, grid, s);
    }
}

static const int kInnerSizes[6] = { 8, 6, 4, 3, 2, 1 };

template <typename T>
int launch_dslash(DslashArgs<T> args, int mode, int nrhs, int inner_cap, bool c14, cudaStream_t stream, LaunchStats* stats)
{
    const Geom& g = args.g;
    // warp -> sites map of one (tile, t) slab: runs of consecutive half-indices (one x-y sheet of the tile, or the whole
    // slab when the tile spans y), each covered by whole warps on aligned blocks of 32 (dslash.cuh)
    args.merged = g.ty == g.L[1] ? 1 : 0;
    args.nseg = args.merged ? 1 : g.tz;
    args.seg_len = args.merged ? g.H * g.L[1] * g.tz : g.H * g.ty;
    args.wps = args.seg_len % 32 == 0 ? args.seg_len / 32 : (args.seg_len + 31) / 32 + 1;
    const int slab_warps = args.nseg * args.wps;
    args.slab_blocks = (slab_warps + kDslashWarps - 1) / kDslashWarps;
    const int ntiles = g.nty * g.ntz;
    const size_t rhs_stride = (size_t)6 * g.Vh;
    // plan: greedy split of nrhs into groups of equal NR
    int plan_nr[8], plan_cnt[8], nplan = 0, left = nrhs;
    while (left > 0) {
        int nr = 1;
        for (int i = 0; i < 6; ++i)
            if (kInnerSizes[i] <= left && kInnerSizes[i] <= inner_cap) { nr = kInnerSizes[i]; break; }
        plan_nr[nplan] = nr;
        plan_cnt[nplan] = left / nr;
        left -= nr * plan_cnt[nplan];
        ++nplan;
    }
    unsigned total = 0;
    for (int i = 0; i < nplan; ++i) total += (unsigned)args.slab_blocks * plan_cnt[i] * g.t_cnt * ntiles;
    args.total_blocks = total;
    args.nrhs_total = nrhs;
    int k = 0;
    for (int i = 0; i < nplan; ++i) {
        DslashArgs<T> a = args;
        a.in = args.in + (size_t)k * rhs_stride;
        a.out = args.out + (size_t)k * rhs_stride;
        if (args.u) a.u = args.u + (size_t)k * rhs_stride;
        if (args.v) a.v = args.v + (size_t)k * rhs_stride;
        a.k0 = k;
        a.nchunks = plan_cnt[i];
        a.wide_dot = args.wide_dot < 0 ? (plan_nr[i] <= 2 ? 1 : 0) : args.wide_dot;   // -1: widen where it is free
        dim3 grid((unsigned)(a.slab_blocks * a.nchunks), (unsigned)a.tn, (unsigned)ntiles);
        cudaError_t e;
        switch (plan_nr[i]) {
        case 8: e = launch_mode<T, 8>(a, mode, c14, grid, stream); break;
        case 6: e = launch_mode<T, 6>(a, mode, c14, grid, stream); break;
        case 4: e = launch_mode<T, 4>(a, mode, c14, grid, stream); break;
        case 3: e = launch_mode<T, 3>(a, mode, c14, grid, stream); break;
        case 2: e = launch_mode<T, 2>(a, mode, c14, grid, stream); break;
        default: e = launch_mode<T, 1>(a, mode, c14, grid, stream); break;
        }
        if (stats) stats->launches += 1;
        if (e != cudaSuccess) return (int)e;
        k += plan_nr[i] * plan_cnt[i];
    }
    return 0;
}

template <typename T, int NR>
static int regs_mode(int mode)
{
    cudaFuncAttributes at;
    cudaError_t e;
    switch (mode) {
    case MODE_PLAIN: e = cudaFuncGetAttributes(&at, dslash_kernel<T, NR, MODE_PLAIN, false>); break;
    case MODE_APPLY_A: e = cudaFuncGetAttributes(&at, dslash_kernel<T, NR, MODE_APPLY_A, false>); break;
    default: e = cudaFuncGetAttributes(&at, dslash_kernel<T, NR, MODE_RESID, false>); break;
    }
    return e == cudaSuccess ? at.numRegs : -1;
}

template <typename T> int dslash_regs(int nr, int mode)
{
    switch (nr) {
    case 8: return regs_mode<T, 8>(mode);
    case 6: return regs_mode<T, 6>(mode);
    case 4: return regs_mode<T, 4>(mode);
    case 3: return regs_mode<T, 3>(mode);
    case 2: return regs_mode<T, 2>(mode);
    default: return regs_mode<T, 1>(mode);
    }
}

}  // namespace hisq
