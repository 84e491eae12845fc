// dslash_launch_impl.cuh -- included by exactly one .cu per precision (explicit instantiation).
#pragma once
#include "dslash_launch.cuh"

namespace hisq {

template <typename T, int NR, int MODE>
static cudaError_t launch_one(const DslashArgs<T>& a, dim3 grid, cudaStream_t s)
{
#if HISQ_PDL
    // programmatic dependent launch: the CTAs of this launch may become resident while the previous kernel of the
    // stream drains its last wave; they wait in griddepcontrol.wait (top of dslash_kernel) until it has completed
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(kDslashBlock); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    if (a.naik_c14) return cudaLaunchKernelEx(&cfg, dslash_kernel<T, NR, MODE, kDslashBlock, true>, a);
    return cudaLaunchKernelEx(&cfg, dslash_kernel<T, NR, MODE, kDslashBlock, false>, a);
#else
    if (a.naik_c14) dslash_kernel<T, NR, MODE, kDslashBlock, true><<<grid, kDslashBlock, 0, s>>>(a);
    else dslash_kernel<T, NR, MODE, kDslashBlock, false><<<grid, kDslashBlock, 0, s>>>(a);
    return cudaGetLastError();
#endif
}

template <typename T, int NR>
static cudaError_t launch_mode(const DslashArgs<T>& a, int mode, dim3 grid, cudaStream_t s)
{
    switch (mode) {
    case MODE_PLAIN: return launch_one<T, NR, MODE_PLAIN>(a, grid, s);
    case MODE_APPLY_A: return launch_one<T, NR, MODE_APPLY_A>(a, grid, s);
    default: return launch_one<T, NR, MODE_RESID>(a, grid, s);
    }
}

static const int kInnerSizes[6] = { 8, 6, 4, 3, 2, 1 };

template <typename T>
int launch_dslash(DslashArgs<T> args, int mode, int nrhs, int inner_cap, cudaStream_t stream, LaunchStats* stats)
{
    const Geom& g = args.g;
    const int slab = g.H * g.ty * g.tz;
    args.slab_blocks = (slab + kDslashBlock - 1) / kDslashBlock;
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
        dim3 grid((unsigned)(a.slab_blocks * a.nchunks), (unsigned)a.tn, (unsigned)ntiles);
        cudaError_t e;
        switch (plan_nr[i]) {
        case 8: e = launch_mode<T, 8>(a, mode, grid, stream); break;
        case 6: e = launch_mode<T, 6>(a, mode, grid, stream); break;
        case 4: e = launch_mode<T, 4>(a, mode, grid, stream); break;
        case 3: e = launch_mode<T, 3>(a, mode, grid, stream); break;
        case 2: e = launch_mode<T, 2>(a, mode, grid, stream); break;
        default: e = launch_mode<T, 1>(a, mode, grid, stream); break;
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
    case MODE_PLAIN: e = cudaFuncGetAttributes(&at, dslash_kernel<T, NR, MODE_PLAIN, kDslashBlock, false>); break;
    case MODE_APPLY_A: e = cudaFuncGetAttributes(&at, dslash_kernel<T, NR, MODE_APPLY_A, kDslashBlock, false>); break;
    default: e = cudaFuncGetAttributes(&at, dslash_kernel<T, NR, MODE_RESID, kDslashBlock, false>); break;
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
