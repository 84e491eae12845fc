// dslash_launch.cuh -- host-side launch plan of the Dslash kernel, shared by the per-precision
// translation units (dslash_f32.cu, dslash_f64.cu) and the API (hisq.cu).
#pragma once
#include "dslash.cuh"

namespace hisq {

struct LaunchStats { long long launches = 0; };

// Launch D (or its fused epilogue variants) for `nrhs` right-hand sides starting at args.in/out/u/v.
// `inner_cap`: most RHS one thread may hold (1,2,3,4,6,8); c14: the Naik links are stored compressed.
// Returns a cudaError_t as int.
template <typename T>
int launch_dslash(DslashArgs<T> args, int mode, int nrhs, int inner_cap, bool c14, cudaStream_t stream, LaunchStats* stats);

// Register count / attributes for introspection (tests, DESIGN.md tables).
template <typename T> int dslash_regs(int nr, int mode);

}  // namespace hisq
