// dslash_f64.cu -- fp64 instantiations of the Dslash kernel.
#include "dslash_launch_impl.cuh"
namespace hisq {
template int launch_dslash<double>(DslashArgs<double>, int, int, int, bool, cudaStream_t, LaunchStats*);
template int dslash_regs<double>(int, int);
}
