// dslash_f32.cu -- fp32 instantiations of the Dslash kernel.
#include "dslash_launch_impl.cuh"
namespace hisq {
template int launch_dslash<float>(DslashArgs<float>, int, int, int, bool, cudaStream_t, LaunchStats*);
template int dslash_regs<float>(int, int);
}
