// noalloc.cu -- hisq_norm2_noalloc: the per-RHS squared norm ||a_k||^2 of a field (the reduction every CG start makes:
// cg_init_kernel / norm2_kernel in blas.cuh) for callers that cannot allocate: no context, no workspace, no cudaMalloc --
// code under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  The two-stage reduction needs
// scratch for the per-block partial sums and the last-block ticket; here that scratch is a file-scope __device__ array of
// a fixed size that every GPU loading the library holds until the process exits (2 MiB + 256 B).
//
// The array's NAME is a host-side stand-in in host code, not a device address: a kernel handed `g_scratch` from the host
// would fault (or, where the GPU can reach host memory, silently use the wrong memory).  The device address is obtained
// once per device, with that device current, by cudaGetSymbolAddress below and passed to the kernel.
//
// Every call shares the array (on one device): calls that OVERLAP on the GPU -- two streams, two host threads -- race on the
// partial sums and the ticket and give wrong results; calls on one stream, or otherwise ordered, are fine.  The array keeps
// the last call's contents: the partial sums are overwritten before they are read (every block of a launch writes its own
// column, the last block reads exactly those), the ticket must start at zero and is cleared on the stream before each launch.
#include "../../include/hisq.h"

#include <cuda_runtime.h>

#include <mutex>

#include "common.cuh"

namespace {

constexpr int kBlock = 256;
constexpr int kRealsPerBlock = kBlock * 16;            // the partition cg_init_kernel / norm2_kernel use: 4096 reals per block
constexpr size_t kTicketBytes = 256;
constexpr size_t kScratchBytes = kTicketBytes + (size_t)HISQ_NOALLOC_MAX_NRHS * HISQ_NOALLOC_MAX_COLS * sizeof(double);

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];   // [ticket, padded to 256 B][nrhs][cols] doubles

// out[k] = sum_i a[k][i]^2, k = blockIdx.y, fp64 accumulation, fixed summation order (hisq::grid_reduce): the same block
// partition and order as cg_init_kernel, so the result equals what a solve computes for ||b_k||^2 bit for bit.
template <typename T>
__global__ void __launch_bounds__(kBlock) norm2_static_kernel(const T* __restrict__ a, size_t nreal, unsigned char* scratch,
                                                              double* __restrict__ out)
{
    const int k = blockIdx.y;
    const size_t base = (size_t)k * nreal;
    double sum[1] = { 0.0 };
    for (int it = 0; it < kRealsPerBlock / kBlock; ++it) {
        const size_t i = ((size_t)blockIdx.x * (kRealsPerBlock / kBlock) + it) * kBlock + threadIdx.x;
        if (i < nreal) {
            const double v = (double)a[base + i];
            sum[0] += v * v;
        }
    }
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch);
    double* partial = reinterpret_cast<double*>(scratch + kTicketBytes);
    __shared__ double totals[hisq::kMaxNrhs];
    if (hisq::grid_reduce<1, kBlock>(sum, k, partial, gridDim.x, blockIdx.x, ticket, gridDim.x * gridDim.y, gridDim.y, totals)) {
        if (threadIdx.x < gridDim.y) out[threadIdx.x] = totals[threadIdx.x];
    }
}

// device address of g_scratch per device, resolved on first use with that device current
constexpr int kMaxDevices = 64;
std::mutex g_mutex;
unsigned char* g_addr[kMaxDevices] = { nullptr };

cudaError_t scratch_address(unsigned char** p)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_addr[dev]) {
        void* sym = nullptr;
        e = cudaGetSymbolAddress(&sym, g_scratch);       // no allocation: the array is part of the loaded module
        if (e != cudaSuccess) return e;
        g_addr[dev] = static_cast<unsigned char*>(sym);
    }
    *p = g_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" size_t hisq_norm2_noalloc_max_reals(void) { return (size_t)HISQ_NOALLOC_MAX_COLS * kRealsPerBlock; }

extern "C" int hisq_norm2_noalloc(const void* field, int prec, size_t nreal, int nrhs, double* out, void* cuda_stream)
{
    if (!field || !out || nreal == 0 || nrhs < 1 || ((uintptr_t)field & 15)) return HISQ_EINVAL;
    if (prec != HISQ_FP32 && prec != HISQ_FP64 && prec != HISQ_MIXED) return HISQ_EINVAL;
    // beyond the static scratch: refuse (nothing has been launched or touched)
    if (nrhs > HISQ_NOALLOC_MAX_NRHS || nreal > hisq_norm2_noalloc_max_reals()) return HISQ_ETOOBIG;
    unsigned char* scratch = nullptr;
    if (scratch_address(&scratch) != cudaSuccess) return HISQ_ECUDA;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (cudaMemsetAsync(scratch, 0, sizeof(unsigned), s) != cudaSuccess) return HISQ_ECUDA;   // the ticket starts at zero
    const dim3 grid((unsigned)((nreal + kRealsPerBlock - 1) / kRealsPerBlock), (unsigned)nrhs);
    if (prec == HISQ_FP32) norm2_static_kernel<float><<<grid, kBlock, 0, s>>>((const float*)field, nreal, scratch, out);
    else norm2_static_kernel<double><<<grid, kBlock, 0, s>>>((const double*)field, nreal, scratch, out);
    return cudaGetLastError() == cudaSuccess ? HISQ_OK : HISQ_ECUDA;
}
