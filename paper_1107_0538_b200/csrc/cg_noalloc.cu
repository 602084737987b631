// cg_noalloc.cu -- cg_dot_static: the dot product of include/cg.h (the CGLoop's scalar
// products) for callers that may not allocate: no handle, no workspace, no cudaMalloc / cudaHostAlloc /
// malloc anywhere on its path.  Its scratch (the per-block partial sums that cg_dot keeps in the handle's
// workspace) lives in a file-scope __device__ array of fixed size, which every GPU that loads the library
// holds until the process exits: 32 KB.
//
// The array's NAME is, in host code, a host-side stand-in and not a device address; the kernels get the
// address cudaGetSymbolAddress returns, looked up once per device with that device current.
#include "../../include/cg.h"
#include "cg_kernels.cuh"

#include <cuda_runtime.h>
#include <mutex>

namespace {
using namespace cgk;

constexpr int kChunk = 8192;                        // elements per block: 256 threads x 32
constexpr int kMaxPartials = 4096;                  // blocks per call at most
constexpr long long kMaxN = (long long)kChunk * kMaxPartials;      // 33 554 432 elements

static __device__ __align__(256) double g_dot_scratch[kMaxPartials];

// partial[blockIdx.x] = sum of a_i b_i over the block's chunk: every thread accumulates its 32 elements in
// index order (FMA), then the fixed-order block sum of cg_kernels.cuh.
__global__ void __launch_bounds__(kThreads) k_dot_static_partial(const double* __restrict__ a, const double* __restrict__ b,
                                                                 long long n, double* __restrict__ part) {
    __shared__ double sm[kWarps + 1];
    const long long base = (long long)blockIdx.x * kChunk;
    double acc = 0.0;
#pragma unroll 4
    for (int k = 0; k < kChunk / kThreads; ++k) {
        const long long i = base + (long long)k * kThreads + threadIdx.x;
        if (i < n) acc = fma(a[i], b[i], acc);
    }
    const double t = block_sum(acc, sm);
    if (threadIdx.x == 0) part[blockIdx.x] = t;
}

// One block: thread t adds partials t, t + 256, ... in that order, then the block sum.  Reads only the
// `nparts` entries the launch before it wrote, so nothing in the scratch has to start at zero.
__global__ void __launch_bounds__(kThreads) k_dot_static_final(const double* __restrict__ part, int nparts,
                                                               double* __restrict__ result) {
    __shared__ double sm[kWarps + 1];
    double acc = 0.0;
    for (int j = threadIdx.x; j < nparts; j += kThreads) acc += part[j];
    const double t = block_sum(acc, sm);
    if (threadIdx.x == 0) *result = t;
}

constexpr int kMaxDevices = 64;
std::mutex g_lock;
double* g_scratch_ptr[kMaxDevices];                 // device address of g_dot_scratch, per device; null = not looked up yet

// The device address of the scratch on the CURRENT device (set-up: once per device).
int scratch_address(double** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return CG_ECUDA; }
    std::lock_guard<std::mutex> guard(g_lock);
    if (!g_scratch_ptr[dev]) {
        double* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, g_dot_scratch) != cudaSuccess || !p) { cudaGetLastError(); return CG_ECUDA; }
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return CG_OK;
}

}  // namespace

extern "C" int64_t cg_dot_static_max_n(void) { return kMaxN; }

extern "C" int cg_dot_static(int64_t n, const double* d_a, const double* d_b, double* d_result, void* cuda_stream) {
    if (n < 0 || !d_result || (n > 0 && (!d_a || !d_b))) return CG_EINVAL;
    if (n > kMaxN) return CG_ETOOBIG;
    double* scratch = nullptr;
    const int rc = scratch_address(&scratch);
    if (rc != CG_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int nparts = (int)((n + kChunk - 1) / kChunk);
    if (nparts > 0) {
        k_dot_static_partial<<<nparts, kThreads, 0, st>>>(d_a, d_b, n, scratch);
        if (cudaGetLastError() != cudaSuccess) return CG_ECUDA;
    }
    k_dot_static_final<<<1, kThreads, 0, st>>>(scratch, nparts, d_result);
    if (cudaGetLastError() != cudaSuccess) return CG_ECUDA;
    return CG_OK;
}
