// cg_api.cu -- C ABI (include/cg.h) and kernel entry points of libcg_b200.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -shared -Xcompiler -fPIC
#include "../../include/cg.h"
#include "cg_kernels.cuh"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>

using namespace cgk;

// ---------------------------------------------------------------- kernels

namespace {

__device__ __forceinline__ bool is_finite(double v) { return fabs(v) <= 1.79769313486231570e308; }

// cg_create statistics: longest row, largest nnz span of a kTileRows-row tile.
__global__ void k_stats(const int* __restrict__ rowptr, long long n, Scal* scal) {
    int mrow = 0, mtile = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int len = rowptr[i + 1] - rowptr[i];
        mrow = max(mrow, len);
        if ((i % kTileRows) == 0) {
            const long long j = (i + kTileRows < n) ? i + kTileRows : n;
            mtile = max(mtile, rowptr[j] - rowptr[i]);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        mrow = max(mrow, __shfl_xor_sync(0xffffffffu, mrow, o));
        mtile = max(mtile, __shfl_xor_sync(0xffffffffu, mtile, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(&scal->max_row_len, mrow);
        atomicMax(&scal->max_tile_nnz, mtile);
    }
}

__global__ void k_check_csr(const int* __restrict__ rowptr, const int* __restrict__ colind,
                            long long n, long long nnz, Scal* scal) {
    int bad = 0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t0 == 0 && (rowptr[0] != 0 || (long long)rowptr[n] != nnz)) bad |= 1;
    for (long long i = t0; i < n; i += stride)
        if (rowptr[i + 1] < rowptr[i]) bad |= 2;
    for (long long k = t0; k < nnz; k += stride) {
        const int c = colind[k];
        if (c < 0 || (long long)c >= n) bad |= 4;
    }
    if (bad) atomicOr(&scal->check, bad);
}

// D^-1 from the CSR arrays (duplicates on the diagonal add).  Flags bit 8 when a
// diagonal entry is missing or not positive.
__global__ void k_diag_inv(Params P) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.n; i += stride) {
        double d = 0.0;
        for (int k = P.rowptr[i]; k < P.rowptr[i + 1]; ++k)
            if (P.colind[k] == i) d += P.vals[k];
        if (!(d > 0.0) || !is_finite(d)) { P.scal->diag_bad = 1; d = 1.0; }
        P.dinv[i] = 1.0 / d;
    }
}

template <int V>
__global__ void __launch_bounds__(kThreads, MinBlocks<V>::value) k_spmv(Params P, const double* x, double* y) {
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    stream_smem_init<V>(dyn_smem);
    uint32_t bits = 0;
    phase_spmv<V, false>(P, x, y, blockIdx.x, gridDim.x, dyn_smem, bits);
}

__global__ void __launch_bounds__(kThreads) k_dot_partial(const double* __restrict__ a,
                                                          const double* __restrict__ b,
                                                          long long n, double* part) {
    __shared__ double sm[kWarps + 1];
    double acc = 0.0;
    const long long stride = (long long)gridDim.x * kThreads;
    for (long long i = (long long)blockIdx.x * kThreads + threadIdx.x; i < n; i += stride)
        acc = fma(a[i], b[i], acc);
    const double t = block_sum(acc, sm);
    if (threadIdx.x == 0) part[blockIdx.x] = t;
}

__global__ void __launch_bounds__(kThreads) k_dot_final(const double* part, int G, Scal* scal) {
    __shared__ double sm[kWarps + 1];
    const double s = sum_partials(part, G, sm);
    if (threadIdx.x == 0) scal->dot_out = s;
}

// ---- stand-alone kernels of loop modes 1 (graph) and 2 (stepwise).  They read
// ---- Params from device memory so that a captured graph survives across solves.

template <int V>
__global__ void __launch_bounds__(kThreads, MinBlocks<V>::value) k_init_spmv(const Params* __restrict__ dp) {
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    const Params P = *dp;
    stream_smem_init<V>(dyn_smem);
    uint32_t bits = 0;
    phase_spmv<V, false>(P, P.x, P.q, blockIdx.x, gridDim.x, dyn_smem, bits);
}

__global__ void __launch_bounds__(kThreads, 2) k_init_residual(const Params* __restrict__ dp) {
    __shared__ double sm[kWarps + 1];
    const Params P = *dp;
    phase_init_residual(P, blockIdx.x, gridDim.x, sm);
}

// Everything the loop decides from (rr, rz, bb) before the first iteration.
__device__ __forceinline__ void init_decide(const Params& P, double rr, double bb, long long* k_out,
                                            int* stop, int* status, double* thresh) {
    *thresh = P.rtol * sqrt(bb);
    *k_out = 0;
    *stop = 0; *status = CG_OK;
    if (bb == 0.0 || sqrt(rr) <= *thresh) { *stop = 1; *status = CG_OK; }
    else if (P.maxit <= 0) { *stop = 1; *status = CG_MAXIT; }
}

__global__ void __launch_bounds__(kThreads) k_init_scalars(const Params* __restrict__ dp) {
    __shared__ double sm[kWarps + 1];
    const Params P = *dp;
    const int G = gridDim.x;
    double rr = sum_partials(P.part1, G, sm);
    const double bb = sum_partials(P.part2, G, sm);
    const double rz = P.precond ? sum_partials(P.part3, G, sm) : rr;
    if (bb == 0.0) { phase_zero_x(P, blockIdx.x, G); rr = 0.0; }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        long long k; int stop, status; double thresh;
        init_decide(P, rr, bb, &k, &stop, &status, &thresh);
        if (P.precond && P.scal->diag_bad) { stop = 1; status = CG_BREAKDOWN; }
        Scal* S = P.scal;
        S->bb = bb; S->thresh = thresh;
        S->st[0].rr = rr; S->st[0].rz = rz; S->st[0].k = 0; S->st[0].stop = stop; S->st[0].status = status;
        if (P.hist) P.hist[0] = sqrt(rr);
        S->out_iters = 0; S->out_status = status; S->out_res = sqrt(rr);
    }
}

template <int V>
__global__ void __launch_bounds__(kThreads, MinBlocks<V>::value) k1_spmv_dot(const Params* __restrict__ dp, int s) {
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    __shared__ double sm[kWarps + 1];
    const Params P = *dp;
    if (P.scal->st[s].stop) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) P.scal->brk[s] = 0;
    stream_smem_init<V>(dyn_smem);
    uint32_t bits = 0;
    const double d = phase_spmv<V, true>(P, P.p, P.q, blockIdx.x, gridDim.x, dyn_smem, bits);
    const double t = block_sum(d, sm);
    if (threadIdx.x == 0) P.part0[blockIdx.x] = t;
}

__global__ void __launch_bounds__(kThreads, 2) k2_update_xr(const Params* __restrict__ dp, int s) {
    __shared__ double sm[kWarps + 1];
    const Params P = *dp;
    if (P.scal->st[s].stop) return;
    const double pq = sum_partials(P.part0, gridDim.x, sm);
    if (!(pq > 0.0) || !is_finite(pq)) {
        if (blockIdx.x == 0 && threadIdx.x == 0) P.scal->brk[s] = 1;
        return;
    }
    const double alpha = P.scal->st[s].rz / pq;
    phase_update_xr<4>(P, alpha, blockIdx.x, gridDim.x, sm);
}

__global__ void __launch_bounds__(kThreads, 2) k3_update_p(const Params* __restrict__ dp, int s) {
    __shared__ double sm[kWarps + 1];
    const Params P = *dp;
    Scal* S = P.scal;
    const State st = S->st[s];
    const bool lead = blockIdx.x == 0 && threadIdx.x == 0;
    if (st.stop) { if (lead) S->st[s ^ 1] = st; return; }
    if (S->brk[s]) {
        if (lead) {
            State nx = st; nx.stop = 1; nx.status = CG_BREAKDOWN;
            S->st[s ^ 1] = nx;
            S->out_iters = st.k; S->out_status = CG_BREAKDOWN; S->out_res = sqrt(st.rr);
        }
        return;
    }
    const double rr = sum_partials(P.part1, gridDim.x, sm);
    const double rz = P.precond ? sum_partials(P.part2, gridDim.x, sm) : rr;
    const double beta = rz / st.rz;
    const long long k = st.k + 1;
    const double res = sqrt(rr);
    int stop = 0, status = CG_OK;
    if (res <= S->thresh) { stop = 1; status = CG_OK; }
    else if (k >= P.maxit) { stop = 1; status = CG_MAXIT; }
    if (lead) {
        State nx; nx.rr = rr; nx.rz = rz; nx.k = k; nx.stop = stop; nx.status = status;
        S->st[s ^ 1] = nx;
        if (P.hist) P.hist[k] = res;
        if (stop) { S->out_iters = k; S->out_status = status; S->out_res = res; }
    }
    if (!stop) phase_update_p<4>(P, beta, blockIdx.x, gridDim.x);
}

// ---- loop mode 0: the whole solve as ONE cooperative persistent kernel.
// Scalars live in registers, identical in every CTA; three grid barriers per
// iteration (after K1, K2, K3); nothing leaves the device until the end.
template <int V>
__global__ void __launch_bounds__(kThreads, MinBlocks<V>::value) k_persistent(Params P) {
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    __shared__ double sm[kWarps + 1];
    const int cta = blockIdx.x, G = gridDim.x;
    const bool lead = cta == 0 && threadIdx.x == 0;
    Scal* S = P.scal;
    unsigned long long epoch = 0;
    uint32_t bits = 0;
    stream_smem_init<V>(dyn_smem);

    // a0 prologue: q = A x0 ; r = b - q ; p = r ; rr, bb
    phase_spmv<V, false>(P, P.x, P.q, cta, G, dyn_smem, bits);
    grid_barrier(&S->bar, G, epoch);
    phase_init_residual(P, cta, G, sm);
    grid_barrier(&S->bar, G, epoch);
    double rr = sum_partials(P.part1, G, sm);
    const double bb = sum_partials(P.part2, G, sm);
    double rz = P.precond ? sum_partials(P.part3, G, sm) : rr;
    if (bb == 0.0) { phase_zero_x(P, cta, G); rr = 0.0; }
    long long k; int stop, status; double thresh;
    init_decide(P, rr, bb, &k, &stop, &status, &thresh);
    if (P.precond && S->diag_bad) { stop = 1; status = CG_BREAKDOWN; }
    if (lead && P.hist) P.hist[0] = sqrt(rr);

    while (!stop) {
        // K1
        const double d = phase_spmv<V, true>(P, P.p, P.q, cta, G, dyn_smem, bits);
        const double t = block_sum(d, sm);
        if (threadIdx.x == 0) P.part0[cta] = t;
        grid_barrier(&S->bar, G, epoch);
        // scalar alpha (every CTA, same order, same value)
        const double pq = sum_partials(P.part0, G, sm);
        if (!(pq > 0.0) || !is_finite(pq)) { stop = 1; status = CG_BREAKDOWN; break; }
        const double alpha = rz / pq;
        // K2
        phase_update_xr<(V == 2 ? 4 : 2)>(P, alpha, cta, G, sm);
        grid_barrier(&S->bar, G, epoch);
        // scalar beta, continue-condition
        const double rr_new = sum_partials(P.part1, G, sm);
        const double rz_new = P.precond ? sum_partials(P.part2, G, sm) : rr_new;
        const double beta = rz_new / rz;
        rr = rr_new; rz = rz_new; k += 1;
        const double res = sqrt(rr);
        if (lead && P.hist) P.hist[k] = res;
        if (res <= thresh) { stop = 1; status = CG_OK; break; }
        if (k >= P.maxit) { stop = 1; status = CG_MAXIT; break; }
        // K3
        phase_update_p<(V == 2 ? 4 : 2)>(P, beta, cta, G);
        grid_barrier(&S->bar, G, epoch);
    }
    if (lead) { S->out_iters = k; S->out_status = status; S->out_res = sqrt(rr); }
}

}  // namespace

// ---------------------------------------------------------------- host side

static thread_local char g_cuda_err[256] = "no CUDA error recorded";

#define CK(call)                                                              \
    do {                                                                      \
        cudaError_t e_ = (call);                                              \
        if (e_ != cudaSuccess) {                                              \
            snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s (%s:%d)",        \
                     cudaGetErrorName(e_), cudaGetErrorString(e_), __FILE__, __LINE__); \
            cudaGetLastError();                                               \
            return CG_ECUDA;                                                  \
        }                                                                     \
    } while (0)

#include <stdio.h>

struct cg_handle {
    long long n, nnz;
    const int* rowptr; const int* colind; const double* vals;
    unsigned char* ws; size_t ws_bytes;
    double *r, *p, *q, *dinv, *spare, *part0, *part1, *part2, *part3;
    Scal* scal; Params* dparams;
    Scal* h_scal; Params* h_params;        // pinned host mirrors
    int sms;
    int loop, spmv_opt, chunk, ctas_per_sm;
    int max_row_len, max_tile_nnz, tpr;
    bool stream_ok, dinv_ready;
    int grid_v[3];                         // cooperative grid per SpMV variant (index 1, 2)
    cudaGraphExec_t gexec; int gexec_variant, gexec_chunk, gexec_grid;
    cudaStream_t cap_stream;               // capture-only stream (the legacy stream cannot capture)
    long long launches;
};

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static size_t vec_bytes(long long n) { return align_up((size_t)n * 8u, 256); }
static constexpr int kNumVecs = 5;
static constexpr size_t kPartBytes = (size_t)kMaxGrid * 8u;
static constexpr size_t kScalBytes = 512, kParamBytes = 512;

extern "C" size_t cg_workspace_bytes(int64_t n) {
    if (n <= 0) return 0;
    return kNumVecs * vec_bytes(n) + 4 * kPartBytes + kScalBytes + kParamBytes;
}

extern "C" size_t cg_host_scratch_bytes(int64_t n, int64_t maxit) {
    if (n <= 0 || maxit < 0) return 0;
    return 2 * vec_bytes(n) + align_up((size_t)(maxit + 1) * 8u, 256);
}

template <int V> static size_t variant_smem() { return V == 2 ? kStreamSmemBytes : 0; }

template <int V> static int setup_variant(cg_handle* h) {
    const size_t smem = variant_smem<V>();
    if (smem) {
        CK(cudaFuncSetAttribute(k_persistent<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CK(cudaFuncSetAttribute(k_spmv<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CK(cudaFuncSetAttribute(k_init_spmv<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CK(cudaFuncSetAttribute(k1_spmv_dot<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    }
    int bps = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_persistent<V>, kThreads, smem));
    if (bps < 1) { snprintf(g_cuda_err, sizeof(g_cuda_err), "persistent kernel does not fit an SM"); return CG_ECUDA; }
    int want = h->ctas_per_sm > 0 ? h->ctas_per_sm : (V == 2 ? 1 : 2);
    if (want > bps) want = bps;
    int g = h->sms * want;
    if (g > kMaxGrid) g = kMaxGrid;
    h->grid_v[V] = g;
    return CG_OK;
}

static int pick_variant(const cg_handle* h) {
    if (h->spmv_opt == 1) return 1;
    if (h->spmv_opt == 2) return h->stream_ok ? 2 : 1;
    return h->stream_ok ? 2 : 1;
}

static void fill_params(const cg_handle* h, Params* P, const double* b, double* x, double rtol,
                        long long maxit, double* hist, int precond, int variant) {
    P->n = h->n; P->nnz = h->nnz;
    P->rowptr = h->rowptr; P->colind = h->colind; P->vals = h->vals;
    P->b = b; P->x = x; P->r = h->r; P->p = h->p; P->q = h->q; P->dinv = h->dinv;
    P->part0 = h->part0; P->part1 = h->part1; P->part2 = h->part2; P->part3 = h->part3;
    P->scal = h->scal; P->hist = hist; P->rtol = rtol; P->maxit = maxit;
    P->precond = precond; P->spmv = variant; P->tpr = h->tpr;
}

extern "C" int cg_create(cg_handle** out, int64_t n, int64_t nnz, const int32_t* d_rowptr,
                         const int32_t* d_colind, const double* d_vals, void* d_workspace,
                         size_t workspace_bytes) {
    if (!out) return CG_EINVAL;
    *out = nullptr;
    if (n <= 0 || nnz < 0 || n >= (1LL << 31) - 1 || nnz >= (1LL << 31) - 8) return CG_EINVAL;
    if (!d_rowptr || !d_workspace || (nnz > 0 && (!d_colind || !d_vals))) return CG_EINVAL;
    if (!aligned16(d_rowptr) || !aligned16(d_colind) || !aligned16(d_vals)) return CG_EINVAL;
    if ((reinterpret_cast<uintptr_t>(d_workspace) & 255u) != 0) return CG_EINVAL;
    if (workspace_bytes < cg_workspace_bytes(n)) return CG_EINVAL;

    int dev = 0;
    CK(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return CG_EUNSUPPORTED;
    int coop = 0;
    CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    if (!coop) return CG_EUNSUPPORTED;

    cg_handle* h = new (std::nothrow) cg_handle();
    if (!h) return CG_EINVAL;
    memset(h, 0, sizeof(*h));
    h->n = n; h->nnz = nnz;
    h->rowptr = d_rowptr; h->colind = d_colind; h->vals = d_vals;
    h->ws = static_cast<unsigned char*>(d_workspace); h->ws_bytes = workspace_bytes;
    unsigned char* w = h->ws;
    const size_t vb = vec_bytes(n);
    h->r = (double*)w; w += vb; h->p = (double*)w; w += vb; h->q = (double*)w; w += vb;
    h->dinv = (double*)w; w += vb; h->spare = (double*)w; w += vb;
    h->part0 = (double*)w; w += kPartBytes; h->part1 = (double*)w; w += kPartBytes;
    h->part2 = (double*)w; w += kPartBytes; h->part3 = (double*)w; w += kPartBytes;
    h->scal = (Scal*)w; w += kScalBytes; h->dparams = (Params*)w; w += kParamBytes;
    static_assert(sizeof(Scal) <= kScalBytes && sizeof(Params) <= kParamBytes, "workspace slots");
    h->sms = prop.multiProcessorCount;
    h->loop = 0; h->spmv_opt = 0; h->chunk = 32; h->ctas_per_sm = 0;

    cudaError_t e = cudaHostAlloc((void**)&h->h_scal, sizeof(Scal), cudaHostAllocDefault);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&h->h_params, sizeof(Params), cudaHostAllocDefault);
    if (e != cudaSuccess) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cudaHostAlloc: %s", cudaGetErrorString(e));
        if (h->h_scal) cudaFreeHost(h->h_scal);
        delete h; cudaGetLastError();
        return CG_ECUDA;
    }
#define CKH(call) do { int rc_ = [&]() -> int { CK(call); return CG_OK; }(); \
        if (rc_ != CG_OK) { cg_destroy(h); return rc_; } } while (0)
    // matrix statistics (one pass over rowptr on the legacy default stream)
    CKH(cudaMemsetAsync(h->scal, 0, sizeof(Scal), 0));
    k_stats<<<h->sms * 4, 256, 0, 0>>>(h->rowptr, h->n, h->scal);
    CKH(cudaGetLastError());
    CKH(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, 0));
    CKH(cudaStreamSynchronize(0));
    h->max_row_len = h->h_scal->max_row_len;
    h->max_tile_nnz = h->h_scal->max_tile_nnz;
    h->stream_ok = h->max_tile_nnz <= kTileCap;
    const double mean = (double)nnz / (double)n;
    h->tpr = mean <= 3 ? 2 : mean <= 6 ? 4 : mean <= 40 ? 8 : mean <= 96 ? 16 : 32;
    int rc = setup_variant<1>(h);
    if (rc == CG_OK) rc = setup_variant<2>(h);
    if (rc != CG_OK) { cg_destroy(h); return rc; }
    *out = h;
    return CG_OK;
}

extern "C" int cg_destroy(cg_handle* h) {
    if (!h) return CG_OK;
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
    if (h->h_scal) cudaFreeHost(h->h_scal);
    if (h->h_params) cudaFreeHost(h->h_params);
    delete h;
    return CG_OK;
}

extern "C" const char* cg_strerror(int code) {
    switch (code) {
        case CG_OK: return "success / converged";
        case CG_MAXIT: return "maximum number of iterations reached";
        case CG_BREAKDOWN: return "breakdown: p.Ap <= 0 or not finite (matrix not SPD)";
        case CG_EINVAL: return "invalid argument";
        case CG_ECUDA: return g_cuda_err;
        case CG_EUNSUPPORTED: return "device not supported (needs compute capability 10.x with cooperative launch)";
        default: return "unknown code";
    }
}

extern "C" int cg_set_option(cg_handle* h, const char* name, int64_t value) {
    if (!h || !name) return CG_EINVAL;
    if (!strcmp(name, "loop")) { if (value < 0 || value > 2) return CG_EINVAL; h->loop = (int)value; return CG_OK; }
    if (!strcmp(name, "spmv")) { if (value < 0 || value > 2) return CG_EINVAL; h->spmv_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "chunk")) { if (value < 2 || value > 4096 || (value & 1)) return CG_EINVAL; h->chunk = (int)value; return CG_OK; }
    if (!strcmp(name, "tpr")) {
        if (value != 2 && value != 4 && value != 8 && value != 16 && value != 32) return CG_EINVAL;
        h->tpr = (int)value; return CG_OK;
    }
    if (!strcmp(name, "ctas_per_sm")) {
        if (value < 0 || value > 8) return CG_EINVAL;
        h->ctas_per_sm = (int)value;
        int rc = setup_variant<1>(h);
        if (rc == CG_OK) rc = setup_variant<2>(h);
        return rc;
    }
    return CG_EINVAL;
}

extern "C" int cg_get_info(cg_handle* h, const char* name, int64_t* value) {
    if (!h || !name || !value) return CG_EINVAL;
    const int v = pick_variant(h);
    if (!strcmp(name, "loop")) *value = h->loop;
    else if (!strcmp(name, "spmv")) *value = v;
    else if (!strcmp(name, "grid")) *value = h->grid_v[v];
    else if (!strcmp(name, "block")) *value = kThreads;
    else if (!strcmp(name, "smem")) *value = (int64_t)(v == 2 ? kStreamSmemBytes : 0);
    else if (!strcmp(name, "launches")) *value = h->launches;
    else if (!strcmp(name, "sms")) *value = h->sms;
    else if (!strcmp(name, "tpr")) *value = h->tpr;
    else if (!strcmp(name, "max_row_len")) *value = h->max_row_len;
    else if (!strcmp(name, "max_tile_nnz")) *value = h->max_tile_nnz;
    else if (!strcmp(name, "stream_ok")) *value = h->stream_ok ? 1 : 0;
    else return CG_EINVAL;
    return CG_OK;
}

extern "C" int cg_check_csr(cg_handle* h, void* cuda_stream) {
    if (!h) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    CK(cudaMemsetAsync(&h->scal->check, 0, sizeof(int), st));
    k_check_csr<<<h->sms * 4, 256, 0, st>>>(h->rowptr, h->colind, h->n, h->nnz, h->scal);
    CK(cudaGetLastError());
    h->launches = 1;
    CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return h->h_scal->check ? CG_EINVAL : CG_OK;
}

extern "C" int cg_spmv(cg_handle* h, const double* d_x, double* d_y, void* cuda_stream) {
    if (!h || !d_x || !d_y || d_x == d_y || !aligned16(d_x) || !aligned16(d_y)) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int v = pick_variant(h);
    Params P;
    fill_params(h, &P, nullptr, nullptr, 0.0, 0, nullptr, 0, v);
    if (v == 2) k_spmv<2><<<h->grid_v[2], kThreads, kStreamSmemBytes, st>>>(P, d_x, d_y);
    else        k_spmv<1><<<h->grid_v[1], kThreads, 0, st>>>(P, d_x, d_y);
    CK(cudaGetLastError());
    h->launches = 1;
    return CG_OK;
}

extern "C" int cg_dot(cg_handle* h, const double* d_a, const double* d_b, double* h_result,
                      void* cuda_stream) {
    if (!h || !d_a || !d_b || !h_result) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int G = h->sms * 2;
    k_dot_partial<<<G, kThreads, 0, st>>>(d_a, d_b, h->n, h->part0);
    CK(cudaGetLastError());
    k_dot_final<<<1, kThreads, 0, st>>>(h->part0, G, h->scal);
    CK(cudaGetLastError());
    h->launches = 2;
    CK(cudaMemcpyAsync(&h->h_scal->dot_out, &h->scal->dot_out, sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    *h_result = h->h_scal->dot_out;
    return CG_OK;
}

template <int V>
static int launch_iteration_kernels(cg_handle* h, cudaStream_t st, int iters) {
    const int G = h->grid_v[V];
    const size_t smem = variant_smem<V>();
    for (int it = 0; it < iters; ++it) {
        const int s = it & 1;
        k1_spmv_dot<V><<<G, kThreads, smem, st>>>(h->dparams, s);
        k2_update_xr<<<G, kThreads, 0, st>>>(h->dparams, s);
        k3_update_p<<<G, kThreads, 0, st>>>(h->dparams, s);
    }
    CK(cudaGetLastError());
    return CG_OK;
}

template <int V>
static int ensure_graph(cg_handle* h) {
    if (h->gexec && h->gexec_variant == V && h->gexec_chunk == h->chunk && h->gexec_grid == h->grid_v[V])
        return CG_OK;
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    cudaGraph_t g = nullptr;
    if (!h->cap_stream) CK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = launch_iteration_kernels<V>(h, h->cap_stream, h->chunk);
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
    if (rc != CG_OK) { if (g) cudaGraphDestroy(g); return rc; }
    CK(e);
    e = cudaGraphInstantiate(&h->gexec, g, 0);
    cudaGraphDestroy(g);
    CK(e);
    h->gexec_variant = V; h->gexec_chunk = h->chunk; h->gexec_grid = h->grid_v[V];
    return CG_OK;
}

template <int V>
static int solve_impl(cg_handle* h, const double* d_b, double* d_x, double rtol, long long maxit,
                      double* d_hist, int precond, int64_t* h_iters, double* h_res,
                      cudaStream_t st) {
    const int G = h->grid_v[V];
    const size_t smem = variant_smem<V>();
    h->launches = 0;
    if (precond && !h->dinv_ready) {
        Params P; fill_params(h, &P, d_b, d_x, rtol, maxit, d_hist, precond, V);
        CK(cudaMemsetAsync(&h->scal->diag_bad, 0, sizeof(int), st));
        k_diag_inv<<<h->sms * 4, 256, 0, st>>>(P);
        CK(cudaGetLastError());
        h->launches += 1;
        h->dinv_ready = true;
    }
    // zero the iteration state (everything before `check`), keep check / statistics
    CK(cudaMemsetAsync(h->scal, 0, offsetof(Scal, check), st));
    fill_params(h, h->h_params, d_b, d_x, rtol, maxit, d_hist, precond, V);

    if (h->loop == 0) {
        Params P = *h->h_params;
        void* args[] = {&P};
        CK(cudaLaunchCooperativeKernel((const void*)k_persistent<V>, dim3(G), dim3(kThreads), args, smem, st));
        h->launches += 1;
    } else {
        CK(cudaMemcpyAsync(h->dparams, h->h_params, sizeof(Params), cudaMemcpyHostToDevice, st));
        if (h->loop == 1) { int rc = ensure_graph<V>(h); if (rc != CG_OK) return rc; }
        k_init_spmv<V><<<G, kThreads, smem, st>>>(h->dparams);
        k_init_residual<<<G, kThreads, 0, st>>>(h->dparams);
        k_init_scalars<<<G, kThreads, 0, st>>>(h->dparams);
        CK(cudaGetLastError());
        h->launches += 3;
        while (true) {
            CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            if (h->h_scal->st[0].stop) break;
            if (h->loop == 1) { CK(cudaGraphLaunch(h->gexec, st)); }
            else { int rc = launch_iteration_kernels<V>(h, st, h->chunk); if (rc != CG_OK) return rc; }
            h->launches += 3LL * h->chunk;
        }
    }
    CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (h_iters) *h_iters = h->h_scal->out_iters;
    if (h_res) *h_res = h->h_scal->out_res;
    return (int)h->h_scal->out_status;
}

static int solve_checked(cg_handle* h, const double* d_b, double* d_x, double rtol, int64_t maxit,
                         double* d_hist, int precond, int64_t* h_iters, double* h_res, void* stream) {
    if (!h || !d_b || !d_x || d_b == d_x) return CG_EINVAL;
    if (!(rtol >= 0.0) || maxit < 0) return CG_EINVAL;          // also rejects NaN
    if (!aligned16(d_b) || !aligned16(d_x) || (reinterpret_cast<uintptr_t>(d_hist) & 7u)) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (pick_variant(h) == 2)
        return solve_impl<2>(h, d_b, d_x, rtol, maxit, d_hist, precond, h_iters, h_res, st);
    return solve_impl<1>(h, d_b, d_x, rtol, maxit, d_hist, precond, h_iters, h_res, st);
}

extern "C" int cg_solve(cg_handle* h, const double* d_b, double* d_x, double rtol, int64_t maxit,
                        double* d_hist, int64_t* h_iters, double* h_final_resnorm, void* cuda_stream) {
    return solve_checked(h, d_b, d_x, rtol, maxit, d_hist, 0, h_iters, h_final_resnorm, cuda_stream);
}

extern "C" int cg_solve_jacobi(cg_handle* h, const double* d_b, double* d_x, double rtol,
                               int64_t maxit, double* d_hist, int64_t* h_iters,
                               double* h_final_resnorm, void* cuda_stream) {
    return solve_checked(h, d_b, d_x, rtol, maxit, d_hist, 1, h_iters, h_final_resnorm, cuda_stream);
}

extern "C" int cg_solve_host(cg_handle* h, const double* h_b, double* h_x, double rtol, int64_t maxit,
                             double* h_hist, int64_t* h_iters, double* h_final_resnorm,
                             void* d_scratch, size_t scratch_bytes, void* cuda_stream) {
    if (!h || !h_b || !h_x || !d_scratch || maxit < 0) return CG_EINVAL;
    if ((reinterpret_cast<uintptr_t>(d_scratch) & 255u) || scratch_bytes < cg_host_scratch_bytes(h->n, maxit))
        return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* w = static_cast<unsigned char*>(d_scratch);
    double* d_b = (double*)w; w += vec_bytes(h->n);
    double* d_x = (double*)w; w += vec_bytes(h->n);
    double* d_hist = h_hist ? (double*)w : nullptr;
    const size_t nb = (size_t)h->n * 8u;
    CK(cudaMemcpyAsync(d_b, h_b, nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(d_x, h_x, nb, cudaMemcpyHostToDevice, st));
    int64_t iters = 0; double res = 0.0;
    const int rc = solve_checked(h, d_b, d_x, rtol, maxit, d_hist, 0, &iters, &res, cuda_stream);
    if (rc < 0) return rc;
    CK(cudaMemcpyAsync(h_x, d_x, nb, cudaMemcpyDeviceToHost, st));
    if (h_hist) CK(cudaMemcpyAsync(h_hist, d_hist, (size_t)(iters + 1) * 8u, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (h_iters) *h_iters = iters;
    if (h_final_resnorm) *h_final_resnorm = res;
    return rc;
}
