// cg_api.cu -- C ABI (include/cg.h) and kernel entry points of libcg_b200.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -shared -Xcompiler -fPIC
#include "../../include/cg.h"
#include "cg_kernels.cuh"
#include "cg_stream_kernels.cuh"

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

// ---- generic variant (spmv = 1): sub-warp per row straight from global memory; any CSR matrix.
__global__ void __launch_bounds__(kThreads, 2) k_spmv(Params P, const double* x, double* y) {
    phase_spmv_vector_dispatch<false>(P, x, y, blockIdx.x, gridDim.x);
}

// cg_probe_read_bandwidth: every thread streams 16-byte loads over the buffer.
__global__ void __launch_bounds__(512) k_probe_read(const uint4* __restrict__ buf, size_t n16, unsigned* sink) {
    unsigned acc = 0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        const uint4 a = __ldcg(buf + i), b = __ldcg(buf + i + stride);
        const uint4 c = __ldcg(buf + i + 2 * stride), d = __ldcg(buf + i + 3 * stride);
        acc += a.x ^ b.y ^ c.z ^ d.w;
    }
    for (; i < n16; i += stride) acc += __ldcg(buf + i).x;
    if (acc == 0x9e3779b9u) *sink = acc;              // never true for the buffers the bench passes: keeps the loads alive
}

// padded copy of rowptr for the streamed variants' 36-int bulk copies
__global__ void k_pad_rowptr(const int* __restrict__ rowptr, long long n, int* __restrict__ out, long long total) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride)
        out[i] = rowptr[i < n ? i : n];
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

__global__ void __launch_bounds__(kThreads, 2) k_init_spmv(const Params* __restrict__ dp) {
    const Params P = *dp;
    phase_spmv_vector_dispatch<false>(P, P.x, P.q, blockIdx.x, gridDim.x);
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

__global__ void __launch_bounds__(kThreads, 2) k1_spmv_dot(const Params* __restrict__ dp, int s) {
    __shared__ double sm[kWarps + 1];
    const Params P = *dp;
    if (P.scal->st[s].stop) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) P.scal->brk[s] = 0;
    const double d = phase_spmv_vector_dispatch<true>(P, P.p, P.q, blockIdx.x, gridDim.x);
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
__global__ void __launch_bounds__(kThreads, 2) k_persistent(Params P) {
    __shared__ double sm[kWarps + 1];
    const int cta = blockIdx.x, G = gridDim.x;
    const bool lead = cta == 0 && threadIdx.x == 0;
    Scal* S = P.scal;
    unsigned long long epoch = 0;

    // a0 prologue: q = A x0 ; r = b - q ; p = r ; rr, bb
    phase_spmv_vector_dispatch<false>(P, P.x, P.q, cta, G);
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

    // Optional trace (cg_set_trace): thread 0 of every CTA stamps clock64 at 8 points of each
    // of the first trace_iters iterations: 0 start, 1 K1 done, 2 past barrier 1, 3 K2 done,
    // 4 past barrier 2, 5 beta known, 6 K3 done, 7 past barrier 3.
    unsigned long long* tr = (P.trace && threadIdx.x == 0)
        ? P.trace + (size_t)cta * (P.trace_iters + 1) * kTraceSlots : nullptr;
#define CG_STAMP(slot) do { if (tr && k < P.trace_iters) tr[k * kTraceSlots + (slot)] = clock64(); } while (0)
    while (!stop) {
        CG_STAMP(0);
        // K1
        const double d = phase_spmv_vector_dispatch<true>(P, P.p, P.q, cta, G);
        const double t = block_sum(d, sm);
        if (threadIdx.x == 0) P.part0[cta] = t;
        CG_STAMP(1);
        grid_barrier(&S->bar, G, epoch);
        CG_STAMP(2);
        // scalar alpha (every CTA, same order, same value)
        const double pq = sum_partials(P.part0, G, sm);
        if (!(pq > 0.0) || !is_finite(pq)) { stop = 1; status = CG_BREAKDOWN; break; }
        const double alpha = rz / pq;
        // K2
        phase_update_xr<2>(P, alpha, cta, G, sm);
        CG_STAMP(3);
        grid_barrier(&S->bar, G, epoch);
        CG_STAMP(4);
        // scalar beta, continue-condition
        const double rr_new = sum_partials(P.part1, G, sm);
        const double rz_new = P.precond ? sum_partials(P.part2, G, sm) : rr_new;
        const double beta = rz_new / rz;
        CG_STAMP(5);
        rr = rr_new; rz = rz_new; k += 1;
        const double res = sqrt(rr);
        if (lead && P.hist) P.hist[k] = res;
        if (res <= thresh) { stop = 1; status = CG_OK; break; }
        if (k >= P.maxit) { stop = 1; status = CG_MAXIT; break; }
        k -= 1;
        // K3
        phase_update_p<2>(P, beta, cta, G);
        CG_STAMP(6);
        grid_barrier(&S->bar, G, epoch);
        CG_STAMP(7);
        k += 1;
    }
#undef CG_STAMP
    if (lead) { S->out_iters = k; S->out_status = status; S->out_res = sqrt(rr); }
}

}  // namespace

// ---------------------------------------------------------------- host side

#include <stdio.h>

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

// Streamed variants: W consumer warps, U entries in flight per lane (cg_stream.cuh).
// "spmv" option value = index + 2.
struct StreamFns {
    int W, NP, U;
    const void* spmv;
    const void* init_spmv; const void* init_residual; const void* init_scalars;
    const void* k1; const void* k2; const void* k3;
    const void* persistent[3][2];          // [R index: 0 -> global vectors, 1 -> R = 2, 2 -> R = 4][Jacobi]
};

template <int W, int NP, int U> static StreamFns make_stream_fns() {
    StreamFns f;
    f.W = W; f.NP = NP; f.U = U;
    f.spmv = (const void*)cgs::ks_spmv<W, NP, U>;
    f.init_spmv = (const void*)cgs::ks_init_spmv<W, NP, U>;
    f.init_residual = (const void*)cgs::ks_init_residual<W, NP>;
    f.init_scalars = (const void*)cgs::ks_init_scalars<W, NP>;
    f.k1 = (const void*)cgs::ks1_spmv_dot<W, NP, U>;
    f.k2 = (const void*)cgs::ks2_update_xr<W, NP>;
    f.k3 = (const void*)cgs::ks3_update_p<W, NP>;
    f.persistent[0][0] = (const void*)cgs::ks_persistent<W, NP, U, 0, false>;
    f.persistent[0][1] = (const void*)cgs::ks_persistent<W, NP, U, 0, true>;
    f.persistent[1][0] = (const void*)cgs::ks_persistent<W, NP, U, 2, false>;
    f.persistent[1][1] = (const void*)cgs::ks_persistent<W, NP, U, 2, true>;
    f.persistent[2][0] = (const void*)cgs::ks_persistent<W, NP, U, 4, false>;
    f.persistent[2][1] = (const void*)cgs::ks_persistent<W, NP, U, 4, true>;
    return f;
}
static constexpr int kNumStream = 4;
static const StreamFns& stream_fns(int idx) {
    static const StreamFns table[kNumStream] = {
        make_stream_fns<12, 4, 9>(), make_stream_fns<8, 4, 27>(), make_stream_fns<8, 4, 9>(),
        make_stream_fns<11, 5, 9>()};
    return table[idx];
}

struct cg_handle {
    long long n, nnz;
    const int* rowptr; const int* colind; const double* vals;
    unsigned char* ws; size_t ws_bytes;
    double *r, *p, *q, *dinv, *spare, *part0, *part1, *part2, *part3, *bslots;
    int* rp_pad;
    Scal* scal; Params* dparams;
    Scal* h_scal; Params* h_params;        // pinned host mirrors
    int sms, smem_optin;
    size_t l2_bytes;
    int loop, spmv_opt, chunk, ctas_per_sm, resident_opt, lookahead, max_slots, fold_opt, l2_hints, l2_prefetch, pin_opt;
    int max_row_len, max_tile_nnz, tpr;
    bool dinv_ready;
    int grid_generic;                      // cooperative grid of the generic variant
    int cap, slots, slot_bytes;            // ring geometry of the streamed variants
    bool stream_ok[kNumStream];
    cudaGraphExec_t gexec; int gexec_variant, gexec_chunk, gexec_grid;
    cudaStream_t cap_stream;               // capture-only stream (the legacy stream cannot capture)
    unsigned long long* trace; int trace_iters;
    long long launches;
    int last_resident;                     // R used by the last persistent solve (info)
};

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static size_t vec_bytes(long long n) { return align_up((size_t)n * 8u, 256); }
static size_t rp_pad_bytes(long long n) { return align_up((size_t)(n + 1 + cgs::kRpPad) * 4u, 256); }
static constexpr int kNumVecs = 5;
static constexpr size_t kPartBytes = (size_t)kMaxGrid * 8u;
static constexpr size_t kBslotBytes = (size_t)cgs::kInboxStride * cgs::kBarGrid * 8u;    // one inbox per CTA
static constexpr size_t kScalBytes = 512, kParamBytes = 512;

extern "C" size_t cg_workspace_bytes(int64_t n) {
    if (n <= 0) return 0;
    return kNumVecs * vec_bytes(n) + rp_pad_bytes(n) + 4 * kPartBytes + kBslotBytes + kScalBytes + kParamBytes;
}

extern "C" size_t cg_host_scratch_bytes(int64_t n, int64_t maxit) {
    if (n <= 0 || maxit < 0) return 0;
    return 2 * vec_bytes(n) + align_up((size_t)(maxit + 1) * 8u, 256);
}

static size_t stream_smem(const cg_handle* h) { return (size_t)h->slots * h->slot_bytes + cgs::kSmemTail; }

static int setup_generic(cg_handle* h) {
    int bps = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, k_persistent, kThreads, 0));
    if (bps < 1) { snprintf(g_cuda_err, sizeof(g_cuda_err), "persistent kernel does not fit an SM"); return CG_ECUDA; }
    int want = h->ctas_per_sm > 0 ? h->ctas_per_sm : 2;
    if (want > bps) want = bps;
    int g = h->sms * want;
    if (g > kMaxGrid) g = kMaxGrid;
    h->grid_generic = g;
    return CG_OK;
}

// Ring geometry from the matrix statistics; the streamed variants need a ring of at least
// 8 slots in the opt-in shared memory, in a number the variant's producer count divides.
static int setup_stream(cg_handle* h) {
    h->cap = (h->max_tile_nnz + 6 + 3) & ~3;
    if (h->cap < 4) h->cap = 4;
    h->slot_bytes = (int)align_up((size_t)h->cap * 12u + (size_t)cgs::kRpInts * 4u, 128);
    const long long budget = (long long)h->smem_optin - cgs::kSmemTail;
    long long S = budget / h->slot_bytes;
    if (S > cgs::kMaxSlots) S = cgs::kMaxSlots;
    if (S > h->max_slots) S = h->max_slots;
    // A slot must always be refilled by the same producer warp (tile j -> warp j mod NP, slot
    // j mod S): otherwise a warp could run two phases ahead of a slot's "empty" barrier, which
    // a parity wait cannot tell from zero phases ahead.  So NP must divide S: multiples of 20
    // serve both producer counts (4 and 5), shallower rings only the variants with 4.
    S -= S % (S >= cgs::kSlotQuantum ? cgs::kSlotQuantum : 4);
    h->slots = (int)S;
    for (int v = 0; v < kNumStream; ++v) {
        const StreamFns& f = stream_fns(v);
        h->stream_ok[v] = S >= 8 && S % f.NP == 0 && h->sms <= cgs::kBarGrid;   // slots are released early: S need not cover W
        if (!h->stream_ok[v]) continue;
        const int smem = h->smem_optin;      // the attribute is per function, not per handle: always the maximum
        const void* fns[] = {f.spmv, f.init_spmv, f.init_residual, f.init_scalars, f.k1, f.k2, f.k3,
                             f.persistent[0][0], f.persistent[0][1], f.persistent[1][0],
                             f.persistent[1][1], f.persistent[2][0], f.persistent[2][1]};
        for (const void* fn : fns)
            CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    }
    return CG_OK;
}

// 1 = generic; 2 + i = streamed variant i.  Auto: 12 consumer + 4 producer warps when the matrix
// streams from HBM (config 4) or is pinned in shared memory (configs 0, 1: the producers
// idle); 11 + 5 when it is re-streamed from the L2 every iteration (configs 2, 3: measured
// 13.40 -> 12.68 and 34.28 -> 34.13 us per iteration; 292 -> 295 at config 4, 16.4 -> 17.2 at
// config 1).
static int pick_variant(const cg_handle* h) {
    if (h->spmv_opt == 1) return 1;
    if (h->spmv_opt >= 2) return h->stream_ok[h->spmv_opt - 2] ? h->spmv_opt : 1;
    const long long tc_max = ((h->n + kTileRows - 1) / kTileRows + h->sms - 1) / h->sms;
    const bool from_hbm = (size_t)h->nnz * 12u > h->l2_bytes / 2;
    const bool pinned = h->pin_opt && !from_hbm && tc_max <= h->slots;
    if (!from_hbm && !pinned && h->stream_ok[3]) return 5;
    return h->stream_ok[0] ? 2 : 1;
}

static int variant_grid(const cg_handle* h, int v) { return v == 1 ? h->grid_generic : h->sms; }

static void fill_params(const cg_handle* h, Params* P, const double* b, double* x, double rtol,
                        long long maxit, double* hist, int precond, int variant) {
    P->n = h->n; P->nnz = h->nnz;
    P->rowptr = h->rowptr; P->colind = h->colind; P->vals = h->vals;
    P->b = b; P->x = x; P->r = h->r; P->p = h->p; P->q = h->q; P->dinv = h->dinv;
    P->part0 = h->part0; P->part1 = h->part1; P->part2 = h->part2; P->part3 = h->part3;
    P->scal = h->scal; P->hist = hist; P->rtol = rtol; P->maxit = maxit;
    P->precond = precond; P->spmv = variant; P->tpr = h->tpr;
    P->trace = h->trace; P->trace_iters = h->trace_iters;
    P->rp_pad = h->rp_pad; P->bslots = h->bslots;
    P->cap = h->cap; P->slots = h->slots; P->slot_bytes = h->slot_bytes;
    P->lookahead = h->lookahead;
    P->l2_prefetch = h->l2_prefetch;
    P->p2 = h->spare;
    // Folding K3 into the next K1 trades a grid synchronisation for a second gather per entry:
    // measured a gain only while K1 is short (<= 8 tiles per CTA), a loss when gathers are
    // irregular (config 3: 38 -> 60 us per iteration).  2 = auto.
    const long long tc_max = ((h->n + kTileRows - 1) / kTileRows + h->sms - 1) / h->sms;
    P->fold = h->fold_opt == 2 ? (tc_max <= 8 ? 1 : 0) : h->fold_opt;
    P->l2_stream = ((size_t)h->nnz * 12u > h->l2_bytes / 2) ? (h->l2_hints ? 3 : 1) : 0;
    // Pinned tiles (cg_stream.cuh): when every CTA's slice of the matrix fits the ring, it is
    // copied into shared memory once per solve and stays there.
    P->pinned = 0; P->stream_slots = h->slots;
    if (h->pin_opt && !P->l2_stream && variant >= 2) {
        if (tc_max <= h->slots) {
            P->pinned = (int)tc_max;
            P->stream_slots = (h->slots - (int)tc_max) / cgs::kSlotQuantum * cgs::kSlotQuantum;   // unused: nothing streams
        }
        // A partial split (pin S - 8 tiles, stream the rest through 8 slots) was measured on
        // config 2 and lost: K1 12.4 k against 10.2 k cycles, the streamed tiles queue up
        // behind too few slots.  The kernels support it; the host never asks for it.
    }
}

extern "C" int cg_create(cg_handle** out, int64_t n, int64_t nnz, const int32_t* d_rowptr,
                         const int32_t* d_colind, const double* d_vals, void* d_workspace,
                         size_t workspace_bytes) {
    if (!out) return CG_EINVAL;
    *out = nullptr;
    if (n <= 0 || nnz < 0 || n >= (1LL << 31) - 64 || nnz >= (1LL << 31) - 8) return CG_EINVAL;
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
    h->rp_pad = (int*)w; w += rp_pad_bytes(n);
    h->part0 = (double*)w; w += kPartBytes; h->part1 = (double*)w; w += kPartBytes;
    h->part2 = (double*)w; w += kPartBytes; h->part3 = (double*)w; w += kPartBytes;
    h->bslots = (double*)w; w += kBslotBytes;
    h->scal = (Scal*)w; w += kScalBytes; h->dparams = (Params*)w; w += kParamBytes;
    static_assert(sizeof(Scal) <= kScalBytes && sizeof(Params) <= kParamBytes, "workspace slots");
    h->sms = prop.multiProcessorCount;
    h->smem_optin = (int)prop.sharedMemPerBlockOptin;
    h->l2_bytes = (size_t)prop.l2CacheSize;
    h->loop = 0; h->spmv_opt = 0; h->chunk = 32; h->ctas_per_sm = 0; h->resident_opt = 1; h->lookahead = 1 << 30; h->max_slots = cgs::kMaxSlots; h->fold_opt = 2; h->l2_hints = 0; h->l2_prefetch = 0; h->pin_opt = 1;

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
    // matrix statistics and the padded rowptr copy (legacy default stream)
    CKH(cudaMemsetAsync(h->scal, 0, sizeof(Scal), 0));
    k_stats<<<h->sms * 4, 256, 0, 0>>>(h->rowptr, h->n, h->scal);
    CKH(cudaGetLastError());
    k_pad_rowptr<<<h->sms * 4, 256, 0, 0>>>(h->rowptr, h->n, h->rp_pad, h->n + 1 + cgs::kRpPad);
    CKH(cudaGetLastError());
    CKH(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, 0));
    CKH(cudaStreamSynchronize(0));
    h->max_row_len = h->h_scal->max_row_len;
    h->max_tile_nnz = h->h_scal->max_tile_nnz;
    const double mean = (double)nnz / (double)n;
    h->tpr = mean <= 3 ? 2 : mean <= 6 ? 4 : mean <= 40 ? 8 : mean <= 96 ? 16 : 32;
    int rc = setup_generic(h);
    if (rc == CG_OK) rc = setup_stream(h);
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
    if (!strcmp(name, "spmv")) { if (value < 0 || value > 1 + kNumStream) return CG_EINVAL; h->spmv_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "chunk")) { if (value < 2 || value > 4096 || (value & 1)) return CG_EINVAL; h->chunk = (int)value; return CG_OK; }
    if (!strcmp(name, "lookahead")) { if (value < 0 || value > (1 << 30)) return CG_EINVAL; h->lookahead = (int)value; return CG_OK; }
    if (!strcmp(name, "ring_slots")) {
        if (value < 8 || value > cgs::kMaxSlots) return CG_EINVAL;
        h->max_slots = (int)value;
        if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }      // captured with the old smem size
        return setup_stream(h);
    }
    if (!strcmp(name, "pin")) {
        if (value < 0 || value > 1) return CG_EINVAL;
        h->pin_opt = (int)value;
        if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }      // kernels read it from Params, but be safe
        return CG_OK;
    }
    if (!strcmp(name, "l2_prefetch")) { if (value < 0 || value > 32) return CG_EINVAL; h->l2_prefetch = (int)value; return CG_OK; }
    if (!strcmp(name, "l2_hints")) { if (value < 0 || value > 1) return CG_EINVAL; h->l2_hints = (int)value; return CG_OK; }
    if (!strcmp(name, "fold")) { if (value < 0 || value > 2) return CG_EINVAL; h->fold_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "resident")) { if (value < 0 || value > 1) return CG_EINVAL; h->resident_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "tpr")) {
        if (value != 2 && value != 4 && value != 8 && value != 16 && value != 32) return CG_EINVAL;
        h->tpr = (int)value; return CG_OK;
    }
    if (!strcmp(name, "ctas_per_sm")) {
        if (value < 0 || value > 8) return CG_EINVAL;
        h->ctas_per_sm = (int)value;
        return setup_generic(h);
    }
    return CG_EINVAL;
}

// Rows per consumer thread the persistent kernel would keep in registers (0: global vectors).
static int resident_rows(const cg_handle* h, int v) {
    if (v < 2 || !h->resident_opt) return 0;
    const long long ntiles = (h->n + kTileRows - 1) / kTileRows;
    const long long tc_max = (ntiles + h->sms - 1) / h->sms;
    const int W = stream_fns(v - 2).W;
    const long long need = (tc_max + W - 1) / W;
    return need <= 2 ? 2 : need <= 4 ? 4 : 0;        // 8 rows per thread spill and gain nothing (measured on config 1)
}

extern "C" int cg_get_info(cg_handle* h, const char* name, int64_t* value) {
    if (!h || !name || !value) return CG_EINVAL;
    const int v = pick_variant(h);
    if (!strcmp(name, "loop")) *value = h->loop;
    else if (!strcmp(name, "spmv")) *value = v;
    else if (!strcmp(name, "grid")) *value = variant_grid(h, v);
    else if (!strcmp(name, "block")) *value = v == 1 ? kThreads : 32 * (stream_fns(v - 2).W + stream_fns(v - 2).NP);
    else if (!strcmp(name, "smem")) *value = (int64_t)(v >= 2 ? stream_smem(h) : 0);
    else if (!strcmp(name, "launches")) *value = h->launches;
    else if (!strcmp(name, "sms")) *value = h->sms;
    else if (!strcmp(name, "tpr")) *value = h->tpr;
    else if (!strcmp(name, "max_row_len")) *value = h->max_row_len;
    else if (!strcmp(name, "max_tile_nnz")) *value = h->max_tile_nnz;
    else if (!strcmp(name, "stream_ok")) *value = h->stream_ok[0] ? 1 : 0;
    else if (!strcmp(name, "consumer_warps")) *value = v >= 2 ? stream_fns(v - 2).W : 0;
    else if (!strcmp(name, "producer_warps")) *value = v >= 2 ? stream_fns(v - 2).NP : 0;
    else if (!strcmp(name, "in_flight")) *value = v >= 2 ? stream_fns(v - 2).U : 4;
    else if (!strcmp(name, "ring_slots")) *value = v >= 2 ? h->slots : 0;
    else if (!strcmp(name, "slot_bytes")) *value = v >= 2 ? h->slot_bytes : 0;
    else if (!strcmp(name, "resident_rows")) *value = resident_rows(h, v);
    else return CG_EINVAL;
    return CG_OK;
}

extern "C" int cg_set_trace(cg_handle* h, uint64_t* d_trace, int64_t iters) {
    if (!h || iters < 0 || iters > (1 << 20) || (d_trace && (reinterpret_cast<uintptr_t>(d_trace) & 7u)))
        return CG_EINVAL;
    h->trace = (d_trace && iters > 0) ? reinterpret_cast<unsigned long long*>(d_trace) : nullptr;
    h->trace_iters = h->trace ? (int)iters : 0;
    return CG_OK;
}

extern "C" int cg_probe_read_bandwidth(cg_handle* h, const void* d_buf, size_t bytes, int reps,
                                       double* h_gbs, void* cuda_stream) {
    if (!h || !d_buf || !h_gbs || bytes < 4096 || reps < 1 || !aligned16(d_buf)) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    const size_t n16 = bytes / 16;
    unsigned* sink = reinterpret_cast<unsigned*>(&h->scal->dot_out);
    const uint4* buf = static_cast<const uint4*>(d_buf);
    k_probe_read<<<h->sms * 4, 512, 0, st>>>(buf, n16, sink);          // warm-up (and L2 fill)
    cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r) k_probe_read<<<h->sms * 4, 512, 0, st>>>(buf, n16, sink);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    CK(e);
    CK(cudaGetLastError());
    h->launches = reps + 1;
    *h_gbs = (double)(n16 * 16) * reps / ((double)ms * 1e-3) / 1e9;
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
    if (v == 1) {
        k_spmv<<<h->grid_generic, kThreads, 0, st>>>(P, d_x, d_y);
    } else {
        const StreamFns& f = stream_fns(v - 2);
        void* args[] = {&P, &d_x, &d_y};
        CK(cudaLaunchKernel(f.spmv, dim3(h->sms), dim3(32 * (f.W + f.NP)), args, stream_smem(h), st));
    }
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

// K1, K2, K3 of `iters` iterations as separate launches (captured into the graph of loop
// mode 1, issued directly in loop mode 2).
static int launch_iteration_kernels(cg_handle* h, int v, cudaStream_t st, int iters) {
    const int G = variant_grid(h, v);
    for (int it = 0; it < iters; ++it) {
        int s = it & 1;
        if (v == 1) {
            k1_spmv_dot<<<G, kThreads, 0, st>>>(h->dparams, s);
            k2_update_xr<<<G, kThreads, 0, st>>>(h->dparams, s);
            k3_update_p<<<G, kThreads, 0, st>>>(h->dparams, s);
        } else {
            const StreamFns& f = stream_fns(v - 2);
            const dim3 blk(32 * (f.W + f.NP));
            const size_t smem = stream_smem(h);
            void* args[] = {&h->dparams, &s};
            CK(cudaLaunchKernel(f.k1, dim3(G), blk, args, smem, st));
            CK(cudaLaunchKernel(f.k2, dim3(G), blk, args, smem, st));
            CK(cudaLaunchKernel(f.k3, dim3(G), blk, args, smem, st));
        }
    }
    CK(cudaGetLastError());
    return CG_OK;
}

static int ensure_graph(cg_handle* h, int v) {
    const int G = variant_grid(h, v);
    if (h->gexec && h->gexec_variant == v && h->gexec_chunk == h->chunk && h->gexec_grid == G)
        return CG_OK;
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    cudaGraph_t g = nullptr;
    if (!h->cap_stream) CK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = launch_iteration_kernels(h, v, h->cap_stream, h->chunk);
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
    if (rc != CG_OK) { if (g) cudaGraphDestroy(g); return rc; }
    CK(e);
    e = cudaGraphInstantiate(&h->gexec, g, 0);
    cudaGraphDestroy(g);
    CK(e);
    h->gexec_variant = v; h->gexec_chunk = h->chunk; h->gexec_grid = G;
    return CG_OK;
}

static int solve_impl(cg_handle* h, int v, const double* d_b, double* d_x, double rtol, long long maxit,
                      double* d_hist, int precond, int64_t* h_iters, double* h_res, cudaStream_t st) {
    const int G = variant_grid(h, v);
    h->launches = 0;
    if (precond && !h->dinv_ready) {
        Params P; fill_params(h, &P, d_b, d_x, rtol, maxit, d_hist, precond, v);
        CK(cudaMemsetAsync(&h->scal->diag_bad, 0, sizeof(int), st));
        k_diag_inv<<<h->sms * 4, 256, 0, st>>>(P);
        CK(cudaGetLastError());
        h->launches += 1;
        h->dinv_ready = true;
    }
    // zero the iteration state (everything before `check`), keep check / statistics
    CK(cudaMemsetAsync(h->scal, 0, offsetof(Scal, check), st));
    fill_params(h, h->h_params, d_b, d_x, rtol, maxit, d_hist, precond, v);

    if (h->loop == 0) {
        Params P = *h->h_params;
        void* args[] = {&P};
        if (v == 1) {
            CK(cudaLaunchCooperativeKernel((const void*)k_persistent, dim3(G), dim3(kThreads), args, 0, st));
        } else {
            const StreamFns& f = stream_fns(v - 2);
            const int R = resident_rows(h, v);
            const int ri = R == 2 ? 1 : R == 4 ? 2 : 0;
            h->last_resident = R;
            CK(cudaMemsetAsync(h->bslots, 0xFF, kBslotBytes, st));        // arm the all-reduce slots
            CK(cudaLaunchCooperativeKernel(f.persistent[ri][precond ? 1 : 0], dim3(G), dim3(32 * (f.W + f.NP)),
                                           args, stream_smem(h), st));
        }
        h->launches += 1;
    } else {
        CK(cudaMemcpyAsync(h->dparams, h->h_params, sizeof(Params), cudaMemcpyHostToDevice, st));
        if (h->loop == 1) { int rc = ensure_graph(h, v); if (rc != CG_OK) return rc; }
        if (v == 1) {
            k_init_spmv<<<G, kThreads, 0, st>>>(h->dparams);
            k_init_residual<<<G, kThreads, 0, st>>>(h->dparams);
            k_init_scalars<<<G, kThreads, 0, st>>>(h->dparams);
        } else {
            const StreamFns& f = stream_fns(v - 2);
            const dim3 blk(32 * (f.W + f.NP));
            const size_t smem = stream_smem(h);
            void* args[] = {&h->dparams};
            CK(cudaLaunchKernel(f.init_spmv, dim3(G), blk, args, smem, st));
            CK(cudaLaunchKernel(f.init_residual, dim3(G), blk, args, smem, st));
            CK(cudaLaunchKernel(f.init_scalars, dim3(G), blk, args, smem, st));
        }
        CK(cudaGetLastError());
        h->launches += 3;
        while (true) {
            CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            if (h->h_scal->st[0].stop) break;
            if (h->loop == 1) { CK(cudaGraphLaunch(h->gexec, st)); }
            else { int rc = launch_iteration_kernels(h, v, st, h->chunk); if (rc != CG_OK) return rc; }
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
    return solve_impl(h, pick_variant(h), d_b, d_x, rtol, maxit, d_hist, precond, h_iters, h_res,
                      static_cast<cudaStream_t>(stream));
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
