// cg_api.cu -- C ABI (include/cg.h) and kernel entry points of libcg_b200.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -shared -Xcompiler -fPIC
#include "../../include/cg.h"
#include "cg_kernels.cuh"
#include "cg_stream_kernels.cuh"
#include "cg_variants.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <limits.h>

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

// cg_create statistic: how many distinct 128-byte lines one warp-wide gather of the streamed
// SpMV touches on average (lane l gathers x[col] of entry t of row 32 tile + l).  ~2.5 for a
// stencil in natural ordering, ~30 for a random permutation: it decides how much of the SM's
// L1 / shared-memory array the ring may take (geometry()).
__global__ void k_gather_stats(const int* __restrict__ rp_pad, const int* __restrict__ colind, long long n,
                               unsigned long long* lines, unsigned long long* requests) {
    const int lane = threadIdx.x & 31;
    const long long ntiles = (n + kTileRows - 1) / kTileRows;
    const long long wstride = (long long)gridDim.x * (blockDim.x >> 5);
    unsigned long long nl = 0, nr = 0;
    for (long long t = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); t < ntiles; t += wstride) {
        const long long row = t * kTileRows + lane;
        const int rs = rp_pad[row], len = rp_pad[row + 1] - rs;
        int maxlen = len;
        for (int o = 16; o > 0; o >>= 1) maxlen = max(maxlen, __shfl_xor_sync(0xffffffffu, maxlen, o));
        for (int tt = 0; tt < maxlen; ++tt) {
            const bool in = tt < len;
            const int line = in ? (colind[rs + tt] >> 4) : -1 - lane;          // idle lanes: a private key each
            const unsigned same = __match_any_sync(0xffffffffu, line);
            const bool leader = in && (__ffs(same) - 1) == lane;
            nl += __popc(__ballot_sync(0xffffffffu, leader));
            nr += 1;
        }
    }
    if (lane == 0) { atomicAdd(lines, nl); atomicAdd(requests, nr); }
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

// ---- cg_compress_index: setup kernels of the compressed column index (cg_stream.cuh).
constexpr int kIdxHash = 1024;                       // open-addressing table of the distinct offsets col - row
constexpr long long kIdxEmpty = LLONG_MIN;
constexpr size_t kIdxTableOff = 0;                   // kMaxCodes ints: the sorted offsets
constexpr size_t kIdxHashOff = 1024;                 // kIdxHash long longs of scratch
constexpr size_t kIdxRecOff = 1024 + 8 * kIdxHash;   // records (a multiple of 128)

// Pass 1: the set of distinct offsets d = col - row, at most kMaxCodes of them (else overflow).
// Offset 0 is always a member (the records pad short rows with its code: a padding gather then
// reads x[row], a valid address).
__device__ __forceinline__ bool idx_insert(long long* table, Scal* scal, long long d) {
    unsigned slot = (unsigned)((unsigned long long)d * 0x9E3779B97F4A7C15ULL >> 54);      // top 10 bits
    for (int probes = 0; probes < kIdxHash; ++probes, slot = (slot + 1) & (kIdxHash - 1)) {
        long long cur = table[slot];                     // a stale "empty" is settled by the CAS
        if (cur == d) return true;
        if (cur == kIdxEmpty) {
            cur = (long long)atomicCAS(reinterpret_cast<unsigned long long*>(table + slot),
                                       (unsigned long long)kIdxEmpty, (unsigned long long)d);
            if (cur == kIdxEmpty) {
                if (atomicAdd(&scal->idx_count, 1) + 1 > cgs::kMaxCodes) scal->idx_overflow = 1;
                return true;
            }
            if (cur == d) return true;
        }
    }
    scal->idx_overflow = 1;
    return false;
}

__global__ void k_idx_collect(const int* __restrict__ rowptr, const int* __restrict__ colind, long long n,
                              long long* table, Scal* scal) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t0 == 0) idx_insert(table, scal, 0);
    for (long long i = t0; i < n; i += stride) {
        if (*reinterpret_cast<volatile int*>(&scal->idx_overflow)) return;
        long long last = kIdxEmpty;
        for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
            const long long d = (long long)colind[k] - i;
            if (d == last) continue;
            last = d;
            if (!idx_insert(table, scal, d)) return;
        }
    }
}

// Pass 2 (one CTA of kIdxHash threads): the offsets in ascending order -> codes 0 .. count - 1.
__global__ void k_idx_sort(const long long* __restrict__ table, int* __restrict__ off) {
    __shared__ long long keys[kIdxHash];
    const long long mine = table[threadIdx.x];
    keys[threadIdx.x] = mine;
    if (threadIdx.x < cgs::kMaxCodes) off[threadIdx.x] = 0;
    __syncthreads();
    if (mine == kIdxEmpty) return;
    int rank = 0;
    for (int j = 0; j < kIdxHash; ++j) rank += (keys[j] != kIdxEmpty && keys[j] < mine) ? 1 : 0;
    if (rank < cgs::kMaxCodes) off[rank] = (int)mine;
}

// Pass 3 (one warp per tile): the tile's record = 33 u16 row starts relative to the tile,
// [33] = parity of the tile's first entry (the vals span starts at an even entry), then the
// codes transposed and packed: the codes of entries 4 g .. 4 g + 3 of the tile's row l are the
// bytes (low to high) of the 32-bit word at byte 80 + 4 (32 g + l).
__global__ void k_idx_build(const int* __restrict__ rp_pad, const int* __restrict__ colind, long long n,
                            const int* __restrict__ off, int ncodes, unsigned char* __restrict__ rec, int rec_stride) {
    __shared__ int so[cgs::kMaxCodes];
    for (int i = threadIdx.x; i < cgs::kMaxCodes; i += blockDim.x) so[i] = off[i];
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const long long ntiles = (n + kTileRows - 1) / kTileRows;
    const long long wstride = (long long)gridDim.x * (blockDim.x >> 5);
    const int nwords = (rec_stride - cgs::kRecHdr) / 128;
    int pad = 0;                                       // the code of offset 0 (always in the table)
    { int lo = 0, hi = ncodes - 1; while (lo < hi) { const int mid = (lo + hi) >> 1; if (so[mid] < 0) lo = mid + 1; else hi = mid; } pad = lo; }
    for (long long t = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); t < ntiles; t += wstride) {
        const long long row = t * kTileRows + lane;
        const int s = rp_pad[t * kTileRows];
        const int rs = rp_pad[row], re = rp_pad[row + 1];
        unsigned char* r = rec + (size_t)t * (size_t)rec_stride;
        unsigned short* hd = reinterpret_cast<unsigned short*>(r);
        hd[lane] = (unsigned short)(rs - s);
        if (lane < 8) hd[32 + lane] = lane == 0 ? (unsigned short)(rp_pad[t * kTileRows + kTileRows] - s)
                                    : lane == 1 ? (unsigned short)(s & 1) : (unsigned short)0;
        unsigned* words = reinterpret_cast<unsigned*>(r + cgs::kRecHdr);
        for (int g = 0; g < nwords; ++g) {
            unsigned w = 0;
            for (int b = 0; b < 4; ++b) {
                const int tt = 4 * g + b;
                int code = pad;
                if (tt < re - rs) {
                    const int d = (int)((long long)colind[rs + tt] - row);
                    int lo = 0, hi = ncodes - 1;
                    while (lo < hi) { const int mid = (lo + hi) >> 1; if (so[mid] < d) lo = mid + 1; else hi = mid; }
                    code = lo;
                }
                w |= (unsigned)code << (8 * b);
            }
            words[g * 32 + lane] = w;
        }
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
    bool dead = grid_barrier(&S->bar, G, epoch, P.spin_budget, &S->abort);
    phase_init_residual(P, cta, G, sm);
    dead = grid_barrier(&S->bar, G, epoch, P.spin_budget, &S->abort) || dead;
    double rr = sum_partials(P.part1, G, sm);
    const double bb = sum_partials(P.part2, G, sm);
    double rz = P.precond ? sum_partials(P.part3, G, sm) : rr;
    if (bb == 0.0) { phase_zero_x(P, cta, G); rr = 0.0; }
    long long k; int stop, status; double thresh;
    init_decide(P, rr, bb, &k, &stop, &status, &thresh);
    if (P.precond && S->diag_bad) { stop = 1; status = CG_BREAKDOWN; }
    if (dead) { stop = 1; status = CG_ETIMEOUT; }
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
        if (grid_barrier(&S->bar, G, epoch, P.spin_budget, &S->abort)) { stop = 1; status = CG_ETIMEOUT; break; }
        CG_STAMP(2);
        // scalar alpha (every CTA, same order, same value)
        const double pq = sum_partials(P.part0, G, sm);
        if (!(pq > 0.0) || !is_finite(pq)) { stop = 1; status = CG_BREAKDOWN; break; }
        const double alpha = rz / pq;
        // K2
        phase_update_xr<2>(P, alpha, cta, G, sm);
        CG_STAMP(3);
        if (grid_barrier(&S->bar, G, epoch, P.spin_budget, &S->abort)) { stop = 1; status = CG_ETIMEOUT; break; }
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
        dead = grid_barrier(&S->bar, G, epoch, P.spin_budget, &S->abort);
        CG_STAMP(7);
        k += 1;
        if (dead) { stop = 1; status = CG_ETIMEOUT; break; }
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

// Streamed kernel shapes: their kernels are instantiated in cg_variant.cu, one translation unit per
// (shape, slot format) so that the build can compile them in parallel (cg_variants.h).
static constexpr int kNumStream = kNumShapes;
static const StreamFns& stream_fns(int idx) {
    static StreamFns table[kNumStream];
    static bool ready = false;
    if (!ready) {
        memset(table, 0, sizeof(table));
        cg_fill_fns_0_0(table[0]); cg_fill_fns_0_1(table[0]);
        cg_fill_fns_1_0(table[1]); cg_fill_fns_1_1(table[1]);
        cg_fill_fns_2_0(table[2]); cg_fill_fns_2_1(table[2]);
        cg_fill_fns_short(table[2]);
        ready = true;
    }
    return table[idx];
}

// Ring geometry and pinning of one launch configuration (a function of the handle's matrix
// statistics, its options and whether the compressed index is in use).
struct Geo {
    bool valid;                 // the streamed kernels can run this matrix
    int cmp;                    // slot format
    int cap, slot_bytes, rec_stride;
    int slots;                  // S = pinned + stream_slots (+ unused remainder)
    int pinned, stream_slots;   // P, Q
    bool from_hbm;              // the matrix stream exceeds half the L2
    size_t smem;
};

struct cg_handle {
    long long n, nnz;
    const int* rowptr; const int* colind; const double* vals;
    unsigned char* ws; size_t ws_bytes;
    double *r, *p, *q, *dinv, *spare, *part0, *part1, *part2, *part3, *bslots;
    unsigned char* bslots_base; int sync_place;
    int* rp_pad;
    Scal* scal; Params* dparams;
    Scal* h_scal; Params* h_params;        // pinned host mirrors
    int sms, smem_optin, clock_khz;
    size_t l2_bytes;
    int loop, spmv_opt, chunk, ctas_per_sm, resident_opt, lookahead, max_slots, fold_opt, pin_opt, compress_opt;
    int spin_budget_ms, inject_fault, algo_opt, checked_opt, short_opt;
    int max_row_len, max_tile_nnz, tpr;
    double lines_per_gather;               // cg_create statistic (k_gather_stats)
    int smem_cap_kb;                       // option: 0 = auto
    bool dinv_ready;
    int grid_generic;                      // cooperative grid of the generic variant
    unsigned char* idx; size_t idx_bytes; bool idx_ready; int idx_codes;     // compressed index (borrowed buffer)
    cudaGraphExec_t gexec; int gexec_variant, gexec_chunk, gexec_grid, gexec_cmp; size_t gexec_smem;
    cudaStream_t cap_stream;               // capture-only stream (the legacy stream cannot capture)
    unsigned long long* trace; int trace_iters, trace_clock;
    long long launches;
    int last_resident, last_fold, last_short;      // what the last persistent solve used (info)
    int last_chk_errors;                   // violations counted by the last checked cg_spmv
    // cg_reorder: the renumbered matrix P A P^T lives in a caller-owned buffer and has a handle of its own
    cg_handle* inner; int reorder_opt;
    const int* perm;                       // device: perm[new row] = old row
    double* rb; double* rx;                // device: b and x in the new numbering
};

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static bool reorder_active(const cg_handle* h) { return h->inner != nullptr && h->reorder_opt != 0; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static size_t vec_bytes(long long n) { return align_up((size_t)n * 8u, 256); }
static size_t rp_pad_bytes(long long n) { return align_up((size_t)(n + 1 + cgs::kRpPad) * 4u, 256); }
static constexpr int kNumVecs = 5;
static constexpr size_t kPartBytes = (size_t)kMaxGrid * 8u;
static constexpr size_t kBslotBytes = (size_t)cgs::kInboxStride * cgs::kBarGrid * 8u;    // one inbox per CTA
static constexpr size_t kScalBytes = 512, kParamBytes = 512;
// The all-reduce inboxes may sit anywhere in a reserve of 16 MB (option "sync_place", in steps of 64 KB): which
// L2 slices and which die their lines map to changes the cost of a grid all-reduce by ~4 % (measured), so
// cg_create tries a few places and keeps the fastest.
static constexpr size_t kBslotStep = 64u << 10, kBslotReserve = 16u << 20;
static constexpr int kBslotPlaces = (int)((kBslotReserve - kBslotBytes) / kBslotStep);

extern "C" size_t cg_workspace_bytes(int64_t n) {
    if (n <= 0) return 0;
    return kNumVecs * vec_bytes(n) + rp_pad_bytes(n) + 4 * kPartBytes + kBslotReserve + kScalBytes + kParamBytes;
}

extern "C" size_t cg_host_scratch_bytes(int64_t n, int64_t maxit) {
    if (n <= 0 || maxit < 0) return 0;
    return 2 * vec_bytes(n) + align_up((size_t)(maxit + 1) * 8u, 256);
}

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

static long long tiles_per_cta_max(const cg_handle* h) {
    return ((h->n + kTileRows - 1) / kTileRows + h->sms - 1) / h->sms;
}
static int rec_stride_of(const cg_handle* h) { return cgs::kRecHdr + 128 * ((h->max_row_len + 3) / 4); }
// the shared-memory copy of the offset table: 128 bytes when the matrix names <= 32 offsets, else 1 KB
static int offtab_entries(const cg_handle* h) { return h->idx_codes <= cgs::kOffTabSmall ? cgs::kOffTabSmall : cgs::kMaxCodes; }
static bool use_cmp(const cg_handle* h) { return h->idx_ready && h->compress_opt != 0; }

// Ring geometry of streamed variant `idx` from the matrix statistics.  A slot holds the largest
// tile: plain CSR cap * 12 + 144 bytes (cap = max tile nnz widened by the 16-byte alignment of
// the colind span), compressed cap * 8 + record bytes.  Pinning (option "pin": 1 = auto,
// 0 = never, k >= 2 = pin k tiles per CTA and stream the rest, for tests): when the matrix is
// re-read from the L2 every iteration anyway and every CTA's slice fits the shared memory, the
// ring is exactly the slice and nothing streams.  Otherwise the tiles stream through a ring
// whose depth Q is a multiple of the variant's producer count NP: a slot must always be
// refilled by the same producer warp (tile j -> warp j mod NP, slot j mod Q), otherwise a warp
// could run two phases ahead of a slot's "empty" barrier, which a parity wait cannot tell from
// zero phases ahead.  A variant without producer warps (NP = 0) needs everything pinned.
static Geo geometry(const cg_handle* h, bool cmp, int idx) {
    Geo g; memset(&g, 0, sizeof(g));
    const int NP = stream_fns(idx).NP;
    g.cmp = cmp ? 1 : 0;
    g.rec_stride = rec_stride_of(h);
    if (cmp) {
        g.cap = (h->max_tile_nnz + 2 + 1) & ~1;
        g.slot_bytes = (int)align_up((size_t)g.cap * 8u + (size_t)g.rec_stride, 16);
    } else {
        g.cap = (h->max_tile_nnz + 6 + 3) & ~3;
        if (g.cap < 4) g.cap = 4;
        g.slot_bytes = (int)align_up((size_t)g.cap * 12u + (size_t)cgs::kRpInts * 4u, 128);
    }
    const size_t fixed = (size_t)cgs::kSmemTail + (cmp ? (size_t)offtab_entries(h) * 4u : 0u);
    g.from_hbm = (size_t)h->nnz * (cmp ? 9u : 12u) > h->l2_bytes / 2;
    // How much of the SM's 256 KB L1 / shared-memory array a STREAMING ring may take.  What is
    // left is the L1, and an L1 line is what an outstanding gather miss occupies: with 227 KB of
    // ring the 28 KB of L1 allow ~220 lines in flight per SM, i.e. 7 warp-wide gathers when every
    // lane hits its own line.  Measured (us per iteration, ring depth): config 3 (permuted) 32.9
    // at 20 slots, 20.5 at 10-15; config 4 263 at 20 compressed slots (158 KB), 276 at 25, 295 at
    // 10; config 2 streamed 11.8 at 20 plain slots, 12.6 at 15.
    long long cap_bytes = h->smem_optin;
    if (h->smem_cap_kb > 0) cap_bytes = (long long)h->smem_cap_kb * 1024;
    else if (h->lines_per_gather > 8.0) cap_bytes = 132 * 1024;
    else if (g.from_hbm) cap_bytes = 164 * 1024;
    if (cap_bytes > h->smem_optin) cap_bytes = h->smem_optin;
    long long raw = ((long long)h->smem_optin - (long long)fixed) / g.slot_bytes;
    const long long raw_stream = (cap_bytes - (long long)fixed) / g.slot_bytes;
    if (raw > cgs::kMaxSlots) raw = cgs::kMaxSlots;
    if (raw > h->max_slots) raw = h->max_slots;
    const long long tc_max = tiles_per_cta_max(h);
    if (h->sms > cgs::kBarGrid || raw < 1) return g;
    if (h->pin_opt == 1 && !g.from_hbm && tc_max <= raw) {
        g.slots = (int)tc_max; g.pinned = (int)tc_max; g.stream_slots = 0; g.valid = true;
    } else if (NP > 0) {
        if (raw > raw_stream && raw_stream >= 8) raw = raw_stream;      // never below the 8 slots that make a matrix streamable
        long long P = h->pin_opt >= 2 ? (h->pin_opt < tc_max ? h->pin_opt : tc_max) : 0;
        if (P > raw - 8) P = raw - 8 > 0 ? raw - 8 : 0;
        long long Q = raw - P;
        Q -= Q % NP;
        g.pinned = (int)P; g.stream_slots = (int)Q; g.slots = (int)(P + Q);
        g.valid = Q >= 8;                   // slots are released early: the ring need not cover the consumer warps
    }
    g.smem = (size_t)g.slots * g.slot_bytes + fixed;
    return g;
}

// 1 = generic; 2 + i = streamed variant i.  Auto:
//   everything pinned in shared memory       16 consumer warps, no producers, 27 gathers in flight
//   re-streamed from the L2 every iteration  11 consumer + 5 producer warps (configs 2, 3 in round
//                                            1: 13.40 -> 12.68 and 34.28 -> 34.13 us per iteration)
//   streamed from HBM                        11 + 5 with the compressed index (two copies per tile,
//                                            config 4: 254 against 276 us per iteration), 12 + 4 with
//                                            plain CSR slots (292 against 295)
static int pick_variant(const cg_handle* h, Geo* out = nullptr) {
    const bool cmp = use_cmp(h);
    Geo g; memset(&g, 0, sizeof(g));
    int v = 1;
    if (h->spmv_opt >= 2) {
        g = geometry(h, cmp, h->spmv_opt - 2);
        v = g.valid ? h->spmv_opt : 1;
    } else if (h->spmv_opt == 0) {
        const Geo g2 = geometry(h, cmp, 2);
        if (g2.valid) { g = g2; v = 4; }
        else {
            const Geo g1 = geometry(h, cmp, 1), g0 = geometry(h, cmp, 0);
            const bool five = g1.valid && (!g1.from_hbm || cmp);
            if (five) { g = g1; v = 3; }
            else if (g0.valid) { g = g0; v = 2; }
            else if (g1.valid) { g = g1; v = 3; }
        }
    }
    if (v == 1) { g = geometry(h, cmp, 0); }
    if (out) *out = g;
    return v;
}

static int variant_grid(const cg_handle* h, int v) { return v == 1 ? h->grid_generic : h->sms; }

// Rows per consumer thread the persistent kernel would keep in registers (0: global vectors).
static int resident_rows(const cg_handle* h, int v) {
    if (v < 2 || !h->resident_opt) return 0;
    const int W = stream_fns(v - 2).W;
    const long long need = (tiles_per_cta_max(h) + W - 1) / W;
    return need <= 2 ? 2 : need <= 4 ? 4 : 0;        // 8 rows per thread spill and gain nothing (measured on config 1)
}

// Short-row kernels (option "short_rows": 0 off, 1 auto): shape 2 with the compressed index, every tile pinned,
// no row longer than 9 entries (the 7-point Laplacian), more than one tile per consumer warp, vectors in
// registers.  They keep several tiles' gathers in flight per warp (cg_stream.cuh: short_batch).
static bool short_rows_possible(const cg_handle* h, int v, const Geo& g) {
    if (!h->short_opt || v != 4 || !g.cmp || resident_rows(h, v) == 0) return false;
    if (stream_fns(2).short_persistent[0] == nullptr) return false;
    const int W = stream_fns(2).W;
    return h->max_row_len <= 9 && g.pinned >= tiles_per_cta_max(h) && tiles_per_cta_max(h) > W;
}

// Folding K3 into the next K1 trades a grid synchronisation for a 16-byte gather per entry
// instead of an 8-byte one.  Option "fold": 0 off, 1 on, 2 auto.
static bool fold_effective(const cg_handle* h, int v, int precond, const Geo& g) {
    if (precond || resident_rows(h, v) == 0) return false;
    if (h->fold_opt != 2) return h->fold_opt == 1;
    // auto: where the short-row kernels apply they win (config 1: 8.9 against 10.6 us per iteration folded)
    if (short_rows_possible(h, v, g)) return false;
    // auto: the 16-byte gathers must cost less than the synchronisation they save.  Since the counter
    // barrier polls with acquire loads that is only so for short rows on small systems.  Measured (us per
    // iteration, folded / not): 27-point 16^3 7.27 / 6.92, 24^3 7.32 / 6.90, 32^3 7.48 / 7.16, 40^3 8.26 / 7.72,
    // 51^3 (config 2) 11.0 / 9.5; 7-point 32^3 6.68 / 6.88, 48^3 7.88 / 7.66 (short-row kernel), 64^3 10.6 / 8.7.
    const double gathers = (double)tiles_per_cta_max(h) * (double)h->nnz / (double)h->n;
    return h->max_row_len <= 9 && gathers <= 500.0;
}

// Options "algo" = 1 (Chronopoulos-Gear) and 2 (pipelined CG) apply to the persistent streamed
// kernel with the vectors in registers and no preconditioner; everything else runs the textbook
// recurrence.
static int algo_effective(const cg_handle* h, int v, int precond) {
    if (h->algo_opt == 0 || h->loop != 0 || precond || resident_rows(h, v) == 0) return 0;
    if (h->algo_opt == 2 && stream_fns(v - 2).pipe[0][0] == nullptr) return 0;
    return h->algo_opt;
}

static void fill_params(const cg_handle* h, Params* P, const double* b, double* x, double rtol,
                        long long maxit, double* hist, int precond, int variant, const Geo& g) {
    memset(P, 0, sizeof(*P));
    P->n = h->n; P->nnz = h->nnz;
    P->rowptr = h->rowptr; P->colind = h->colind; P->vals = h->vals;
    P->b = b; P->x = x; P->r = h->r; P->p = h->p; P->q = h->q; P->dinv = h->dinv;
    P->part0 = h->part0; P->part1 = h->part1; P->part2 = h->part2; P->part3 = h->part3;
    P->scal = h->scal; P->hist = hist; P->rtol = rtol; P->maxit = maxit;
    P->precond = precond; P->spmv = variant; P->tpr = h->tpr;
    P->trace = h->trace; P->trace_iters = h->trace_iters; P->trace_clock = h->trace_clock;
    P->rp_pad = h->rp_pad; P->bslots = h->bslots;
    P->cap = g.cap; P->slots = g.slots; P->slot_bytes = g.slot_bytes;
    P->pinned = g.pinned; P->stream_slots = g.stream_slots;
    P->lookahead = h->lookahead;
    // the pair buffers of the folded loop reuse {r, p} and {q, spare}: with the vectors in
    // registers (the only case that folds) none of the four is used otherwise
    P->pr0 = reinterpret_cast<double2*>(h->r);
    P->pr1 = reinterpret_cast<double2*>(h->q);
    P->l2_stream = g.from_hbm ? 1 : 0;
    P->cmp = g.cmp; P->rec_stride = g.rec_stride; P->ncodes_smem = offtab_entries(h);
    P->idx_off = h->idx ? reinterpret_cast<const int*>(h->idx + kIdxTableOff) : nullptr;
    P->idx_rec = h->idx ? h->idx + kIdxRecOff : nullptr;
    P->spin_budget = (long long)h->spin_budget_ms * (long long)h->clock_khz;
    P->inject_fault = h->inject_fault;
}

// Where the all-reduce inboxes go is decided by measurement (see kBslotReserve): the mixed sequence of the
// textbook loop {all-reduce, all-reduce, counter barrier} is timed at kTunePlaces places, the fastest kept.
// ~30 ms of cg_create; results never depend on the place (the sums have one fixed order).
static constexpr int kTunePlaces = 40, kTuneReps = 400;
static int tune_sync_place(cg_handle* h) {
    if (h->sms > cgs::kBarGrid) return CG_OK;
    int best = 0; double best_c = 0.0;
    for (int k = 0; k < kTunePlaces && k <= kBslotPlaces; ++k) {
        h->bslots = reinterpret_cast<double*>(h->bslots_base + (size_t)k * kBslotStep);
        double c = 0.0;
        const int rc = cg_probe_grid_sync(h, 1, kTuneReps, &c, nullptr);
        // the placement is an optimisation: if the probe cannot run (no room for a cooperative launch right now, a
        // watchdog trip, ...) the inboxes stay at the start of the reserve and cg_create goes on
        if (rc != CG_OK) { cudaGetLastError(); h->bslots = reinterpret_cast<double*>(h->bslots_base); h->sync_place = 0; h->launches = 0; return CG_OK; }
        if (k == 0 || c < best_c) { best = k; best_c = c; }
    }
    h->sync_place = best;
    h->bslots = reinterpret_cast<double*>(h->bslots_base + (size_t)best * kBslotStep);
    h->launches = 0;
    return CG_OK;
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
    int coop = 0, khz = 0;
    CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    if (!coop) return CG_EUNSUPPORTED;
    CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));

    cg_handle* h = new (std::nothrow) cg_handle();
    if (!h) return CG_ENOMEM;
    memset(h, 0, sizeof(*h));
    h->n = n; h->nnz = nnz;
    h->rowptr = d_rowptr; h->colind = d_colind; h->vals = d_vals;
    h->ws = static_cast<unsigned char*>(d_workspace); h->ws_bytes = workspace_bytes;
    unsigned char* w = h->ws;
    const size_t vb = vec_bytes(n);
    // r | p and q | spare are adjacent on purpose: each pair of vectors doubles as one {p, r} pair buffer
    h->r = (double*)w; w += vb; h->p = (double*)w; w += vb; h->q = (double*)w; w += vb;
    h->spare = (double*)w; w += vb; h->dinv = (double*)w; w += vb;
    h->rp_pad = (int*)w; w += rp_pad_bytes(n);
    h->part0 = (double*)w; w += kPartBytes; h->part1 = (double*)w; w += kPartBytes;
    h->part2 = (double*)w; w += kPartBytes; h->part3 = (double*)w; w += kPartBytes;
    h->bslots_base = w; h->bslots = (double*)w; w += kBslotReserve;
    h->scal = (Scal*)w; w += kScalBytes; h->dparams = (Params*)w; w += kParamBytes;
    static_assert(sizeof(Scal) <= kScalBytes && sizeof(Params) <= kParamBytes, "workspace slots");
    h->sms = prop.multiProcessorCount;
    h->smem_optin = (int)prop.sharedMemPerBlockOptin;
    h->clock_khz = khz > 0 ? khz : 2000000;
    h->l2_bytes = (size_t)prop.l2CacheSize;
    h->loop = 0; h->spmv_opt = 0; h->chunk = 32; h->ctas_per_sm = 0; h->resident_opt = 1;
    h->lookahead = 1 << 30; h->max_slots = cgs::kMaxSlots; h->fold_opt = 2; h->pin_opt = 1; h->compress_opt = 1; h->short_opt = 1;
    h->spin_budget_ms = 2000; h->inject_fault = 0;

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
    if (nnz > 0) {
        unsigned long long* cnt = reinterpret_cast<unsigned long long*>(h->part0);     // scratch until the first solve
        CKH(cudaMemsetAsync(cnt, 0, 16, 0));
        k_gather_stats<<<h->sms * 8, 256, 0, 0>>>(h->rp_pad, h->colind, h->n, cnt, cnt + 1);
        CKH(cudaGetLastError());
        unsigned long long hc[2] = {0, 0};
        CKH(cudaMemcpy(hc, cnt, 16, cudaMemcpyDeviceToHost));
        h->lines_per_gather = hc[1] ? (double)hc[0] / (double)hc[1] : 0.0;
    }
    const double mean = (double)nnz / (double)n;
    h->tpr = mean <= 3 ? 2 : mean <= 6 ? 4 : mean <= 40 ? 8 : mean <= 96 ? 16 : 32;
    int rc = setup_generic(h);
    if (rc != CG_OK) { cg_destroy(h); return rc; }
    // the opt-in shared-memory size is a per-function attribute: always the maximum
    for (int v = 0; v < kNumStream; ++v) {
        const StreamFns& f = stream_fns(v);
        const void* one[] = {f.init_residual, f.init_scalars, f.k2, f.k3};
        for (const void* fn : one) CKH(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin));
        for (int c = 0; c < 2; ++c) {
            const void* two[] = {f.spmv[c], f.spmv_checked[c], f.init_spmv[c], f.k1[c]};
            for (const void* fn : two) CKH(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin));
            for (int k = 0; k < kNumPersistent; ++k)
                CKH(cudaFuncSetAttribute(f.persistent[c][k], cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin));
            for (int k = 0; k < 2; ++k) {
                CKH(cudaFuncSetAttribute(f.cg1[c][k], cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin));
                if (f.pipe[c][k]) CKH(cudaFuncSetAttribute(f.pipe[c][k], cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin));
            }
        }
        const void* shorts[] = {f.short_persistent[0], f.short_persistent[1], f.short_cg1, f.short_pipe};
        for (const void* fn : shorts)
            if (fn) CKH(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_optin));
    }
    rc = tune_sync_place(h);
    if (rc != CG_OK) { cg_destroy(h); return rc; }
    *out = h;
    return CG_OK;
}

extern "C" int cg_destroy(cg_handle* h) {
    if (!h) return CG_OK;
    if (h->inner) { cg_destroy(h->inner); h->inner = nullptr; }
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
        case CG_NOTCOMPRESSED: return "index not compressed: more than 256 distinct column offsets, or not worth it";
        case CG_NOTREORDERED: return "matrix left in the caller's numbering: renumbering would not make its gathers more local";
        case CG_EINVAL: return "invalid argument";
        case CG_ECUDA: return g_cuda_err;
        case CG_EUNSUPPORTED: return "device not supported (needs compute capability 10.x with cooperative launch)";
        case CG_ETIMEOUT: return "device watchdog: a spin wait inside the solve exceeded its budget; results are void";
        case CG_ENOMEM: return "out of host memory";
        case CG_ETOOBIG: return "cg_dot_static: n exceeds the 33 554 432 elements its fixed scratch array can serve";
        default: return "unknown code";
    }
}

// ---- compressed column index

// Bytes of the index buffer: offset table, hash scratch, one record per tile.  0 when the
// matrix is not worth compressing: the records are ELL inside a tile (32 x longest row), so
// a matrix with very uneven rows would make them larger than the 4 bytes per entry they replace.
extern "C" size_t cg_index_bytes(cg_handle* h) {
    if (!h || h->nnz == 0 || h->max_row_len == 0 || h->max_tile_nnz > 65535) return 0;
    const size_t ntiles = (size_t)((h->n + kTileRows - 1) / kTileRows);
    const size_t rec = ntiles * (size_t)rec_stride_of(h);
    if (rec > 2u * (size_t)h->nnz + (1u << 20)) return 0;
    return align_up(kIdxRecOff + rec, 256);
}

extern "C" int cg_compress_index(cg_handle* h, void* d_index, size_t index_bytes, void* cuda_stream) {
    if (!h) return CG_EINVAL;
    h->idx_ready = false; h->idx = nullptr; h->idx_bytes = 0; h->idx_codes = 0;
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    const size_t need = cg_index_bytes(h);
    if (need == 0) return CG_NOTCOMPRESSED;
    if (!d_index || (reinterpret_cast<uintptr_t>(d_index) & 255u) || index_bytes < need) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* idx = static_cast<unsigned char*>(d_index);
    long long* table = reinterpret_cast<long long*>(idx + kIdxHashOff);
    int* off = reinterpret_cast<int*>(idx + kIdxTableOff);
    CK(cudaMemsetAsync(&h->scal->idx_count, 0, 2 * sizeof(int), st));
    {   // LLONG_MIN in every hash slot
        static_assert(kIdxEmpty == LLONG_MIN, "empty key");
        long long* hinit = static_cast<long long*>(malloc(sizeof(long long) * kIdxHash));
        if (!hinit) return CG_ENOMEM;
        for (int i = 0; i < kIdxHash; ++i) hinit[i] = kIdxEmpty;
        cudaError_t e = cudaMemcpyAsync(table, hinit, sizeof(long long) * kIdxHash, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        free(hinit);
        CK(e);
    }
    k_idx_collect<<<h->sms * 8, 256, 0, st>>>(h->rowptr, h->colind, h->n, table, h->scal);
    CK(cudaGetLastError());
    k_idx_sort<<<1, kIdxHash, 0, st>>>(table, off);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    h->launches = 2;
    if (h->h_scal->idx_overflow || h->h_scal->idx_count > cgs::kMaxCodes || h->h_scal->idx_count < 1)
        return CG_NOTCOMPRESSED;
    const int ncodes = h->h_scal->idx_count;
    k_idx_build<<<h->sms * 8, 256, 0, st>>>(h->rp_pad, h->colind, h->n, off, ncodes, idx + kIdxRecOff, rec_stride_of(h));
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));
    h->launches = 3;
    h->idx = idx; h->idx_bytes = index_bytes; h->idx_codes = ncodes; h->idx_ready = true;
    return CG_OK;
}

// ---- cg_reorder: reverse Cuthill-McKee renumbering (cg_rcm.cpp) and the renumbered copy of the matrix

static size_t reorder_rowptr_bytes(long long n) { return align_up((size_t)(n + 1) * 4u, 256); }
static size_t reorder_index_bytes(long long m) { return align_up((size_t)(m > 0 ? m : 1) * 4u, 256); }
static size_t reorder_vals_bytes(long long nnz) { return align_up((size_t)(nnz > 0 ? nnz : 1) * 8u, 256); }

extern "C" size_t cg_reorder_bytes(int64_t n, int64_t nnz) {
    if (n <= 0 || nnz < 0) return 0;
    return reorder_index_bytes(n) + reorder_rowptr_bytes(n) + reorder_index_bytes(nnz) + reorder_vals_bytes(nnz)
         + 2 * vec_bytes(n) + cg_workspace_bytes(n);
}

// One warp per new row: the entries of old row perm[i] with their columns renamed and, for rows of up to 256
// entries, sorted by the new column (rank sort; equal columns keep their stored order).  The order inside a
// row is free in CSR, and it matters here: lane l of a warp gathers entry u of row l, so the u-th entries of
// 32 consecutive rows should be neighbours (measured on config 3 after the renumbering: 13 lines per warp-wide
// gather with the stored order, 4.3 sorted, 3.3 in the generator's natural ordering).
__global__ void k_permute_csr(const int* __restrict__ perm, const int* __restrict__ inv, const int* __restrict__ rowptr,
                              const int* __restrict__ colind, const double* __restrict__ vals, const int* __restrict__ new_rowptr,
                              int* new_colind, double* __restrict__ new_vals, long long n) {
    constexpr int K = 8;
    const int lane = threadIdx.x & 31;
    const long long warp = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long i = warp; i < n; i += nwarps) {
        const int o = perm[i];
        const int s = rowptr[o], len = rowptr[o + 1] - s, d = new_rowptr[i];
        for (int e = lane; e < len; e += 32) new_colind[d + e] = inv[colind[s + e]];
        if (len > 32 * K) {
            for (int e = lane; e < len; e += 32) new_vals[d + e] = vals[s + e];
            continue;
        }
        __syncwarp();
        int key[K], rank[K];
        double v[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const int e = lane + 32 * k;
            key[k] = 0; rank[k] = 0; v[k] = 0.0;
            if (e < len) {
                key[k] = new_colind[d + e];
                v[k] = vals[s + e];
                int r = 0;
                for (int f = 0; f < len; ++f) {
                    const int kf = new_colind[d + f];
                    r += (kf < key[k] || (kf == key[k] && f < e)) ? 1 : 0;
                }
                rank[k] = r;
            }
        }
        __syncwarp();
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (lane + 32 * k < len) { new_colind[d + rank[k]] = key[k]; new_vals[d + rank[k]] = v[k]; }
        }
        __syncwarp();
    }
}

extern "C" int cg_reorder(cg_handle* h, void* d_buf, size_t bytes, void* cuda_stream) {
    if (!h) return CG_EINVAL;
    if (h->inner) { cg_destroy(h->inner); h->inner = nullptr; }
    h->perm = nullptr; h->rb = nullptr; h->rx = nullptr;
    if (h->nnz == 0) return CG_NOTREORDERED;
    if (!d_buf || (reinterpret_cast<uintptr_t>(d_buf) & 255u) || bytes < cg_reorder_bytes(h->n, h->nnz)) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const long long n = h->n, nnz = h->nnz;
    unsigned char* w = static_cast<unsigned char*>(d_buf);
    int* d_perm = (int*)w; w += reorder_index_bytes(n);
    int* d_rp = (int*)w; w += reorder_rowptr_bytes(n);
    int* d_ci = (int*)w; w += reorder_index_bytes(nnz);
    double* d_va = (double*)w; w += reorder_vals_bytes(nnz);
    double* d_rb = (double*)w; w += vec_bytes(n);
    double* d_rx = (double*)w; w += vec_bytes(n);
    unsigned char* d_ws = w;
    int* d_inv = reinterpret_cast<int*>(d_rb);              // scratch until the first solve

    // the pattern goes to the host once; the numbering is set-up work, like the statistics of cg_create
    int* hrp = static_cast<int*>(malloc(sizeof(int) * (size_t)(n + 1)));
    int* hci = static_cast<int*>(malloc(sizeof(int) * (size_t)nnz));
    int* hperm = static_cast<int*>(malloc(sizeof(int) * (size_t)n));
    int* hinv = static_cast<int*>(malloc(sizeof(int) * (size_t)n));
    int* hnrp = static_cast<int*>(malloc(sizeof(int) * (size_t)(n + 1)));
    auto release = [&]() { free(hrp); free(hci); free(hperm); free(hinv); free(hnrp); };
    if (!hrp || !hci || !hperm || !hinv || !hnrp) { release(); return CG_ENOMEM; }
    cudaError_t e = cudaMemcpyAsync(hrp, h->rowptr, sizeof(int) * (size_t)(n + 1), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(hci, h->colind, sizeof(int) * (size_t)nnz, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { release(); CK(e); }
    int rc = (hrp[n] == nnz) ? cg_rcm_host(n, hrp, hci, hperm) : CG_EINVAL;
    if (rc != CG_OK) { release(); return rc; }
    hnrp[0] = 0;
    for (long long i = 0; i < n; ++i) {
        hinv[hperm[i]] = (int)i;
        hnrp[i + 1] = hnrp[i] + (hrp[hperm[i] + 1] - hrp[hperm[i]]);
    }
    e = cudaMemcpyAsync(d_perm, hperm, sizeof(int) * (size_t)n, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_inv, hinv, sizeof(int) * (size_t)n, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_rp, hnrp, sizeof(int) * (size_t)(n + 1), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        k_permute_csr<<<h->sms * 8, 256, 0, st>>>(d_perm, d_inv, h->rowptr, h->colind, h->vals, d_rp, d_ci, d_va, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    release();
    CK(e);
    cg_handle* in = nullptr;
    rc = cg_create(&in, n, nnz, d_rp, d_ci, d_va, d_ws, cg_workspace_bytes(n));
    if (rc != CG_OK) return rc;
    h->launches = 1;
    // worth it only when a warp-wide gather touches clearly fewer lines than before
    if (!(in->lines_per_gather < (2.0 / 3.0) * h->lines_per_gather)) { cg_destroy(in); return CG_NOTREORDERED; }
    // the inner handle solves with the options this one has now (later changes are forwarded)
    in->loop = h->loop; in->spmv_opt = h->spmv_opt; in->chunk = h->chunk; in->resident_opt = h->resident_opt;
    in->lookahead = h->lookahead; in->max_slots = h->max_slots; in->fold_opt = h->fold_opt; in->pin_opt = h->pin_opt;
    in->short_opt = h->short_opt; in->spin_budget_ms = h->spin_budget_ms; in->inject_fault = h->inject_fault;
    in->algo_opt = h->algo_opt; in->smem_cap_kb = h->smem_cap_kb; in->tpr = h->tpr; in->trace_clock = h->trace_clock;
    in->trace = h->trace; in->trace_iters = h->trace_iters;
    if (h->ctas_per_sm != in->ctas_per_sm) { in->ctas_per_sm = h->ctas_per_sm; rc = setup_generic(in); if (rc != CG_OK) { cg_destroy(in); return rc; } }
    h->inner = in; h->reorder_opt = 1; h->perm = d_perm; h->rb = d_rb; h->rx = d_rx;
    return CG_OK;
}

static int set_option_one(cg_handle* h, const char* name, int64_t value);

extern "C" int cg_set_option(cg_handle* h, const char* name, int64_t value) {
    if (!h || !name) return CG_EINVAL;
    if (!strcmp(name, "reorder")) { if (value < 0 || value > 1) return CG_EINVAL; h->reorder_opt = (int)value; return CG_OK; }
    const int rc = set_option_one(h, name, value);
    if (rc != CG_OK || !h->inner) return rc;
    // the renumbered copy holds the values as they were: rewritten values need a new cg_reorder
    if (!strcmp(name, "values_changed")) { cg_destroy(h->inner); h->inner = nullptr; return CG_OK; }
    if (!strcmp(name, "checked")) return CG_OK;           // cg_spmv runs on the caller's matrix only
    return set_option_one(h->inner, name, value);
}

static int set_option_one(cg_handle* h, const char* name, int64_t value) {
    auto drop_graph = [&]() { if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; } };
    if (!strcmp(name, "loop")) { if (value < 0 || value > 2) return CG_EINVAL; h->loop = (int)value; return CG_OK; }
    if (!strcmp(name, "spmv")) { if (value < 0 || value > 1 + kNumStream) return CG_EINVAL; h->spmv_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "chunk")) { if (value < 2 || value > 4096 || (value & 1)) return CG_EINVAL; h->chunk = (int)value; return CG_OK; }
    if (!strcmp(name, "lookahead")) { if (value < 0 || value > (1 << 30)) return CG_EINVAL; h->lookahead = (int)value; return CG_OK; }
    if (!strcmp(name, "ring_slots")) {
        if (value < 8 || value > cgs::kMaxSlots) return CG_EINVAL;
        h->max_slots = (int)value; drop_graph();
        return CG_OK;
    }
    if (!strcmp(name, "pin")) {
        if (value < 0 || value > cgs::kMaxSlots) return CG_EINVAL;
        h->pin_opt = (int)value; drop_graph();
        return CG_OK;
    }
    if (!strcmp(name, "checked")) { if (value < 0 || value > 1) return CG_EINVAL; h->checked_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "algo")) { if (value < 0 || value > 2) return CG_EINVAL; h->algo_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "smem_cap_kb")) { if (value < 0 || value > 227) return CG_EINVAL; h->smem_cap_kb = (int)value; drop_graph(); return CG_OK; }
    if (!strcmp(name, "compress")) { if (value < 0 || value > 1) return CG_EINVAL; h->compress_opt = (int)value; drop_graph(); return CG_OK; }
    if (!strcmp(name, "fold")) { if (value < 0 || value > 2) return CG_EINVAL; h->fold_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "trace_clock")) { if (value < 0 || value > 1) return CG_EINVAL; h->trace_clock = (int)value; return CG_OK; }
    if (!strcmp(name, "sync_place")) {
        if (value < 0 || value > kBslotPlaces) return CG_EINVAL;
        h->sync_place = (int)value; h->bslots = reinterpret_cast<double*>(h->bslots_base + (size_t)value * kBslotStep);
        return CG_OK;
    }
    if (!strcmp(name, "short_rows")) { if (value < 0 || value > 1) return CG_EINVAL; h->short_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "resident")) { if (value < 0 || value > 1) return CG_EINVAL; h->resident_opt = (int)value; return CG_OK; }
    if (!strcmp(name, "spin_budget_ms")) { if (value < 1 || value > 600000) return CG_EINVAL; h->spin_budget_ms = (int)value; return CG_OK; }
    if (!strcmp(name, "inject_fault")) { if (value < 0 || value > (1 << 30)) return CG_EINVAL; h->inject_fault = (int)value; return CG_OK; }
    if (!strcmp(name, "values_changed")) { h->dinv_ready = false; return CG_OK; }
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

extern "C" int cg_get_info(cg_handle* h, const char* name, int64_t* value) {
    if (!h || !name || !value) return CG_EINVAL;
    if (!strncmp(name, "solve_", 6)) return cg_get_info(reorder_active(h) ? h->inner : h, name + 6, value);
    if (!strcmp(name, "reordered")) { *value = reorder_active(h) ? 1 : 0; return CG_OK; }
    Geo g;
    const int v = pick_variant(h, &g);
    if (!strcmp(name, "loop")) *value = h->loop;
    else if (!strcmp(name, "spmv")) *value = v;
    else if (!strcmp(name, "grid")) *value = variant_grid(h, v);
    else if (!strcmp(name, "block")) *value = v == 1 ? kThreads : 32 * (stream_fns(v - 2).W + stream_fns(v - 2).NP);
    else if (!strcmp(name, "smem")) *value = (int64_t)(v >= 2 ? g.smem : 0);
    else if (!strcmp(name, "launches")) *value = h->launches;
    else if (!strcmp(name, "sms")) *value = h->sms;
    else if (!strcmp(name, "tpr")) *value = h->tpr;
    else if (!strcmp(name, "max_row_len")) *value = h->max_row_len;
    else if (!strcmp(name, "max_tile_nnz")) *value = h->max_tile_nnz;
    else if (!strcmp(name, "stream_ok")) *value = geometry(h, use_cmp(h), 0).valid ? 1 : 0;
    else if (!strcmp(name, "consumer_warps")) *value = v >= 2 ? stream_fns(v - 2).W : 0;
    else if (!strcmp(name, "producer_warps")) *value = v >= 2 ? stream_fns(v - 2).NP : 0;
    else if (!strcmp(name, "in_flight")) *value = v >= 2 ? stream_fns(v - 2).U : 4;
    else if (!strcmp(name, "ring_slots")) *value = v >= 2 ? g.slots : 0;
    else if (!strcmp(name, "pinned_tiles")) *value = v >= 2 ? g.pinned : 0;
    else if (!strcmp(name, "slot_bytes")) *value = v >= 2 ? g.slot_bytes : 0;
    else if (!strcmp(name, "resident_rows")) *value = resident_rows(h, v);
    else if (!strcmp(name, "fold")) *value = fold_effective(h, v, 0, g) ? 1 : 0;
    else if (!strcmp(name, "algo")) *value = algo_effective(h, v, 0);
    else if (!strcmp(name, "sync_place")) *value = h->sync_place;
    else if (!strcmp(name, "sync_places")) *value = kBslotPlaces;
    else if (!strcmp(name, "short_rows")) *value = (short_rows_possible(h, v, g) && !(fold_effective(h, v, 0, g) && algo_effective(h, v, 0) == 0)) ? 1 : 0;
    else if (!strcmp(name, "compressed")) *value = (v >= 2 && g.cmp) ? 1 : 0;
    else if (!strcmp(name, "index_codes")) *value = h->idx_ready ? h->idx_codes : 0;
    else if (!strcmp(name, "from_hbm")) *value = g.from_hbm ? 1 : 0;
    else if (!strcmp(name, "check_errors")) *value = h->last_chk_errors;
    else if (!strcmp(name, "lines_per_gather_x100")) *value = (int64_t)(h->lines_per_gather * 100.0 + 0.5);
    else return CG_EINVAL;
    return CG_OK;
}

extern "C" int cg_set_trace(cg_handle* h, uint64_t* d_trace, int64_t iters) {
    if (!h || iters < 0 || iters > (1 << 20) || (d_trace && (reinterpret_cast<uintptr_t>(d_trace) & 7u)))
        return CG_EINVAL;
    h->trace = (d_trace && iters > 0) ? reinterpret_cast<unsigned long long*>(d_trace) : nullptr;
    h->trace_iters = h->trace ? (int)iters : 0;
    if (h->inner) { h->inner->trace = h->trace; h->inner->trace_iters = h->trace_iters; }
    return CG_OK;
}

extern "C" int cg_probe_read_bandwidth(cg_handle* h, const void* d_buf, size_t bytes, int reps,
                                       double* h_gbs, void* cuda_stream) {
    if (!h || !d_buf || !h_gbs || bytes < 4096 || reps < 1 || !aligned16(d_buf)) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    cudaError_t e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); CK(e); }
    const size_t n16 = bytes / 16;
    unsigned* sink = reinterpret_cast<unsigned*>(&h->scal->dot_out);
    const uint4* buf = static_cast<const uint4*>(d_buf);
    k_probe_read<<<h->sms * 4, 512, 0, st>>>(buf, n16, sink);          // warm-up (and L2 fill)
    e = cudaEventRecord(e0, st);
    for (int r = 0; r < reps; ++r) k_probe_read<<<h->sms * 4, 512, 0, st>>>(buf, n16, sink);
    if (e == cudaSuccess) e = cudaEventRecord(e1, st);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    CK(e);
    CK(cudaGetLastError());
    h->launches = reps + 1;
    *h_gbs = (double)(n16 * 16) * reps / ((double)ms * 1e-3) / 1e9;
    return CG_OK;
}

extern "C" int cg_probe_grid_sync(cg_handle* h, int kind, int reps, double* h_cycles, void* cuda_stream) {
    if (!h || !h_cycles || kind < 0 || kind > 2 || reps < 1 || reps > (1 << 20) || h->sms > cgs::kBarGrid) return CG_EINVAL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    constexpr int W = 16;
    const void* fn = (const void*)cgs::ks_probe_sync<W>;
    Geo g; memset(&g, 0, sizeof(g));
    g.slots = 1; g.slot_bytes = 128;
    Params P;
    fill_params(h, &P, nullptr, nullptr, 0.0, 0, nullptr, 0, 4, g);
    unsigned long long* out = reinterpret_cast<unsigned long long*>(h->part1);       // kMaxGrid slots of scratch
    CK(cudaMemsetAsync(&h->scal->bar, 0, sizeof(unsigned long long) + 2 * sizeof(int), st));     // bar, abort
    CK(cudaMemsetAsync(h->bslots, 0xFF, kBslotBytes, st));
    void* args[] = {&P, &kind, &reps, &out};
    const size_t smem = (size_t)g.slots * g.slot_bytes + cgs::kSmemTail;
    CK(cudaLaunchCooperativeKernel(fn, dim3(h->sms), dim3(32 * W), args, smem, st));
    unsigned long long* host = static_cast<unsigned long long*>(malloc(sizeof(unsigned long long) * (size_t)h->sms));
    if (!host) return CG_ENOMEM;
    cudaError_t e = cudaMemcpyAsync(host, out, sizeof(unsigned long long) * (size_t)h->sms, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    double sum = 0.0; bool dead = false;
    for (int i = 0; i < h->sms; ++i) { sum += (double)host[i]; dead = dead || host[i] == 0; }
    free(host);
    CK(e);
    h->launches = 1;
    if (dead) return CG_ETIMEOUT;
    // in kind 1 every third synchronisation is the counter barrier the recycling rule asks for
    *h_cycles = sum / h->sms / reps;
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
    Geo g;
    const int v = pick_variant(h, &g);
    Params P;
    fill_params(h, &P, nullptr, nullptr, 0.0, 0, nullptr, 0, v, g);
    if (v == 1) {
        k_spmv<<<h->grid_generic, kThreads, 0, st>>>(P, d_x, d_y);
    } else {
        const StreamFns& f = stream_fns(v - 2);
        void* args[] = {&P, &d_x, &d_y};
        if (h->checked_opt) {
            // the library's own memcheck: every index validated and clamped on the device, violations
            // counted; this call synchronises and reports them
            CK(cudaMemsetAsync(&h->scal->chk_errors, 0, sizeof(int), st));
            CK(cudaLaunchKernel(f.spmv_checked[g.cmp], dim3(h->sms), dim3(32 * (f.W + f.NP)), args, g.smem, st));
            CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            h->launches = 1;
            h->last_chk_errors = h->h_scal->chk_errors;
            if (h->h_scal->chk_errors) {
                snprintf(g_cuda_err, sizeof(g_cuda_err), "checked cg_spmv: %d out-of-range indices caught and clamped (corrupt CSR arrays?)",
                         h->h_scal->chk_errors);
                return CG_ECUDA;
            }
            return CG_OK;
        }
        CK(cudaLaunchKernel(f.spmv[g.cmp], dim3(h->sms), dim3(32 * (f.W + f.NP)), args, g.smem, st));
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
static int launch_iteration_kernels(cg_handle* h, int v, const Geo& g, cudaStream_t st, int iters) {
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
            void* args[] = {&h->dparams, &s};
            CK(cudaLaunchKernel(f.k1[g.cmp], dim3(G), blk, args, g.smem, st));
            CK(cudaLaunchKernel(f.k2, dim3(G), blk, args, g.smem, st));
            CK(cudaLaunchKernel(f.k3, dim3(G), blk, args, g.smem, st));
        }
    }
    CK(cudaGetLastError());
    return CG_OK;
}

static int ensure_graph(cg_handle* h, int v, const Geo& g) {
    const int G = variant_grid(h, v);
    if (h->gexec && h->gexec_variant == v && h->gexec_chunk == h->chunk && h->gexec_grid == G &&
        h->gexec_cmp == g.cmp && h->gexec_smem == g.smem)
        return CG_OK;
    if (h->gexec) { cudaGraphExecDestroy(h->gexec); h->gexec = nullptr; }
    cudaGraph_t gr = nullptr;
    if (!h->cap_stream) CK(cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking));
    CK(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = launch_iteration_kernels(h, v, g, h->cap_stream, h->chunk);
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &gr);
    if (rc != CG_OK) { if (gr) cudaGraphDestroy(gr); return rc; }
    CK(e);
    e = cudaGraphInstantiate(&h->gexec, gr, 0);
    cudaGraphDestroy(gr);
    CK(e);
    h->gexec_variant = v; h->gexec_chunk = h->chunk; h->gexec_grid = G; h->gexec_cmp = g.cmp; h->gexec_smem = g.smem;
    return CG_OK;
}

static int solve_core(cg_handle* h, const double* d_b, double* d_x, double rtol, long long maxit,
                      double* d_hist, int precond, int64_t* h_iters, double* h_res, cudaStream_t st) {
    Geo g;
    const int v = pick_variant(h, &g);
    const int G = variant_grid(h, v);
    h->launches = 0;
    if (precond && !h->dinv_ready) {
        Params P; fill_params(h, &P, d_b, d_x, rtol, maxit, d_hist, precond, v, g);
        CK(cudaMemsetAsync(&h->scal->diag_bad, 0, sizeof(int), st));
        k_diag_inv<<<h->sms * 4, 256, 0, st>>>(P);
        CK(cudaGetLastError());
        h->launches += 1;
        h->dinv_ready = true;
    }
    // zero the iteration state (everything before `check`), keep check / statistics
    CK(cudaMemsetAsync(h->scal, 0, offsetof(Scal, check), st));
    fill_params(h, h->h_params, d_b, d_x, rtol, maxit, d_hist, precond, v, g);

    if (h->loop == 0) {
        Params P = *h->h_params;
        void* args[] = {&P};
        if (v == 1) {
            CK(cudaLaunchCooperativeKernel((const void*)k_persistent, dim3(G), dim3(kThreads), args, 0, st));
        } else {
            const StreamFns& f = stream_fns(v - 2);
            const int R = resident_rows(h, v);
            const bool fold = fold_effective(h, v, precond, g);
            const int kind = R == 0 ? (precond ? kR0Jacobi : kR0)
                           : R == 2 ? (precond ? kR2Jacobi : fold ? kR2Fold : kR2)
                                    : (precond ? kR4Jacobi : fold ? kR4Fold : kR4);
            h->last_resident = R; h->last_fold = fold ? 1 : 0;
            const int algo = algo_effective(h, v, precond);
            const void* fn = algo == 1 ? f.cg1[g.cmp][R == 4 ? 1 : 0] : algo == 2 ? f.pipe[g.cmp][R == 4 ? 1 : 0]
                                       : f.persistent[g.cmp][kind];
            // short rows, every tile pinned, vectors in registers: the kernels that keep several tiles' gathers in flight
            h->last_short = 0;
            if (short_rows_possible(h, v, g) && !(fold && algo == 0)) {
                fn = algo == 1 ? f.short_cg1 : algo == 2 ? f.short_pipe : f.short_persistent[precond ? 1 : 0];
                h->last_short = 1; h->last_resident = 4;
            }
            CK(cudaMemsetAsync(h->bslots, 0xFF, kBslotBytes, st));        // arm the all-reduce slots
            CK(cudaLaunchCooperativeKernel(fn, dim3(G), dim3(32 * (f.W + f.NP)), args, g.smem, st));
        }
        h->launches += 1;
    } else {
        CK(cudaMemcpyAsync(h->dparams, h->h_params, sizeof(Params), cudaMemcpyHostToDevice, st));
        if (h->loop == 1) { int rc = ensure_graph(h, v, g); if (rc != CG_OK) return rc; }
        if (v == 1) {
            k_init_spmv<<<G, kThreads, 0, st>>>(h->dparams);
            k_init_residual<<<G, kThreads, 0, st>>>(h->dparams);
            k_init_scalars<<<G, kThreads, 0, st>>>(h->dparams);
        } else {
            const StreamFns& f = stream_fns(v - 2);
            const dim3 blk(32 * (f.W + f.NP));
            void* args[] = {&h->dparams};
            CK(cudaLaunchKernel(f.init_spmv[g.cmp], dim3(G), blk, args, g.smem, st));
            CK(cudaLaunchKernel(f.init_residual, dim3(G), blk, args, g.smem, st));
            CK(cudaLaunchKernel(f.init_scalars, dim3(G), blk, args, g.smem, st));
        }
        CK(cudaGetLastError());
        h->launches += 3;
        while (true) {
            CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
            CK(cudaStreamSynchronize(st));
            if (h->h_scal->st[0].stop || h->h_scal->abort) break;
            if (h->loop == 1) { CK(cudaGraphLaunch(h->gexec, st)); }
            else { int rc = launch_iteration_kernels(h, v, g, st, h->chunk); if (rc != CG_OK) return rc; }
            h->launches += 3LL * h->chunk;
        }
    }
    CK(cudaMemcpyAsync(h->h_scal, h->scal, sizeof(Scal), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (h_iters) *h_iters = h->h_scal->out_iters;
    if (h_res) *h_res = h->h_scal->out_res;
    if (h->h_scal->abort || h->h_scal->out_status == CG_ETIMEOUT) return CG_ETIMEOUT;
    return (int)h->h_scal->out_status;
}

// b and x0 into the renumbered system, and x back (cg_reorder): new[i] = old[perm[i]].
__global__ void k_gather_bx(const int* __restrict__ perm, const double* __restrict__ b, const double* __restrict__ x,
                            double* __restrict__ rb, double* __restrict__ rx, long long n) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int o = perm[i];
        rb[i] = b[o]; rx[i] = x[o];
    }
}
__global__ void k_scatter_x(const int* __restrict__ perm, const double* __restrict__ rx, double* __restrict__ x, long long n) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        x[perm[i]] = rx[i];
}

static int solve_impl(cg_handle* h, const double* d_b, double* d_x, double rtol, long long maxit,
                      double* d_hist, int precond, int64_t* h_iters, double* h_res, cudaStream_t st) {
    if (!reorder_active(h)) return solve_core(h, d_b, d_x, rtol, maxit, d_hist, precond, h_iters, h_res, st);
    k_gather_bx<<<h->sms * 4, 256, 0, st>>>(h->perm, d_b, d_x, h->rb, h->rx, h->n);
    CK(cudaGetLastError());
    const int rc = solve_core(h->inner, h->rb, h->rx, rtol, maxit, d_hist, precond, h_iters, h_res, st);
    h->launches = h->inner->launches + 1;
    if (rc < 0) return rc;
    k_scatter_x<<<h->sms * 4, 256, 0, st>>>(h->perm, h->rx, d_x, h->n);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));
    h->launches += 1;
    return rc;
}

static int solve_checked(cg_handle* h, const double* d_b, double* d_x, double rtol, int64_t maxit,
                         double* d_hist, int precond, int64_t* h_iters, double* h_res, void* stream) {
    if (!h || !d_b || !d_x || d_b == d_x) return CG_EINVAL;
    if (!(rtol >= 0.0) || maxit < 0) return CG_EINVAL;          // also rejects NaN
    if (!aligned16(d_b) || !aligned16(d_x) || (reinterpret_cast<uintptr_t>(d_hist) & 7u)) return CG_EINVAL;
    return solve_impl(h, d_b, d_x, rtol, maxit, d_hist, precond, h_iters, h_res,
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
