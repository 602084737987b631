// cg_kernels.cuh -- shared device code of the fp64 CSR conjugate-gradient hot path for sm_100a:
// the parameter / state structs, load-store and mbarrier / bulk-copy primitives, and the
// GENERIC variant ("spmv" = 1): sub-warp per row straight from global memory, grid-stride
// vector phases, a counter grid barrier.  The default, streamed variant lives in
// cg_stream.cuh / cg_stream_kernels.cuh.
//
// Steps (the paper names only the first, PAPER.md:44
// "Tasks, such as DGEMV(sparse), are repetitive"; the rest is the textbook CG of
// its ref [5]):
//   K1  q = A p fused with the p.q partial sums           (phase_spmv_*)
//   K2  x += alpha p ; r -= alpha q ; partial sums of r.r (phase_update_xr)
//   K3  p = r + beta p                                    (phase_update_p)
// alpha, beta and the continue-condition are evaluated on the
// device, redundantly and identically by every CTA, from per-CTA partials summed
// in a fixed order -- the paper's CPU-side scalar step and its transfers
// do not exist here.
//
// Within a variant the same phase functions are used by the persistent cooperative kernel
// and by the three stand-alone kernels of the graph / stepwise loop, so all loop modes give
// bitwise identical results.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cgk {

constexpr int kThreads = 256;       // threads per CTA, every kernel
constexpr int kWarps = kThreads / 32;
constexpr int kMaxGrid = 2048;
constexpr int kTileRows = 32;       // rows per tile of the streamed SpMV (one lane per row)

struct State {            // one per iteration parity (loop modes 1, 2)
    double rr;            // ||r_k||^2
    double rz;            // r_k . z_k (== rr without preconditioner)
    long long k;          // iterations done
    int stop;             // 0 run, 1 stop
    int status;           // CG_OK / CG_MAXIT / CG_BREAKDOWN once stopped
};

struct Scal {             // device-resident scalar state, zeroed before each solve
    State st[2];
    double bb;            // ||b||^2
    double thresh;        // rtol * ||b||
    int brk[2];           // breakdown seen by K2 of this parity
    unsigned long long bar;       // grid barrier arrival counter
    int abort;            // a device-side spin ran out of its budget (watchdog): the results are void
    int chk_errors;       // option "checked": index violations caught (and clamped) by a checked cg_spmv
    long long out_iters;  // result block, copied to the host at the end
    long long out_status;
    double out_res;
    double dot_out;       // cg_dot result
    int check;            // cg_check_csr error bits            (not zeroed per solve from here on)
    int diag_bad;         // Jacobi: a diagonal entry is missing or not positive
    int max_row_len;      // cg_create statistics
    int max_tile_nnz;
    int idx_count;        // cg_compress_index: distinct column offsets found
    int idx_overflow;     //                    more than kMaxCodes of them (or the hash table filled up)
};

struct Params {
    long long n, nnz;
    const int* rowptr;
    const int* colind;
    const double* vals;
    const double* b;
    double* x;
    double* r;
    double* p;
    double* q;
    double* dinv;
    double* part0;        // p.q
    double* part1;        // r.r
    double* part2;        // r.z (Jacobi) ; b.b in the prologue
    double* part3;        // r0.z0 in the prologue (Jacobi)
    Scal* scal;
    double* hist;         // may be null
    double rtol;
    long long maxit;
    int precond;          // 0 none (the paper's path), 1 Jacobi
    int spmv;             // 1 sub-warp per row from global, >= 2 streamed (cg_stream.cuh)
    int tpr;              // lanes per row of the vector variant
    unsigned long long* trace;   // optional phase stamps of the persistent kernel (cg_set_trace)
    int trace_iters;
    int trace_clock;             // 0: clock64 (SM cycles, per SM); 1: %globaltimer (ns, one clock for all SMs)
    // streamed variants (cg_stream.cuh)
    const int* rp_pad;    // rowptr copied into the workspace, padded with nnz (bulk copies of 36 ints)
    double* bslots;       // grid all-reduce inboxes [cta][3][kBarVals][kBarGrid], all-ones when idle
    int cap;              // entries per ring slot (multiple of 4)
    int slots;            // ring depth S
    int pinned;           // P: tiles per CTA that stay in their slot for the whole solve
    int stream_slots;     // Q: slots the other tiles stream through (a multiple of the producer count)
    int slot_bytes;       // cap * 12 + 144, rounded up to 128
    double2* pr0;         // the two {p, r} pair buffers of the folded loop (cg_stream_kernels.cuh)
    double2* pr1;
    int lookahead;        // producer run-ahead (tiles) into a pass the consumers have not started
    int l2_stream;        // 1: the matrix does not fit the L2 -> evict-first hint on its copies
    // compressed index (cg_compress_index): one record per tile, see cg_stream.cuh
    int cmp;              // 1: slots hold {vals span, index record}
    int rec_stride;       // bytes per record: 80 + 128 * ceil(longest row / 4)
    int ncodes_smem;      // entries of the offset table copied into shared memory (32 or 256)
    const unsigned char* idx_rec;   // records, tile t at idx_rec + t * rec_stride
    const int* idx_off;   // kMaxCodes column offsets (col - row) named by the codes
    long long spin_budget;          // cycles any device-side spin may last before the watchdog trips
    int inject_fault;     // tests: producer warp 0 of CTA 0 never copies its inject_fault-th tile (0 = off)
};

constexpr int kTraceSlots = 16;  // stamps per iteration and CTA, see k_persistent

// ---------------------------------------------------------------- small helpers

__device__ __forceinline__ double ld_stream_f64(const double* p) {
    double v;   // matrix values are read once per SpMV: read-only path, do not allocate in L1
    asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ int ld_stream_s32(const int* p) {
    int v;
    asm volatile("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ double ld_global_f64(const double* p) {
    double v;   // explicit global-space load (vectors are read AND written inside one launch: no .nc).
    // No "memory" clobber (it would serialise the batched gathers against the shared-memory
    // loads around them): a thread that reads back its OWN earlier plain store through this
    // must put a compiler barrier between the two (the one place is the R = 0 prologue).
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum of one value per thread over the CTA, fixed order.  Result valid in thread 0.
__device__ __forceinline__ double block_sum(double v, double* sm) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();                       // sm may still be read from a previous call
    if (lane == 0) sm[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < kWarps ? sm[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

// Fixed-order sum of the G per-CTA partials; every thread of the CTA gets the value.
__device__ __forceinline__ double sum_partials(const double* part, int G, double* sm) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (warp == 0) {
        double s = 0.0;
        for (int j = lane; j < G; j += 32) s += __ldcg(part + j);
        s = warp_sum(s);
        if (lane == 0) sm[kWarps] = s;
    }
    __syncthreads();
    return sm[kWarps];
}

// Grid-wide barrier for the cooperative persistent kernel (all CTAs co-resident).
// One arrival counter, never reset inside a solve; `epoch` is the local target.  The spin is
// bounded: after `budget` cycles thread 0 raises *abort and the barrier returns true (in every
// thread of the CTA), after which the caller leaves the loop.
__device__ __forceinline__ bool grid_barrier(unsigned long long* bar, unsigned int G,
                                             unsigned long long& epoch, long long budget, int* abort) {
    __syncthreads();
    int dead = 0;
    if (threadIdx.x == 0) {
        epoch += G;
        __threadfence();
        red_release_add_u64(bar, 1ULL);
        const long long t0 = clock64();
        unsigned n = 0;
        while (ld_acquire_u64(bar) < epoch) {
            if ((++n & 0x3ffu) == 0u && clock64() - t0 > budget) {
                *reinterpret_cast<volatile int*>(abort) = 1;
                dead = 1;
                break;
            }
        }
        // no fence after the poll: the acquire loads pair with the other CTAs' release adds and invalidate
        // this SM's L1 (CCTL.IVALL) themselves
    }
    return __syncthreads_or(dead) != 0;
}

// ---------------------------------------------------------------- K1, variant A
// Sub-warp of TPR lanes per row, straight from global memory.  Generic fallback:
// any CSR matrix, any row length.
template <int TPR, bool DOT>
__device__ __forceinline__ double phase_spmv_vector(const Params& P, const double* x, double* y,
                                                    int cta, int G) {
    const int* __restrict__ rowptr = P.rowptr;
    const int* __restrict__ colind = P.colind;
    const double* __restrict__ vals = P.vals;
    constexpr int kRows = kThreads / TPR;
    const int lir = threadIdx.x % TPR;
    const int sub = threadIdx.x / TPR;
    double dot = 0.0;
    for (long long row0 = (long long)cta * kRows; row0 < P.n; row0 += (long long)G * kRows) {
        const long long row = row0 + sub;
        double acc = 0.0;
        if (row < P.n) {
            const int s = __ldg(rowptr + row), e = __ldg(rowptr + row + 1);
            for (int k = s + lir; k < e; k += 4 * TPR) {
                const int k1 = k + TPR, k2 = k + 2 * TPR, k3 = k + 3 * TPR;
                const bool b1 = k1 < e, b2 = k2 < e, b3 = k3 < e;
                const int c0 = ld_stream_s32(colind + k);
                const int c1 = b1 ? ld_stream_s32(colind + k1) : c0;
                const int c2 = b2 ? ld_stream_s32(colind + k2) : c0;
                const int c3 = b3 ? ld_stream_s32(colind + k3) : c0;
                const double v0 = ld_stream_f64(vals + k);
                const double v1 = b1 ? ld_stream_f64(vals + k1) : 0.0;
                const double v2 = b2 ? ld_stream_f64(vals + k2) : 0.0;
                const double v3 = b3 ? ld_stream_f64(vals + k3) : 0.0;
                const double x0 = ld_global_f64(x + c0), x1 = ld_global_f64(x + c1), x2 = ld_global_f64(x + c2), x3 = ld_global_f64(x + c3);
                acc = fma(v0, x0, acc);
                acc = fma(v1, x1, acc);
                acc = fma(v2, x2, acc);
                acc = fma(v3, x3, acc);
            }
        }
#pragma unroll
        for (int o = TPR / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (row < P.n && lir == 0) {
            y[row] = acc;
            if (DOT) dot = fma(acc, x[row], dot);
        }
    }
    return dot;
}

template <bool DOT>
__device__ __forceinline__ double phase_spmv_vector_dispatch(const Params& P, const double* x,
                                                             double* y, int cta, int G) {
    switch (P.tpr) {
        case 2:  return phase_spmv_vector<2, DOT>(P, x, y, cta, G);
        case 4:  return phase_spmv_vector<4, DOT>(P, x, y, cta, G);
        case 8:  return phase_spmv_vector<8, DOT>(P, x, y, cta, G);
        case 16: return phase_spmv_vector<16, DOT>(P, x, y, cta, G);
        default: return phase_spmv_vector<32, DOT>(P, x, y, cta, G);
    }
}

// ---------------------------------------------------------------- mbarrier / bulk-copy primitives
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                 :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) { }
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1], %2, [%3], %4;"
        :: "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy) : "memory");
}
__device__ __forceinline__ void bulk_g2s_plain(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        :: "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}

// ---------------------------------------------------------------- vector phases

// Prologue: r = b - q (q = A x0); p = r (or D^-1 r); partials of r.r, b.b, r.z.
__device__ __forceinline__ void phase_init_residual(const Params& P, int cta, int G, double* sm) {
    const double* __restrict__ b = P.b;
    const double* __restrict__ q = P.q;
    const double* __restrict__ dinv = P.dinv;
    double* __restrict__ r = P.r;
    double* __restrict__ p = P.p;
    double arr = 0.0, abb = 0.0, arz = 0.0;
    const long long stride = (long long)G * kThreads;
    for (long long i = (long long)cta * kThreads + threadIdx.x; i < P.n; i += stride) {
        const double bi = b[i];
        const double ri = bi - q[i];
        r[i] = ri;
        abb = fma(bi, bi, abb);
        arr = fma(ri, ri, arr);
        if (P.precond) {
            const double zi = dinv[i] * ri;
            p[i] = zi;
            arz = fma(ri, zi, arz);
        } else {
            p[i] = ri;
        }
    }
    double t = block_sum(arr, sm); if (threadIdx.x == 0) P.part1[cta] = t;
    t = block_sum(abb, sm);        if (threadIdx.x == 0) P.part2[cta] = t;
    if (P.precond) { t = block_sum(arz, sm); if (threadIdx.x == 0) P.part3[cta] = t; }
}

// Streaming accesses for x: touched exactly once per iteration (read + write in K2), so it
// is marked evict-first and leaves the L2 to p, q, r, which are re-read by the next phase.
__device__ __forceinline__ double2 ld_cs_f64x2(const double2* p) {
    double2 v;
    asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_cs_f64x2(double2* p, double2 v) {
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" :: "l"(p), "d"(v.x), "d"(v.y) : "memory");
}

// VU = double2 elements in flight per thread and array.  It only batches the loads; the
// per-thread accumulation order (hence every bit of the result) does not depend on it.

// K2: x += alpha p ; r -= alpha q ; partial r.r (and r.z with Jacobi).
template <int kVecUnroll>
__device__ __forceinline__ void phase_update_xr(const Params& P, double alpha, int cta, int G,
                                                double* sm) {
    const double na = -alpha;
    double arr = 0.0, arz = 0.0;
    const long long np2 = P.n >> 1;
    const long long stride = (long long)G * kThreads;
    double2* x2 = reinterpret_cast<double2*>(P.x);
    double2* r2 = reinterpret_cast<double2*>(P.r);
    const double2* p2 = reinterpret_cast<const double2*>(P.p);
    const double2* q2 = reinterpret_cast<const double2*>(P.q);
    const double2* d2 = reinterpret_cast<const double2*>(P.dinv);
    for (long long i0 = (long long)cta * kThreads + threadIdx.x; i0 < np2; i0 += stride * kVecUnroll) {
        double2 xv[kVecUnroll], rv[kVecUnroll], pv[kVecUnroll], qv[kVecUnroll], dv[kVecUnroll];
#pragma unroll
        for (int u = 0; u < kVecUnroll; ++u) {
            const long long i = i0 + u * stride;
            if (i < np2) {
                xv[u] = ld_cs_f64x2(x2 + i); rv[u] = r2[i]; pv[u] = p2[i]; qv[u] = q2[i];
                if (P.precond) dv[u] = d2[i];
            }
        }
#pragma unroll
        for (int u = 0; u < kVecUnroll; ++u) {
            const long long i = i0 + u * stride;
            if (i < np2) {
                xv[u].x = fma(alpha, pv[u].x, xv[u].x); xv[u].y = fma(alpha, pv[u].y, xv[u].y);
                rv[u].x = fma(na, qv[u].x, rv[u].x);    rv[u].y = fma(na, qv[u].y, rv[u].y);
                st_cs_f64x2(x2 + i, xv[u]); r2[i] = rv[u];
                arr = fma(rv[u].x, rv[u].x, arr); arr = fma(rv[u].y, rv[u].y, arr);
                if (P.precond) {
                    arz = fma(rv[u].x, dv[u].x * rv[u].x, arz);
                    arz = fma(rv[u].y, dv[u].y * rv[u].y, arz);
                }
            }
        }
    }
    if ((P.n & 1) && cta == G - 1 && threadIdx.x == kThreads - 1) {      // odd tail element
        const long long i = P.n - 1;
        const double xi = fma(alpha, P.p[i], P.x[i]);
        const double ri = fma(na, P.q[i], P.r[i]);
        P.x[i] = xi; P.r[i] = ri;
        arr = fma(ri, ri, arr);
        if (P.precond) arz = fma(ri, P.dinv[i] * ri, arz);
    }
    double t = block_sum(arr, sm); if (threadIdx.x == 0) P.part1[cta] = t;
    if (P.precond) { t = block_sum(arz, sm); if (threadIdx.x == 0) P.part2[cta] = t; }
}

// K3: p = r + beta p   (Jacobi: p = D^-1 r + beta p).
template <int kVecUnroll>
__device__ __forceinline__ void phase_update_p(const Params& P, double beta, int cta, int G) {
    const long long np2 = P.n >> 1;
    const long long stride = (long long)G * kThreads;
    double2* p2 = reinterpret_cast<double2*>(P.p);
    const double2* r2 = reinterpret_cast<const double2*>(P.r);
    const double2* d2 = reinterpret_cast<const double2*>(P.dinv);
    constexpr int U = 2 * kVecUnroll;
    for (long long i0 = (long long)cta * kThreads + threadIdx.x; i0 < np2; i0 += stride * U) {
        double2 pv[U], rv[U], dv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = i0 + u * stride;
            if (i < np2) { pv[u] = p2[i]; rv[u] = r2[i]; if (P.precond) dv[u] = d2[i]; }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long i = i0 + u * stride;
            if (i < np2) {
                if (P.precond) { rv[u].x *= dv[u].x; rv[u].y *= dv[u].y; }
                pv[u].x = fma(beta, pv[u].x, rv[u].x); pv[u].y = fma(beta, pv[u].y, rv[u].y);
                p2[i] = pv[u];
            }
        }
    }
    if ((P.n & 1) && cta == G - 1 && threadIdx.x == kThreads - 1) {
        const long long i = P.n - 1;
        double ri = P.r[i];
        if (P.precond) ri *= P.dinv[i];
        P.p[i] = fma(beta, P.p[i], ri);
    }
}

// x = 0 (the b = 0 convention)
__device__ __forceinline__ void phase_zero_x(const Params& P, int cta, int G) {
    const long long stride = (long long)G * kThreads;
    for (long long i = (long long)cta * kThreads + threadIdx.x; i < P.n; i += stride) P.x[i] = 0.0;
}

}  // namespace cgk
