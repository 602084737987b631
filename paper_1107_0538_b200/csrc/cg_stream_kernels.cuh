// cg_stream_kernels.cuh -- kernel entry points of the streamed CG path (see cg_stream.cuh).
// Every kernel is launched with 32 (W + NP) threads: W consumer warps and the producer
// warps, which return at once in kernels that do not stream the matrix.
#pragma once
#include "cg_stream.cuh"
#include "../../include/cg.h"
#include <limits.h>

namespace cgs {

__device__ __forceinline__ bool finite_d(double v) { return fabs(v) <= 1.79769313486231570e308; }

// Everything the loop decides from (rr, bb) before the first iteration.
__device__ __forceinline__ void decide_start(const Params& P, double rr, double bb, int* stop,
                                             int* status, double* thresh) {
    *thresh = P.rtol * sqrt(bb);
    *stop = 0; *status = CG_OK;
    if (bb == 0.0 || sqrt(rr) <= *thresh) { *stop = 1; *status = CG_OK; }
    else if (P.maxit <= 0) { *stop = 1; *status = CG_MAXIT; }
}

#define CGS_PROLOGUE(W)                                                         \
    extern __shared__ __align__(128) unsigned char dyn[];                       \
    Ring rg = ring_view(P, dyn);                                                \
    const int cta = blockIdx.x, G = gridDim.x;                                  \
    const int warp = threadIdx.x >> 5;                                          \
    long long tb; int Tc;                                                       \
    cta_tiles(P, cta, G, tb, Tc);                                               \
    (void)warp

// ---- cg_spmv: y = A x
template <int W, int NP, int U, bool GF, bool CMP, bool CHK = false>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks_spmv(Params P, const double* x, double* y) {
    CGS_PROLOGUE(W);
    ring_init(P, rg);
    if (warp >= W) { producer_loop<CMP, CHK>(P, rg, tb, Tc, 1, warp - W, NP); return; }
    if constexpr (NP == 0) consumers_pin_tiles<W, CMP, CHK>(P, rg, tb, Tc);
    phase_spmv_tiles<W, U, false, CMP, GF, CHK>(P, rg, x, y, tb, Tc, RingPos{0u, 0u, 0u});
}

// ---- stand-alone kernels of loop modes 1 (graph) and 2 (stepwise).  They read Params from
// ---- device memory so that a captured graph survives across solves.

template <int W, int NP, int U, bool GF, bool CMP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks_init_spmv(const Params* __restrict__ dp) {
    const Params P = *dp;
    CGS_PROLOGUE(W);
    ring_init(P, rg);
    if (warp >= W) { producer_loop<CMP>(P, rg, tb, Tc, 1, warp - W, NP); return; }
    if constexpr (NP == 0) consumers_pin_tiles<W, CMP>(P, rg, tb, Tc);
    phase_spmv_tiles<W, U, false, CMP, GF>(P, rg, P.x, P.q, tb, Tc, RingPos{0u, 0u, 0u});
}

template <int W, int NP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks_init_residual(const Params* __restrict__ dp) {
    const Params P = *dp;
    CGS_PROLOGUE(W);
    if (warp >= W) return;
    double arr = 0.0, abb = 0.0, arz = 0.0;
    if (P.precond) phase_init_tiles<W, true>(P, tb, Tc, arr, abb, arz);
    else           phase_init_tiles<W, false>(P, tb, Tc, arr, abb, arz);
    double t = block_sum_w<W>(arr, rg.red); if (threadIdx.x == 0) P.part1[cta] = t;
    t = block_sum_w<W>(abb, rg.red);        if (threadIdx.x == 0) P.part2[cta] = t;
    if (P.precond) { t = block_sum_w<W>(arz, rg.red); if (threadIdx.x == 0) P.part3[cta] = t; }
}

template <int W, int NP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks_init_scalars(const Params* __restrict__ dp) {
    const Params P = *dp;
    CGS_PROLOGUE(W);
    if (warp >= W) return;
    double rr = sum_partials_w<W>(P.part1, G, rg.red);
    const double bb = sum_partials_w<W>(P.part2, G, rg.red);
    const double rz = P.precond ? sum_partials_w<W>(P.part3, G, rg.red) : rr;
    if (bb == 0.0) { phase_zero_x_tiles<W>(P, tb, Tc); rr = 0.0; }
    if (cta == 0 && threadIdx.x == 0) {
        int stop, status; double thresh;
        decide_start(P, rr, bb, &stop, &status, &thresh);
        if (P.precond && P.scal->diag_bad) { stop = 1; status = CG_BREAKDOWN; }
        Scal* S = P.scal;
        S->bb = bb; S->thresh = thresh;
        S->st[0].rr = rr; S->st[0].rz = rz; S->st[0].k = 0; S->st[0].stop = stop; S->st[0].status = status;
        if (P.hist) P.hist[0] = sqrt(rr);
        S->out_iters = 0; S->out_status = status; S->out_res = sqrt(rr);
    }
}

template <int W, int NP, int U, bool GF, bool CMP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks1_spmv_dot(const Params* __restrict__ dp, int s) {
    const Params P = *dp;
    if (P.scal->st[s].stop) return;
    CGS_PROLOGUE(W);
    if (cta == 0 && threadIdx.x == 0) P.scal->brk[s] = 0;
    ring_init(P, rg);
    if (warp >= W) { producer_loop<CMP>(P, rg, tb, Tc, 1, warp - W, NP); return; }
    if constexpr (NP == 0) consumers_pin_tiles<W, CMP>(P, rg, tb, Tc);
    const double d = phase_spmv_tiles<W, U, true, CMP, GF>(P, rg, P.p, P.q, tb, Tc, RingPos{0u, 0u, 0u});
    const double t = block_sum_w<W>(d, rg.red);
    if (threadIdx.x == 0) P.part0[cta] = t;
}

template <int W, int NP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks2_update_xr(const Params* __restrict__ dp, int s) {
    const Params P = *dp;
    if (P.scal->st[s].stop) return;
    CGS_PROLOGUE(W);
    if (warp >= W) return;
    const double pq = sum_partials_w<W>(P.part0, G, rg.red);
    if (!(pq > 0.0) || !finite_d(pq)) {
        if (cta == 0 && threadIdx.x == 0) P.scal->brk[s] = 1;
        return;
    }
    const double alpha = P.scal->st[s].rz / pq;
    double arr = 0.0, arz = 0.0;
    if (P.precond) phase_xr_tiles<W, true>(P, alpha, tb, Tc, arr, arz);
    else           phase_xr_tiles<W, false>(P, alpha, tb, Tc, arr, arz);
    double t = block_sum_w<W>(arr, rg.red); if (threadIdx.x == 0) P.part1[cta] = t;
    if (P.precond) { t = block_sum_w<W>(arz, rg.red); if (threadIdx.x == 0) P.part2[cta] = t; }
}

template <int W, int NP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks3_update_p(const Params* __restrict__ dp, int s) {
    const Params P = *dp;
    CGS_PROLOGUE(W);
    if (warp >= W) return;
    Scal* S = P.scal;
    const State st = S->st[s];
    const bool lead = cta == 0 && threadIdx.x == 0;
    if (st.stop) { if (lead) S->st[s ^ 1] = st; return; }
    if (S->brk[s]) {
        if (lead) {
            State nx = st; nx.stop = 1; nx.status = CG_BREAKDOWN;
            S->st[s ^ 1] = nx;
            S->out_iters = st.k; S->out_status = CG_BREAKDOWN; S->out_res = sqrt(st.rr);
        }
        return;
    }
    const double rr = sum_partials_w<W>(P.part1, G, rg.red);
    const double rz = P.precond ? sum_partials_w<W>(P.part2, G, rg.red) : rr;
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
    if (!stop) {
        if (P.precond) phase_p_tiles<W, true>(P, beta, tb, Tc);
        else           phase_p_tiles<W, false>(P, beta, tb, Tc);
    }
}

// ---- loop mode 0: the whole solve as ONE cooperative persistent kernel.
// R > 0: every consumer thread owns at most R rows (tiles warp, warp + W, ...) and keeps
//        x, r, p, q (and D^-1) of those rows in registers from the prologue to the end; the
//        only vector traffic left per iteration is the store of p and the gathers of K1.
// R = 0: vectors in global memory (systems with more than R_max * 32 * W * G rows).
// Scalars live in registers, identical in every CTA.
//
// The synchronisations of one iteration, in order, are fixed HERE and nowhere else:
//   plain loop   all-reduce (p.q) after K1, all-reduce (r.r) after K2, both carrying only their
//                payload, then the counter barrier after K3 that publishes p;
//   folded loop  (FOLD: R > 0, no preconditioner) all-reduce (p.q) after K1, then a FENCED
//                all-reduce (r.r) after K2 that also publishes the {p, r} pairs the next K1
//                gathers; K3 happens inside that K1.
// grid_allreduce's slot recycling needs a fully fenced synchronisation strictly between any
// all-reduce and the third all-reduce after it (see cg_stream.cuh); plan_is_safe checks that
// for the cyclic sequence, and the call sites below take their kind from the plan.
// Time stamp of the phase trace: SM cycles, or (option "trace_clock" = 1) the nanosecond clock all SMs share,
// which makes stamps of different CTAs comparable (arrival and release skew at the grid synchronisations).
__device__ __forceinline__ unsigned long long trace_now(const Params& P) {
    if (P.trace_clock) { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
    return (unsigned long long)clock64();
}
enum SyncKind { kArRelaxed = 0, kArFenced = 1, kCounter = 2 };
template <bool FOLD> struct SyncPlan;
template <> struct SyncPlan<false> { static constexpr int n = 3; static constexpr SyncKind seq[3] = {kArRelaxed, kArRelaxed, kCounter}; };
template <> struct SyncPlan<true>  { static constexpr int n = 2; static constexpr SyncKind seq[2] = {kArRelaxed, kArFenced}; };

template <class Plan> constexpr bool plan_is_safe() {
    for (int i = 0; i < Plan::n; ++i) {
        if (Plan::seq[i] == kCounter) continue;
        int ars = 0; bool fenced = false;
        for (int d = 1; d <= 4 * Plan::n && ars < 3; ++d) {       // walk on (cyclically) to the third all-reduce after i
            const SyncKind k = Plan::seq[(i + d) % Plan::n];
            if (k != kCounter) { ++ars; if (ars == 3) break; }
            if (k == kArFenced || k == kCounter) fenced = true;
        }
        if (!fenced) return false;
    }
    return true;
}
static_assert(plan_is_safe<SyncPlan<false>>() && plan_is_safe<SyncPlan<true>>(), "all-reduce slots could be rewritten before their reset is ordered");

// Step STEP of the plan: an all-reduce of v (NV values) or the payload-free counter barrier.
template <int W, class Plan, int STEP, int NV>
__device__ __forceinline__ bool iter_sync(const Params& P, const Ring& rg, unsigned& bcount, unsigned long long& nbar,
                                          int cta, int G, double (&v)[NV], unsigned long long* dbg = nullptr) {
    static_assert(STEP < Plan::n, "no such step");
    if constexpr (Plan::seq[STEP] == kCounter) return grid_barrier_counter<W>(P, rg, nbar, G, dbg);
    else return grid_allreduce<W, NV, Plan::seq[STEP] == kArFenced>(P, rg, bcount, cta, G, v, dbg);
}

template <int W, int NP, int U, bool GF, int R, bool PRE, bool FOLD, bool CMP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks_persistent(Params P) {
    static_assert(!FOLD || (R > 0 && !PRE), "the folded loop needs the vectors in registers and no preconditioner");
    using Plan = SyncPlan<FOLD>;
    CGS_PROLOGUE(W);
    ring_init(P, rg);
    if (warp >= W) { producer_loop<CMP>(P, rg, tb, Tc, LLONG_MAX, warp - W, NP); return; }
    if constexpr (NP == 0) consumers_pin_tiles<W, CMP>(P, rg, tb, Tc);
    const int lane = threadIdx.x & 31;
    const bool lead = cta == 0 && threadIdx.x == 0;
    Scal* S = P.scal;
    unsigned bcount = 0;
    unsigned long long nbar = 0;
    unsigned long long pass = 0;
    RingPos pos{0u, 0u, 0u};
    constexpr int RR = R > 0 ? R : 1;
    double xr[RR], rv[RR], pv[RR], qv[RR], dv[RR];
    long long row[RR];

    // a0 prologue: q = A x0 ; r = b - q ; p = r ; rr, bb
    double arr = 0.0, abb = 0.0, arz = 0.0;
    consumers_begin_pass(rg, pass);
    if constexpr (R > 0) {
        double bv[RR];
#pragma unroll
        for (int kk = 0; kk < R; ++kk) {
            const int j = warp + kk * W;
            const long long i = (tb + j) * kTileRows + lane;
            row[kk] = (j < Tc && i < P.n) ? i : -1;
            xr[kk] = 0.0; bv[kk] = 0.0; dv[kk] = 1.0; qv[kk] = 0.0; rv[kk] = 0.0; pv[kk] = 0.0;
            if (row[kk] >= 0) { xr[kk] = P.x[i]; bv[kk] = P.b[i]; if (PRE) dv[kk] = P.dinv[i]; }
        }
#pragma unroll
        for (int kk = 0; kk < R; ++kk) {
            const int j = warp + kk * W;
            if (j < Tc) qv[kk] = consume_tile<U, false, CMP, GF>(rg, P.x, pos, j, lane, (int)((tb + j) * kTileRows + lane));
        }
#pragma unroll
        for (int kk = 0; kk < R; ++kk) {
            if (row[kk] < 0) continue;
            const double ri = bv[kk] - qv[kk];
            rv[kk] = ri;
            abb = fma(bv[kk], bv[kk], abb);
            arr = fma(ri, ri, arr);
            if (PRE) { const double zi = dv[kk] * ri; pv[kk] = zi; arz = fma(ri, zi, arz); }
            else pv[kk] = ri;
            if (FOLD) P.pr0[row[kk]] = make_double2(pv[kk], rv[kk]);      // the pair the first K1 gathers
            else P.p[row[kk]] = pv[kk];
        }
    } else {
        phase_spmv_tiles<W, U, false, CMP, GF>(P, rg, P.x, P.q, tb, Tc, pos);
        asm volatile("" ::: "memory");                          // q below is what this thread just stored
        phase_init_tiles<W, PRE>(P, tb, Tc, arr, abb, arz);     // reads only this thread's own q
    }
    ++pass; pos = ring_next_pass(rg, pos, Tc);
    // Short-row kernels (gather-first with U = 9: the host picks them when no row has more than 9 entries):
    // a warp whose tiles are all pinned and complete keeps several tiles' gathers in flight (short_batch).
    constexpr bool SB = ShortBatchKernel<U, GF, CMP, R>::value && !FOLD;
    bool batch = false;
    if constexpr (SB) batch = tiles_are_short<W, R>(rg, warp, lane, tb, Tc);
    double rr, bb, rz;
    bool dead;
    {
        double v[PRE ? 3 : 2];
        v[0] = arr; v[1] = abb;
        if (PRE) v[PRE ? 2 : 0] = arz;
        dead = grid_allreduce<W, (PRE ? 3 : 2), true>(P, rg, bcount, cta, G, v);
        rr = v[0]; bb = v[1]; rz = PRE ? v[PRE ? 2 : 0] : rr;
    }
    if (bb == 0.0) {
        if constexpr (R > 0) {
#pragma unroll
            for (int kk = 0; kk < R; ++kk) xr[kk] = 0.0;
        } else {
            phase_zero_x_tiles<W>(P, tb, Tc);
        }
        rr = 0.0;
    }
    long long k = 0; int stop, status; double thresh;
    decide_start(P, rr, bb, &stop, &status, &thresh);
    if (PRE && S->diag_bad) { stop = 1; status = CG_BREAKDOWN; }
    if (dead) { stop = 1; status = CG_ETIMEOUT; }
    if (lead && P.hist) P.hist[0] = sqrt(rr);

    // Optional trace (cg_set_trace): thread 0 of every CTA stamps clock64 at 8 points of each
    // of the first trace_iters iterations: 0 start, 1 K1 done, 2 past all-reduce 1, 3 K2 done,
    // 4 past all-reduce 2, 5 beta known, 6 K3 done, 7 past barrier 3.
    unsigned long long* tr = (P.trace && threadIdx.x == 0)
        ? P.trace + (size_t)cta * (P.trace_iters + 1) * kTraceSlots : nullptr;
    unsigned long long full_wait = 0;
    if (tr) rg.acc = &full_wait;
    // Folded loop: cur = which pair buffer holds the {p, r} the next K1 gathers; the first K1 runs
    // with beta = 0, for which fma(beta, p, r) is r = p_0 to the bit.
    double beta_prev = 0.0;
    int cur = 0;
#define CGS_STAMP(it, slot) do { if (tr && (it) < P.trace_iters) tr[(it) * kTraceSlots + (slot)] = trace_now(P); } while (0)
    while (!stop) {
        CGS_STAMP(k, 0);
        // K1: q = A p, partial p.q
        double dot = 0.0;
        consumers_begin_pass(rg, pass);
        if constexpr (R > 0) {
            if constexpr (FOLD) {
                // K3 folded in: p = r + beta p for the rows this thread owns (registers, and
                // the other pair buffer for next iteration's gathers) ...
                const double2* psrc = cur ? P.pr1 : P.pr0;
                double2* pdst = cur ? P.pr0 : P.pr1;
#pragma unroll
                for (int kk = 0; kk < R; ++kk) {
                    if (row[kk] < 0) continue;
                    pv[kk] = fma(beta_prev, pv[kk], rv[kk]);
                    pdst[row[kk]].x = pv[kk];
                }
                // ... and, recomputed on the fly, for every column the SpMV gathers
#pragma unroll
                for (int kk = 0; kk < R; ++kk) {
                    const int j = warp + kk * W;
                    if (j < Tc) {
                        qv[kk] = consume_tile<(U > 9 ? 9 : U), true, CMP, GF>(rg, reinterpret_cast<const double*>(psrc), pos, j, lane,
                                                            (int)((tb + j) * kTileRows + lane), beta_prev);
                        if (row[kk] >= 0) dot = fma(qv[kk], pv[kk], dot);
                    }
                }
                cur ^= 1;
            } else {
                if constexpr (SB) {
                    k1_resident_tiles<W, U, R, CMP, GF>(rg, P.p, pos, warp, lane, tb, Tc, batch, qv);
#pragma unroll
                    for (int kk = 0; kk < R; ++kk)
                        if (warp + kk * W < Tc && row[kk] >= 0) dot = fma(qv[kk], pv[kk], dot);
                } else {
#pragma unroll
                    for (int kk = 0; kk < R; ++kk) {
                        const int j = warp + kk * W;
                        if (j < Tc) {
                            qv[kk] = consume_tile<U, false, CMP, GF>(rg, P.p, pos, j, lane, (int)((tb + j) * kTileRows + lane));
                            if (row[kk] >= 0) dot = fma(qv[kk], pv[kk], dot);
                        }
                    }
                }
            }
        } else {
            dot = phase_spmv_tiles<W, U, true, CMP, GF>(P, rg, P.p, P.q, tb, Tc, pos);
        }
        ++pass; pos = ring_next_pass(rg, pos, Tc);
        CGS_STAMP(k, 1);
        double v1[1] = {dot};
        dead = iter_sync<W, Plan, 0>(P, rg, bcount, nbar, cta, G, v1);
        CGS_STAMP(k, 2);
        if (dead) { stop = 1; status = CG_ETIMEOUT; break; }
        // scalar alpha (every CTA, same order, same value)
        const double pq = v1[0];
        if (!(pq > 0.0) || !finite_d(pq)) { stop = 1; status = CG_BREAKDOWN; break; }
        const double alpha = rz / pq;
        // K2: x += alpha p ; r -= alpha q ; partial r.r
        arr = 0.0; arz = 0.0;
        if constexpr (R > 0) {
            const double na = -alpha;
            double2* pnext = cur ? P.pr1 : P.pr0;              // FOLD: the buffer this K1 stored p into
#pragma unroll
            for (int kk = 0; kk < R; ++kk) {
                if (row[kk] < 0) continue;
                xr[kk] = fma(alpha, pv[kk], xr[kk]);
                rv[kk] = fma(na, qv[kk], rv[kk]);
                arr = fma(rv[kk], rv[kk], arr);
                if (PRE) arz = fma(rv[kk], dv[kk] * rv[kk], arz);
                if (FOLD) pnext[row[kk]].y = rv[kk];          // gathered by the next K1
            }
        } else {
            phase_xr_tiles<W, PRE>(P, alpha, tb, Tc, arr, arz);
        }
        CGS_STAMP(k, 3);
        double v2[PRE ? 2 : 1];
        v2[0] = arr;
        if (PRE) v2[PRE ? 1 : 0] = arz;
        dead = iter_sync<W, Plan, 1>(P, rg, bcount, nbar, cta, G, v2);      // FOLD: fenced, publishes the pairs
        CGS_STAMP(k, 4);
        if (dead) { stop = 1; status = CG_ETIMEOUT; break; }
        // scalar beta, continue-condition
        const double rr_new = v2[0];
        const double rz_new = PRE ? v2[PRE ? 1 : 0] : rr_new;
        const double beta = rz_new / rz;
        rr = rr_new; rz = rz_new;
        const double res = sqrt(rr);
        CGS_STAMP(k, 5);
        k += 1;
        if (lead && P.hist) P.hist[k] = res;
        if (res <= thresh) { stop = 1; status = CG_OK; break; }
        if (k >= P.maxit) { stop = 1; status = CG_MAXIT; break; }
        if constexpr (FOLD) {              // K3 happens inside the next K1
            beta_prev = beta;
            CGS_STAMP(k - 1, 6);
            CGS_STAMP(k - 1, 7);
        } else {
            // K3: p = r + beta p
            if constexpr (R > 0) {
#pragma unroll
                for (int kk = 0; kk < R; ++kk) {
                    if (row[kk] < 0) continue;
                    const double zi = PRE ? rv[kk] * dv[kk] : rv[kk];
                    pv[kk] = fma(beta, pv[kk], zi);
                    P.p[row[kk]] = pv[kk];
                }
            } else {
                phase_p_tiles<W, PRE>(P, beta, tb, Tc);
            }
            CGS_STAMP(k - 1, 6);
            double none[1] = {0.0};
            dead = iter_sync<W, Plan, Plan::n - 1>(P, rg, bcount, nbar, cta, G, none,      // publishes p
                                                   (tr && k - 1 < P.trace_iters) ? tr + (k - 1) * kTraceSlots + 8 : nullptr);
            CGS_STAMP(k - 1, 7);
            if (dead) { stop = 1; status = CG_ETIMEOUT; break; }
        }
    }
#undef CGS_STAMP
    if constexpr (R > 0) {
#pragma unroll
        for (int kk = 0; kk < R; ++kk)
            if (row[kk] >= 0) P.x[row[kk]] = xr[kk];
    }
    if (tr) tr[(size_t)P.trace_iters * kTraceSlots + 3] = full_wait;
    if (threadIdx.x == 0) consumers_stop(rg, pass);
    if (lead) { S->out_iters = k; S->out_status = status; S->out_res = sqrt(rr); }
}

// ---- option "algo" = 1: Chronopoulos-Gear conjugate gradients (second half).
// The same Krylov iteration with ONE reduction per step: w = A r is formed instead of q = A p, the
// two inner products gamma = r.r and delta = w.r share one all-reduce, and s = A p follows from the
// recurrence s = w + beta s.  Per iteration (G. Meurant's form of Chronopoulos & Gear 1989):
//     p = r + beta p ; s = w + beta s ; x += alpha p ; r -= alpha s          (registers of the owner)
//     -- counter barrier: r is published --
//     w = A r  fused with the partials of gamma' = r.r and delta = w.r        (K1)
//     -- all-reduce (gamma', delta) --
//     beta = gamma' / gamma ; alpha = gamma' / (delta - beta gamma' / alpha)   (the denominator is p'.A p')
// Two grid synchronisations per iteration instead of three, 8-byte gathers as in the textbook
// loop.  In exact arithmetic the iterates are those of the textbook recurrence;
// in floating point they differ by rounding, so this is an OPTION, never the default: it is held
// to the same parity bands as the textbook path in the tests and reported beside it.
// k counts in-loop SpMVs as everywhere (the prologue has two: A x0 and A r0); hist[k] = ||r_k||.
// Vectors in registers only (R > 0), no preconditioner; the host falls back to the textbook
// kernel otherwise.
struct SyncPlanCG1 { static constexpr int n = 2; static constexpr SyncKind seq[2] = {kCounter, kArRelaxed}; };
static_assert(plan_is_safe<SyncPlanCG1>(), "all-reduce slots could be rewritten before their reset is ordered");

template <int W, int NP, int U, bool GF, int R, bool CMP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks_persistent_cg1(Params P) {
    static_assert(R > 0, "vectors in registers");
    using Plan = SyncPlanCG1;
    CGS_PROLOGUE(W);
    ring_init(P, rg);
    if (warp >= W) { producer_loop<CMP>(P, rg, tb, Tc, LLONG_MAX, warp - W, NP); return; }
    if constexpr (NP == 0) consumers_pin_tiles<W, CMP>(P, rg, tb, Tc);
    const int lane = threadIdx.x & 31;
    const bool lead = cta == 0 && threadIdx.x == 0;
    Scal* S = P.scal;
    unsigned bcount = 0;
    unsigned long long nbar = 0;
    unsigned long long pass = 0;
    RingPos pos{0u, 0u, 0u};
    double xr[R], rv[R], pv[R], sv[R], wv[R];
    long long row[R];
    double* const rpub = P.p;                 // the published copy of r that K1 gathers

    // prologue: r0 = b - A x0 (published), then w0 = A r0 with gamma0 = r0.r0, delta0 = w0.r0, b.b
    double abb = 0.0;
    consumers_begin_pass(rg, pass);
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        const long long i = (tb + j) * kTileRows + lane;
        row[kk] = (j < Tc && i < P.n) ? i : -1;
        xr[kk] = 0.0; rv[kk] = 0.0; pv[kk] = 0.0; sv[kk] = 0.0; wv[kk] = 0.0;
        double bi = 0.0;
        if (row[kk] >= 0) { xr[kk] = P.x[i]; bi = P.b[i]; }
        rv[kk] = bi;                           // b for now
    }
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        double q = 0.0;
        if (j < Tc) q = consume_tile<U, false, CMP, GF>(rg, P.x, pos, j, lane, (int)((tb + j) * kTileRows + lane));
        if (row[kk] >= 0) {
            abb = fma(rv[kk], rv[kk], abb);
            rv[kk] = rv[kk] - q;
            rpub[row[kk]] = rv[kk];
        }
    }
    ++pass; pos = ring_next_pass(rg, pos, Tc);
    double none[1] = {0.0};
    bool dead = iter_sync<W, Plan, 0>(P, rg, bcount, nbar, cta, G, none);          // r0 is published
    double agam = 0.0, adel = 0.0;
    consumers_begin_pass(rg, pass);
    constexpr bool SB = ShortBatchKernel<U, GF, CMP, R>::value;
    bool batch = false;
    if constexpr (SB) batch = tiles_are_short<W, R>(rg, warp, lane, tb, Tc);
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        if (j < Tc) wv[kk] = consume_tile<U, false, CMP, GF>(rg, rpub, pos, j, lane, (int)((tb + j) * kTileRows + lane));
        if (row[kk] >= 0) { agam = fma(rv[kk], rv[kk], agam); adel = fma(wv[kk], rv[kk], adel); }
    }
    ++pass; pos = ring_next_pass(rg, pos, Tc);
    double gam, del, bb;
    {
        double v[3] = {agam, adel, abb};
        dead = grid_allreduce<W, 3, true>(P, rg, bcount, cta, G, v) || dead;
        gam = v[0]; del = v[1]; bb = v[2];
    }
    if (bb == 0.0) {
#pragma unroll
        for (int kk = 0; kk < R; ++kk) xr[kk] = 0.0;
        gam = 0.0;
    }
    long long k = 0; int stop, status; double thresh;
    decide_start(P, gam, bb, &stop, &status, &thresh);
    if (dead) { stop = 1; status = CG_ETIMEOUT; }
    if (lead && P.hist) P.hist[0] = sqrt(gam);
    double alpha = 0.0, beta = 0.0;
    if (!stop) {
        if (!(del > 0.0) || !finite_d(del)) { stop = 1; status = CG_BREAKDOWN; }      // p0.A p0 = r0.A r0
        else alpha = gam / del;
    }
    unsigned long long* tr = (P.trace && threadIdx.x == 0)
        ? P.trace + (size_t)cta * (P.trace_iters + 1) * kTraceSlots : nullptr;
#define CGS_STAMP(it, slot) do { if (tr && (it) < P.trace_iters) tr[(it) * kTraceSlots + (slot)] = trace_now(P); } while (0)
    while (!stop) {
        // trace slots of this loop, in order: 0 pass start, 1 vector updates done, 2 past the publish
        // barrier, 3 K1 done, 4 past the all-reduce, 5 = 6 = 7 scalars done
        CGS_STAMP(k, 0);
        // vector updates (the textbook's K3 and K2 in one pass over the registers)
        const double na = -alpha;
#pragma unroll
        for (int kk = 0; kk < R; ++kk) {
            if (row[kk] < 0) continue;
            pv[kk] = fma(beta, pv[kk], rv[kk]);
            sv[kk] = fma(beta, sv[kk], wv[kk]);
            xr[kk] = fma(alpha, pv[kk], xr[kk]);
            rv[kk] = fma(na, sv[kk], rv[kk]);
            rpub[row[kk]] = rv[kk];
        }
        CGS_STAMP(k, 1);
        dead = iter_sync<W, Plan, 0>(P, rg, bcount, nbar, cta, G, none,               // publishes r
                                     (tr && k < P.trace_iters) ? tr + k * kTraceSlots + 8 : nullptr);
        CGS_STAMP(k, 2);
        if (dead) { stop = 1; status = CG_ETIMEOUT; break; }
        // K1: w = A r, partials of gamma' = r.r and delta = w.r
        agam = 0.0; adel = 0.0;
        consumers_begin_pass(rg, pass);
        if constexpr (SB) {
            k1_resident_tiles<W, U, R, CMP, GF>(rg, rpub, pos, warp, lane, tb, Tc, batch, wv);
#pragma unroll
            for (int kk = 0; kk < R; ++kk)
                if (warp + kk * W < Tc && row[kk] >= 0) { agam = fma(rv[kk], rv[kk], agam); adel = fma(wv[kk], rv[kk], adel); }
        } else {
#pragma unroll
            for (int kk = 0; kk < R; ++kk) {
                const int j = warp + kk * W;
                if (j < Tc) {
                    wv[kk] = consume_tile<U, false, CMP, GF>(rg, rpub, pos, j, lane, (int)((tb + j) * kTileRows + lane));
                    if (row[kk] >= 0) { agam = fma(rv[kk], rv[kk], agam); adel = fma(wv[kk], rv[kk], adel); }
                }
            }
        }
        ++pass; pos = ring_next_pass(rg, pos, Tc);
        CGS_STAMP(k, 3);
        double v2[2] = {agam, adel};
        dead = iter_sync<W, Plan, 1>(P, rg, bcount, nbar, cta, G, v2);
        CGS_STAMP(k, 4);
        if (dead) { stop = 1; status = CG_ETIMEOUT; break; }
        const double gam_new = v2[0];
        del = v2[1];
        const double res = sqrt(gam_new);
        k += 1;
        if (lead && P.hist) P.hist[k] = res;
        if (res <= thresh) { gam = gam_new; stop = 1; status = CG_OK; break; }
        if (k >= P.maxit) { gam = gam_new; stop = 1; status = CG_MAXIT; break; }
        beta = gam_new / gam;
        const double denom = del - beta * gam_new / alpha;       // = p'.A p' for the next direction
        gam = gam_new;
        if (!(denom > 0.0) || !finite_d(denom)) { stop = 1; status = CG_BREAKDOWN; break; }
        alpha = gam / denom;
        CGS_STAMP(k - 1, 5); CGS_STAMP(k - 1, 6); CGS_STAMP(k - 1, 7);
    }
#undef CGS_STAMP
#pragma unroll
    for (int kk = 0; kk < R; ++kk)
        if (row[kk] >= 0) P.x[row[kk]] = xr[kk];
    if (threadIdx.x == 0) consumers_stop(rg, pass);
    if (lead) { S->out_iters = k; S->out_status = status; S->out_res = sqrt(gam); }
}

// ---- option "algo" = 2: pipelined conjugate gradients (Ghysels & Vanroose 2014), the form of the
// iteration whose ONE reduction is hidden behind the SpMV.  With w = A r and q = A w:
//     gamma = r.r ; delta = w.r                    (partials written BEFORE the barrier below)
//     q = A w                                      (K1; the partials are read while it runs)
//     beta = gamma / gamma_old ; alpha = gamma / (delta - beta gamma / alpha_old)
//     z = q + beta z ; s = w + beta s ; p = r + beta p ; x += alpha p ; r -= alpha s ; w -= alpha z
//     -- counter barrier: w and the partials are published --
// One grid synchronisation per iteration: the counter barrier's release fence and acquire polls make
// every CTA's partials (one plain store per CTA and value, double-buffered by iteration parity)
// visible to everyone who leaves the barrier, so the "all-reduce" is 148 L2 reads per value that
// every warp issues after its K1 tiles and sums in one fixed order: nobody polls, and the
// reduction costs no grid synchronisation of its own.
// Same iterates as the textbook recurrence in exact arithmetic; more recurrences,
// hence more rounding: an OPTION, held to the same parity bands in the tests, never the default.
// hist[k] = ||r_k||; k counts the updates of x (each pass also starts the SpMV of the next
// one before it can know that the stop test is met: that one is the price of the overlap).
template <int W>
__device__ __forceinline__ bool grid_barrier_partials(const Params& P, const Ring& rg, unsigned long long& nbar, int G,
                                                      int cta, int buf, double a, double b, double c) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
    if (lane == 0) { rg.red[warp] = a; rg.red[32 + warp] = b; rg.red[64 + warp] = c; }
    consumer_sync<W>();                    // also: all phase stores of the CTA happen-before the fence below
    if (warp == 0) {
        a = warp_sum(lane < W ? rg.red[lane] : 0.0);
        b = warp_sum(lane < W ? rg.red[32 + lane] : 0.0);
        c = warp_sum(lane < W ? rg.red[64 + lane] : 0.0);
        if (lane == 0) {
            double* slot = P.part0 + (size_t)buf * 3 * kBarGrid + cta;
            slot[0] = a; slot[kBarGrid] = b; slot[2 * kBarGrid] = c;
            unsigned long long* ctr = &P.scal->bar;
            asm volatile("fence.acq_rel.gpu;" ::: "memory");
            asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" :: "l"(ctr), "l"(1ULL) : "memory");
            const unsigned long long target = (++nbar) * (unsigned long long)G;
            bounded_spin(rg, [&] { return ld_acquire_u64(ctr) >= target; });      // acquire poll, as in grid_barrier_counter
            rg.red[kRedTot + kBarVals] = rg.ctl[4] != 0 ? 1.0 : 0.0;
        }
    }
    consumer_sync<W>();
    return rg.red[kRedTot + kBarVals] != 0.0;
}

// Every warp: start the reads of the G per-CTA partials of NV values (lane l takes CTAs l, l + 32, ...).
template <int NV>
__device__ __forceinline__ void partials_issue(const Params& P, int G, int buf, double (&u)[NV][kBarM]) {
    const int lane = threadIdx.x & 31;
    const double* base = P.part0 + (size_t)buf * 3 * kBarGrid;
#pragma unroll
    for (int i = 0; i < NV; ++i)
#pragma unroll
        for (int m = 0; m < kBarM; ++m) {
            const int j = lane + 32 * m;
            u[i][m] = j < G ? __longlong_as_double((long long)ld_relaxed_u64(reinterpret_cast<const unsigned long long*>(base + i * kBarGrid + j))) : 0.0;
        }
}
template <int NV>
__device__ __forceinline__ void partials_sum(const double (&u)[NV][kBarM], double (&tot)[NV]) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double t = 0.0;
#pragma unroll
        for (int m = 0; m < kBarM; ++m) t += u[i][m];
        tot[i] = warp_sum(t);              // xor tree: the same bits in every lane, warp and CTA
    }
}

template <int W, int NP, int U, bool GF, int R, bool CMP>
__global__ void __launch_bounds__(Shape<W, NP>::kThreads, 1) ks_persistent_pipe(Params P) {
    static_assert(R > 0, "vectors in registers");
    CGS_PROLOGUE(W);
    ring_init(P, rg);
    if (warp >= W) { producer_loop<CMP>(P, rg, tb, Tc, LLONG_MAX, warp - W, NP); return; }
    if constexpr (NP == 0) consumers_pin_tiles<W, CMP>(P, rg, tb, Tc);
    const int lane = threadIdx.x & 31;
    const bool lead = cta == 0 && threadIdx.x == 0;
    Scal* S = P.scal;
    unsigned long long nbar = 0;
    unsigned long long pass = 0;
    RingPos pos{0u, 0u, 0u};
    double xr[R], rv[R], pv[R], sv[R], wv[R], zv[R];
    long long row[R];
    // two published vectors, used alternately: pass k gathers w_k from one and stores w_{k+1} into the
    // other, so a CTA that is ahead never overwrites what a CTA still in its K1 is gathering (there is
    // no synchronisation between K1 and the update here, unlike the other loops)
    double* const wpub[2] = {P.p, P.q};

    // prologue: r0 = b - A x0 (published), w0 = A r0 (published with the partials of gamma0, delta0, b.b)
    double abb = 0.0;
    consumers_begin_pass(rg, pass);
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        const long long i = (tb + j) * kTileRows + lane;
        row[kk] = (j < Tc && i < P.n) ? i : -1;
        xr[kk] = 0.0; pv[kk] = 0.0; sv[kk] = 0.0; wv[kk] = 0.0; zv[kk] = 0.0;
        double bi = 0.0;
        if (row[kk] >= 0) { xr[kk] = P.x[i]; bi = P.b[i]; }
        rv[kk] = bi;
    }
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        double q = 0.0;
        if (j < Tc) q = consume_tile<U, false, CMP, GF>(rg, P.x, pos, j, lane, (int)((tb + j) * kTileRows + lane));
        if (row[kk] >= 0) {
            abb = fma(rv[kk], rv[kk], abb);
            rv[kk] = rv[kk] - q;
            wpub[0][row[kk]] = rv[kk];
        }
    }
    ++pass; pos = ring_next_pass(rg, pos, Tc);
    bool dead = grid_barrier_partials<W>(P, rg, nbar, G, cta, 0, 0.0, 0.0, abb);            // r0 and b.b are published
    double agam = 0.0, adel = 0.0;
    consumers_begin_pass(rg, pass);
    constexpr bool SB = ShortBatchKernel<U, GF, CMP, R>::value;
    bool batch = false;
    if constexpr (SB) batch = tiles_are_short<W, R>(rg, warp, lane, tb, Tc);
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        if (j < Tc) wv[kk] = consume_tile<U, false, CMP, GF>(rg, wpub[0], pos, j, lane, (int)((tb + j) * kTileRows + lane));
        if (row[kk] >= 0) { agam = fma(rv[kk], rv[kk], agam); adel = fma(wv[kk], rv[kk], adel); wpub[1][row[kk]] = wv[kk]; }
    }
    ++pass; pos = ring_next_pass(rg, pos, Tc);
    double bb;
    {
        double u[1][kBarM], t[1];
        const double* base = P.part0 + 2 * kBarGrid;                                            // value 2 of buffer 0
#pragma unroll
        for (int m = 0; m < kBarM; ++m) { const int j = lane + 32 * m; u[0][m] = j < G ? __ldcg(base + j) : 0.0; }
        partials_sum<1>(u, t);
        bb = t[0];
    }
    dead = grid_barrier_partials<W>(P, rg, nbar, G, cta, 1, agam, adel, 0.0) || dead;     // w0 and (gamma0, delta0) are published
    int buf = 1;                               // parity of the published vector AND of the partials this pass reads

    long long k = 0; int stop = 0, status = CG_OK;
    double gam = 0.0, gam_old = 1.0, alpha = 1.0, thresh = P.rtol * sqrt(bb);
    if (dead) { stop = 1; status = CG_ETIMEOUT; }
    unsigned long long* tr = (P.trace && threadIdx.x == 0)
        ? P.trace + (size_t)cta * (P.trace_iters + 1) * kTraceSlots : nullptr;
#define CGS_STAMP(it, slot) do { if (tr && (it) < P.trace_iters) tr[(it) * kTraceSlots + (slot)] = trace_now(P); } while (0)
    while (!stop) {
        CGS_STAMP(k, 0);
        // K1: q = A w
        double qv[R];
        consumers_begin_pass(rg, pass);
        if constexpr (SB) {
#pragma unroll
            for (int kk = 0; kk < R; ++kk) qv[kk] = 0.0;
            k1_resident_tiles<W, U, R, CMP, GF>(rg, wpub[buf], pos, warp, lane, tb, Tc, batch, qv);
        } else {
#pragma unroll
            for (int kk = 0; kk < R; ++kk) {
                const int j = warp + kk * W;
                qv[kk] = 0.0;
                if (j < Tc) qv[kk] = consume_tile<U, false, CMP, GF>(rg, wpub[buf], pos, j, lane, (int)((tb + j) * kTileRows + lane));
            }
        }
        ++pass; pos = ring_next_pass(rg, pos, Tc);
        CGS_STAMP(k, 1);
        // the reduction: every warp reads the 148 x 2 partials (published by the barrier that ended the
        // previous pass) and sums them in the one fixed order.  Issuing these reads before K1 hides their
        // L2 round trip but holds 20 registers through K1, which then spills (measured: K1 9.4 k against
        // 6.9 k cycles); here they cost one exposed round trip and no CTA barrier.
        double u[2][kBarM];
        partials_issue<2>(P, G, buf, u);
        double t2[2];
        partials_sum<2>(u, t2);
        gam = t2[0];
        const double del = t2[1];
        CGS_STAMP(k, 2);
        // continue-condition on ||r_k|| (k = 0: the test "before the first iteration")
        if (bb == 0.0) {
#pragma unroll
            for (int kk = 0; kk < R; ++kk) xr[kk] = 0.0;
            gam = 0.0;
        }
        const double res = sqrt(gam);
        if (lead && P.hist) P.hist[k] = res;
        if (bb == 0.0 || res <= thresh) { stop = 1; status = CG_OK; break; }
        if (k >= P.maxit) { stop = 1; status = CG_MAXIT; break; }
        const double beta = k > 0 ? gam / gam_old : 0.0;
        const double denom = k > 0 ? del - beta * gam / alpha : del;         // = p.A p of the direction about to be used
        if (!(denom > 0.0) || !finite_d(denom)) { stop = 1; status = CG_BREAKDOWN; break; }
        alpha = gam / denom;
        gam_old = gam;
        CGS_STAMP(k, 3); CGS_STAMP(k, 4); CGS_STAMP(k, 5);
        // vector recurrences, registers only; partials of the next gamma, delta
        const double na = -alpha;
        agam = 0.0; adel = 0.0;
#pragma unroll
        for (int kk = 0; kk < R; ++kk) {
            if (row[kk] < 0) continue;
            zv[kk] = fma(beta, zv[kk], qv[kk]);
            sv[kk] = fma(beta, sv[kk], wv[kk]);
            pv[kk] = fma(beta, pv[kk], rv[kk]);
            xr[kk] = fma(alpha, pv[kk], xr[kk]);
            rv[kk] = fma(na, sv[kk], rv[kk]);
            wv[kk] = fma(na, zv[kk], wv[kk]);
            wpub[buf ^ 1][row[kk]] = wv[kk];
            agam = fma(rv[kk], rv[kk], agam);
            adel = fma(wv[kk], rv[kk], adel);
        }
        k += 1;
        CGS_STAMP(k - 1, 6);
        buf ^= 1;
        dead = grid_barrier_partials<W>(P, rg, nbar, G, cta, buf, agam, adel, 0.0);        // the one synchronisation
        CGS_STAMP(k - 1, 7);
        if (dead) { stop = 1; status = CG_ETIMEOUT; break; }
    }
#undef CGS_STAMP
#pragma unroll
    for (int kk = 0; kk < R; ++kk)
        if (row[kk] >= 0) P.x[row[kk]] = xr[kk];
    if (threadIdx.x == 0) consumers_stop(rg, pass);
    if (lead) { S->out_iters = k; S->out_status = status; S->out_res = sqrt(gam); }
}

// ---- cg_probe_grid_sync: the cost of the grid synchronisations themselves, measured with the very
// device functions the solve uses, on the solve's grid (one CTA per SM, cooperative launch).
// kind 0 = counter barrier, 1 = push/poll all-reduce carrying its payload only, 2 = fenced.
// Thread 0 of every CTA writes the cycles of its `reps` synchronisations to out[cta].
template <int W>
__global__ void __launch_bounds__(32 * W, 1) ks_probe_sync(Params P, int kind, int reps, unsigned long long* out) {
    CGS_PROLOGUE(W);
    ring_init(P, rg);
    unsigned bcount = 0;
    unsigned long long nbar = 0;
    double v[1] = {(double)threadIdx.x};
    // one fenced all-reduce first: every CTA is resident and past its set-up before the clock starts
    grid_allreduce<W, 1, true>(P, rg, bcount, cta, G, v);
    const long long t0 = clock64();
    bool dead = false;
    for (int i = 0; i < reps && !dead; ++i) {
        if (kind == 0) dead = grid_barrier_counter<W>(P, rg, nbar, G);
        else if (kind == 1) {
            // a relaxed all-reduce needs a fenced synchronisation within every window of three
            dead = (i % 3 == 2) ? grid_barrier_counter<W>(P, rg, nbar, G) : grid_allreduce<W, 1, false>(P, rg, bcount, cta, G, v);
        } else dead = grid_allreduce<W, 1, true>(P, rg, bcount, cta, G, v);
    }
    if (threadIdx.x == 0) out[cta] = dead ? 0ULL : (unsigned long long)(clock64() - t0);
    (void)tb; (void)Tc;
}

}  // namespace cgs
