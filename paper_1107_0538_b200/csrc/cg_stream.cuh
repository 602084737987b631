// cg_stream.cuh -- the streamed CG path for sm_100a: warp-specialised bulk-async (TMA)
// producers, W consumer warps with one lane per row, grid all-reduce fused with the grid
// barrier, and (for systems small enough) x, r, p, q kept in registers for the whole solve.
//
// What is computed is unchanged ("DGEMV(sparse)" + the CG of
// PAPER.md:76): K1 q = A p with the p.q partials, K2 x += alpha p, r -= alpha q with the r.r
// partials, K3 p = r + beta p, scalars on the device.
//
// Work split.  The matrix is cut into tiles of 32 consecutive rows.  CTA c owns the
// contiguous tiles [c*T/G, (c+1)*T/G); inside a CTA tile j (0-based) belongs to consumer warp
// j mod W, lane l of that warp owns row 32*tile + l in EVERY phase.  The thread that
// computes q_i is therefore the thread that updates x_i, r_i, p_i, and all per-thread
// partial sums are accumulated in tile order: every loop mode (persistent with vectors in
// registers, persistent with vectors in global memory, graph, stepwise) performs the same
// floating-point operations in the same order and gives bitwise identical results.
//
// K1 data flow.  NP extra warps (the producers) walk the CTA's tiles in order and,
// for each, wait for a free ring slot and issue three cp.async.bulk copies (SASS UBLKCP)
// into it: the tile's contiguous vals span, its colind span and its 33 row pointers (36
// ints from a padded copy of rowptr).  Consumers wait on the slot's "full" mbarrier, copy
// their row bounds and entries from shared memory into registers, hand the slot back, then
// gather x through L1/L2.  No consumer ever waits on a row-pointer or matrix load from
// global memory; the only global loads in its loop are the x gathers.  In the persistent
// kernel the producers run ahead into the next iteration's tiles (the matrix does not
// change) while the consumers do K2/K3 and wait at the grid barriers, so K1 starts on a
// full ring.
//
// Alignment of the bulk copies: source, destination and size must be multiples of 16
// bytes.  A tile's span [s, e) is widened to [s & ~3, (e + 3) & ~3), clamped to nnz & ~3;
// the <= 3 entries of the whole matrix past that bound are written into the slot by the
// producer with ordinary loads/stores, so nothing outside the caller's arrays is touched.
#pragma once
#include "cg_kernels.cuh"

namespace cgs {
using namespace cgk;

constexpr int kRpInts = 36;          // 33 row pointers of a tile, padded to 144 bytes
constexpr int kRpPad = 40;           // extra ints at the end of the padded rowptr copy
constexpr int kBarVals = 3;          // values per grid all-reduce
constexpr int kBarGrid = 160;        // max CTAs of a streamed persistent grid (1 per SM; B200 has 148)
constexpr int kBarM = kBarGrid / 32;
constexpr int kMaxSlots = 64;
constexpr int kSmemTail = 2304;      // mbarriers + reduction scratch + flags after the slots
constexpr int kRedTot = 96;          // red[0..95]: per-warp partials (3 values x 32 warps); red[96..]: totals

// W consumer warps + NP producer warps per CTA; W + NP is a multiple of 4 so the warps spread
// evenly over the SM's four sub-partitions (their register files bound the registers per thread).
template <int W, int NP> struct Shape {
    static constexpr int kConsumers = W;
    static constexpr int kProducers = NP;
    static constexpr int kConsumerThreads = 32 * W;
    static constexpr int kThreads = 32 * (W + NP);
};
constexpr int kSlotQuantum = 20;     // ring depths are multiples of this (lcm of the producer counts 4 and 5) when they can be

struct Ring {
    unsigned char* slots;
    uint64_t* full;
    uint64_t* empty;
    double* red;                      // 104 doubles of reduction scratch (see kRedTot)
    volatile int* ctl;                // [0] stop flag, [1] passes consumed (low), [2] (high), [3] passes started
    volatile unsigned* tag;           // per slot: 1 + number (mod 2^32) of the tile last issued into it
    int S, slot_bytes, cap;
    int P, Q;                         // pinned slots [0, P) and streaming slots [P, P + Q), P + Q <= S
    unsigned long long* acc;          // optional: cycles this thread waited on full barriers (trace)
    __device__ __forceinline__ double* vals(int slot) const {
        return reinterpret_cast<double*>(slots + (size_t)slot * slot_bytes);
    }
    __device__ __forceinline__ int* cols(int slot) const {
        return reinterpret_cast<int*>(slots + (size_t)slot * slot_bytes + (size_t)cap * 8);
    }
    __device__ __forceinline__ int* rp(int slot) const {
        return reinterpret_cast<int*>(slots + (size_t)slot * slot_bytes + (size_t)cap * 12);
    }
};

__device__ __forceinline__ Ring ring_view(const Params& P, unsigned char* dyn) {
    Ring rg;
    rg.S = P.slots; rg.slot_bytes = P.slot_bytes; rg.cap = P.cap; rg.acc = nullptr;
    rg.P = P.pinned; rg.Q = P.stream_slots;
    rg.slots = dyn;
    unsigned char* tail = dyn + (size_t)P.slots * P.slot_bytes;
    rg.full = reinterpret_cast<uint64_t*>(tail);
    rg.empty = rg.full + kMaxSlots;
    rg.red = reinterpret_cast<double*>(rg.empty + kMaxSlots);
    rg.ctl = reinterpret_cast<volatile int*>(rg.red + 104);
    rg.tag = reinterpret_cast<volatile unsigned*>(rg.ctl + 8);       // kMaxSlots entries
    return rg;
}

// Called by every thread of the CTA (producer warp included) before anything else.
__device__ __forceinline__ void ring_init(const Ring& rg) {
    if ((int)threadIdx.x < rg.S) {
        mbar_init(&rg.full[threadIdx.x], 1);
        mbar_init(&rg.empty[threadIdx.x], 1);
        rg.tag[threadIdx.x] = 0u;
    }
    if (threadIdx.x == 0) { rg.ctl[0] = 0; rg.ctl[1] = 0; rg.ctl[2] = 0; rg.ctl[3] = 0; }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
}

// Barrier among the consumer warps only (the producer never joins it).
template <int W> __device__ __forceinline__ void consumer_sync() {
    asm volatile("bar.sync 1, %0;" :: "n"(32 * W) : "memory");
}

// The CTA's contiguous tile range.
__device__ __forceinline__ void cta_tiles(const Params& P, int cta, int G, long long& tb, int& Tc) {
    const long long ntiles = (P.n + kTileRows - 1) / kTileRows;
    tb = (long long)cta * ntiles / G;
    const long long te = (long long)(cta + 1) * ntiles / G;
    Tc = (int)(te - tb);
}

// ---------------------------------------------------------------- producer

__device__ __forceinline__ void producer_issue(const Params& P, const Ring& rg, int slot, long long t,
                                               int s, int e, uint64_t policy, unsigned tag) {
    const int s4 = s & ~3;
    const int lim = (int)(P.nnz & ~3LL);              // last entry reachable by bulk copies
    int e4 = (e + 3) & ~3;
    if (e4 > lim) e4 = lim;
    const int cnt = e4 > s4 ? e4 - s4 : 0;            // multiple of 4
    double* sv = rg.vals(slot);
    int* sc = rg.cols(slot);
    if (e > lim) {                                    // the matrix's last <= 3 entries, by hand
        for (int k = (lim > s4 ? lim : s4); k < e; ++k) {
            sv[k - s4] = ld_stream_f64(P.vals + k);
            sc[k - s4] = ld_stream_s32(P.colind + k);
        }
    }
    uint64_t* bar = &rg.full[slot];
    rg.tag[slot] = tag;                               // before the arrive below (release): see consume_tile
    mbar_expect_tx(bar, (uint32_t)cnt * 12u + (uint32_t)kRpInts * 4u);
    if (cnt > 0) {
        if (P.l2_stream) {
            bulk_g2s(sv, P.vals + s4, (uint32_t)cnt * 8u, bar, policy);
            bulk_g2s(sc, P.colind + s4, (uint32_t)cnt * 4u, bar, policy);
        } else {
            bulk_g2s_plain(sv, P.vals + s4, (uint32_t)cnt * 8u, bar);
            bulk_g2s_plain(sc, P.colind + s4, (uint32_t)cnt * 4u, bar);
        }
    }
    bulk_g2s_plain(rg.rp(slot), P.rp_pad + t * kTileRows, (uint32_t)kRpInts * 4u, bar);
}

constexpr int kPrefetchBatch = 8;    // tiles per producer warp sent towards the L2 ahead of their ring copies

// Start a tile's vals / colind spans towards the L2 (same widening and clamping as producer_issue).
__device__ __forceinline__ void prefetch_tile_l2(const Params& P, int s, int e) {
    const int s4 = s & ~3;
    const int lim = (int)(P.nnz & ~3LL);
    int e4 = (e + 3) & ~3;
    if (e4 > lim) e4 = lim;
    const int cnt = e4 > s4 ? e4 - s4 : 0;
    if (cnt > 0) {
        const uint64_t pol = l2_policy_evict_first();      // must not push p out of the L2
        asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;"
                     :: "l"(P.vals + s4), "r"((uint32_t)cnt * 8u), "l"(pol) : "memory");
        asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;"
                     :: "l"(P.colind + s4), "r"((uint32_t)cnt * 4u), "l"(pol) : "memory");
    }
}

// Pinned and streamed tiles.  When the matrix is L2-resident anyway (it is re-read every
// iteration), the first P tiles of a CTA are PINNED: tile j < P is copied into slot j once,
// in the first pass, and stays there for the whole solve (no L2 traffic, no shared-memory
// write, no producer work for it in later iterations).  The other Ts = Tc - P tiles of a
// pass are STREAMED through the Q slots [P, P + Q): streamed tile number seq (counted over
// all passes) uses slot P + seq mod Q.  P = Tc (everything pinned, nothing streamed) when
// the CTA's whole slice fits the ring.
//
// A pass starts at stream position `pos` = (slot offset, parity, number) of its first streamed
// tile; streamed tile i of the pass sits i slots further on.
struct RingPos { unsigned slot; unsigned par; unsigned seq; };      // seq: streamed tile number mod 2^32
__device__ __forceinline__ RingPos ring_advance(const Ring& rg, RingPos p, unsigned tiles) {
    const unsigned Q = rg.Q > 0 ? (unsigned)rg.Q : 1u;
    const unsigned t = p.slot + tiles;
    const unsigned q = t / Q;
    RingPos r; r.slot = t - q * Q; r.par = p.par ^ (q & 1u); r.seq = p.seq + tiles;
    return r;
}
// Position of the next pass: a pass streams Tc - P tiles.
__device__ __forceinline__ RingPos ring_next_pass(const Ring& rg, RingPos p, int Tc) {
    return Tc > rg.P ? ring_advance(rg, p, (unsigned)(Tc - rg.P)) : p;
}

// Producer warp q of NP.  The CTA's tiles form one endless sequence: `passes` sweeps over
// [tb, tb + Tc) (a huge number in the persistent kernel, which ends it through the stop flag
// instead); tile number seq sits in slot seq mod S.  This warp serves seq = q, q + NP, ...
// (One warp issuing three bulk copies per tile is a serial instruction stream of several
// hundred cycles per tile -- too slow for one SM's share of the HBM stream, hence NP warps.
// The ring depth S is a multiple of NP, so slot x is always refilled by warp x mod NP, which
// waits for the slot's phases in order: with a different warp per phase a parity wait could
// not tell "two phases ahead" from "ready".)  Tile bounds come from rowptr 32 tiles at a
// time, one per lane; a CTA with <= 32 tiles fetches them once.  The warp runs ahead of the
// consumers by as many tiles as the ring has free slots, also into the next pass, but there
// by at most P.lookahead tiles until the consumers start that pass (ctl[3] counts the
// passes they have started).
__device__ __forceinline__ void producer_loop(const Params& P, const Ring& rg, long long tb, int Tc,
                                              long long passes, int q, int NP) {
    const int lane = threadIdx.x & 31;
    const uint64_t policy = l2_policy_evict_first();
    if (Tc <= 0) return;
    const int Pn = rg.P < Tc ? rg.P : Tc;                  // my CTA's pinned tiles: [0, Pn)
    const int Ts = Tc - Pn;                                 // streamed tiles per pass
    const int Q = rg.Q;
    int s = 0, e = 0;
    const bool cached = Tc <= 32;                           // lane l keeps the bounds of tile l
    if (cached && lane < Tc) {
        s = ld_stream_s32(P.rp_pad + (tb + lane) * kTileRows);
        e = ld_stream_s32(P.rp_pad + (tb + lane) * kTileRows + kTileRows);
    }
    // Pinned tiles: mine are j = q, q + NP, ... < Pn; each goes into slot j once (its slot was
    // never used: no empty wait).  Lane l fetches the bounds of my l-th one (Pn <= 64).
    {
        int ps = 0, pe = 0;
        const int mine = Pn > q ? (Pn - q + NP - 1) / NP : 0;
        if (!cached && lane < mine) {
            const long long t = tb + q + (long long)lane * NP;
            ps = ld_stream_s32(P.rp_pad + t * kTileRows);
            pe = ld_stream_s32(P.rp_pad + t * kTileRows + kTileRows);
        }
        for (int l = 0; l < mine; ++l) {
            const int j = q + l * NP;
            const int si = __shfl_sync(0xffffffffu, cached ? s : ps, cached ? j : l);
            const int ei = __shfl_sync(0xffffffffu, cached ? e : pe, cached ? j : l);
            if (lane == 0) producer_issue(P, rg, j, tb + j, si, ei, policy, (unsigned)j + 1u);
        }
    }
    if (Ts <= 0 || Q <= 0) return;
    unsigned long long seq = (unsigned long long)q;        // next streamed tile number I issue
    long long pass = 0;
    int j = q;                                              // = seq - pass * Ts, index among the streamed tiles
    while (j >= Ts) { j -= Ts; ++pass; }
    unsigned slot = (unsigned)q, par = 0;                   // = seq mod Q, (seq / Q) & 1
    // Optional (option "l2_prefetch", off by default), matrix >> L2: the producers start every
    // tile towards the L2 one batch of their tiles before they copy it into shared memory
    // (cp.async.bulk.prefetch.L2 needs no slot and no barrier), to have more bytes in flight
    // towards HBM than the ring holds.  Measured at config 4: with 4 tiles per warp ahead K1
    // drops from 451 k to 429 k cycles on average but the CTAs drift apart (the barrier
    // after K1 grows from 16 k to 40 k cycles): no gain; 8 and 16 ahead are slower outright.
    const bool pf = P.l2_stream != 0 && P.l2_prefetch != 0;
    const int B = cached ? 32 : (pf ? (P.l2_prefetch > 1 ? P.l2_prefetch : kPrefetchBatch) : 32);
    if (!cached && lane < B) {             // bounds of my first batch
        const int jl = (int)(((long long)j + (long long)lane * NP) % Ts);
        s = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows);
        e = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows + kTileRows);
        if (pf) prefetch_tile_l2(P, s, e);
    }
    bool stopped = false;
    unsigned long long t_wait = 0;
    const long long t_begin = clock64();
    const bool timing = P.trace != nullptr;
    while (pass < passes && !stopped) {
        int s2 = 0, e2 = 0;
        if (!cached) {                     // bounds of the batch AFTER this one; start them towards the L2
            const int jl = (int)(((long long)j + (long long)(B + lane) * NP) % Ts);
            if (lane < B) {
                s2 = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows);
                e2 = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows + kTileRows);
                if (pf) prefetch_tile_l2(P, s2, e2);
            }
        }
        for (int l = 0; l < B && pass < passes; ++l) {
            int ok = 1;
            if (lane == 0) {
                const long long t0 = timing ? clock64() : 0;
                if (passes > 1 && j >= P.lookahead) {
                    while ((long long)rg.ctl[3] <= pass) { if (rg.ctl[0]) { ok = 0; break; } }
                }
                while (ok && !mbar_try_wait(&rg.empty[Pn + slot], par ^ 1u)) {
                    if (rg.ctl[0]) ok = 0;
                }
                if (timing) t_wait += (unsigned long long)(clock64() - t0);
            }
            ok = __shfl_sync(0xffffffffu, ok, 0);
            if (!ok) { stopped = true; break; }
            const int src = cached ? Pn + j : l;
            const int si = __shfl_sync(0xffffffffu, s, src);
            const int ei = __shfl_sync(0xffffffffu, e, src);
            if (lane == 0) producer_issue(P, rg, Pn + (int)slot, tb + Pn + j, si, ei, policy, (unsigned)seq + 1u);
            seq += (unsigned long long)NP;
            j += NP;
            while (j >= Ts) { j -= Ts; ++pass; }
            slot += (unsigned)NP;
            if (slot >= (unsigned)Q) { slot -= (unsigned)Q; par ^= 1u; }
        }
        if (!cached) { s = s2; e = e2; }
    }
    if (timing && lane == 0 && q == 0) {   // producer statistics in the row after the last traced iteration
        unsigned long long* row = P.trace + ((size_t)blockIdx.x * (P.trace_iters + 1) + P.trace_iters) * kTraceSlots;
        row[0] = t_wait; row[1] = (unsigned long long)(clock64() - t_begin); row[2] = seq / (unsigned)NP;
    }
    if (stopped) {
        // Drain: my copies for tiles nobody will consume must land before the CTA exits.  The
        // consumers finished `done` whole passes, i.e. the streamed tiles below done * Ts.
        const unsigned long long done = (((unsigned long long)(unsigned)rg.ctl[2] << 32) | (unsigned)rg.ctl[1])
                                        * (unsigned long long)Ts;
        unsigned long long w = done + (((unsigned long long)q + (unsigned long long)NP
                                        - done % (unsigned long long)NP) % (unsigned long long)NP);
        for (; w < seq; w += (unsigned long long)NP)
            mbar_wait(&rg.full[Pn + (int)(w % (unsigned)Q)], (uint32_t)((w / (unsigned)Q) & 1ULL));
    }
}

// Consumer side of the end of a persistent solve: publish how many passes were consumed,
// then raise the stop flag the producer polls.
__device__ __forceinline__ void consumers_begin_pass(const Ring& rg, unsigned long long pass) {
    if (threadIdx.x == 0) rg.ctl[3] = (int)(pass + 1 > 0x7fffffffULL ? 0x7fffffffULL : pass + 1);
}
__device__ __forceinline__ void consumers_stop(const Ring& rg, unsigned long long passes_done) {
    rg.ctl[1] = (int)(unsigned)(passes_done & 0xffffffffULL);
    rg.ctl[2] = (int)(unsigned)(passes_done >> 32);
    __threadfence_block();
    rg.ctl[0] = 1;
}

// ---------------------------------------------------------------- consumer

// One tile: wait for its slot, y_row = sum_k a_k x[col_k] for this lane's row.  U entries are
// in flight per lane and trip: their column indices and values are read from shared memory,
// then the U gathers are issued, then the FMAs go into three independent accumulators
// (27 = 3 x 9 for the stencil rows).  The trip count is made warp-uniform so that the slot
// can be handed back to the producer as soon as the LAST trip has copied its entries into
// registers -- before the gathers, which are the long-latency part: with U >= the row
// length a slot is held for a few hundred cycles only and nearly the whole ring is in
// flight.  Padding entries (k >= ke) use value 0 and column 0.
//
// FOLD: the gathered operand is not stored anywhere yet: it is p_new[c] = fma(beta, p_old[c],
// r[c]), the very expression K3 evaluates for row c, recomputed here by every thread that
// needs it (x = p_old, r = the residual K2 just stored).  Same operation, same operands, same
// bits as the owner's own update; it saves the third grid synchronisation of an iteration.
template <int U, bool FOLD = false>
__device__ __forceinline__ double consume_tile(const Ring& rg, const double* x, RingPos pos, int j,
                                               int lane, const double* r = nullptr, double beta = 0.0) {
    static_assert(U % 3 == 0, "three accumulators");
    const bool pinned = j < rg.P;
    RingPos at;
    if (pinned) { at.slot = (unsigned)j; at.par = 0u; at.seq = (unsigned)j; }        // its only phase
    else { at = ring_advance(rg, pos, (unsigned)(j - rg.P)); at.slot += (unsigned)rg.P; }
    const int slot = (int)at.slot;
    // The parity wait below cannot tell "this tile has landed" from "the slot's PREVIOUS tile
    // has not landed yet" (two phases apart).  The previous tile belongs to another warp, and
    // bulk copies complete out of order, so first wait until this tile has been issued into
    // the slot: from then on the barrier's pending phase is this tile's.
    while (rg.tag[slot] != at.seq + 1u) { }
    if (rg.acc) {
        const long long t0 = clock64();
        mbar_wait(&rg.full[slot], at.par);
        *rg.acc += (unsigned long long)(clock64() - t0);
    } else {
        mbar_wait(&rg.full[slot], at.par);
    }
    const int* rp = rg.rp(slot);
    const int base = rp[0] & ~3;
    const int ks = rp[lane] - base, ke = rp[lane + 1] - base;
    const double* sv = rg.vals(slot);
    const int* sc = rg.cols(slot);
    const int trips = __reduce_max_sync(0xffffffffu, (ke - ks + U - 1) / U);
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    if (trips == 0 && !pinned) {
        __syncwarp();
        if (lane == 0) mbar_arrive(&rg.empty[slot]);
    }
    for (int t = 0; t < trips; ++t) {
        const int k = ks + t * U;
        int c[U];
        double v[U], xv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const bool ok = k + u < ke;
            const int kk = ok ? k + u : 0;
            const int cc = sc[kk];
            const double vv = sv[kk];
            c[u] = ok ? cc : 0;
            v[u] = ok ? vv : 0.0;
        }
        if (t == trips - 1 && !pinned) {
            __syncwarp();                  // every lane has its last entries in registers
            if (lane == 0) mbar_arrive(&rg.empty[slot]);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) xv[u] = ld_global_f64(x + c[u]);
        if constexpr (FOLD) {
            double rg_[U];
#pragma unroll
            for (int u = 0; u < U; ++u) rg_[u] = ld_global_f64(r + c[u]);
#pragma unroll
            for (int u = 0; u < U; ++u) xv[u] = fma(beta, xv[u], rg_[u]);
        }
#pragma unroll
        for (int u = 0; u < U; u += 3) {
            a0 = fma(v[u], xv[u], a0);
            a1 = fma(v[u + 1], xv[u + 1], a1);
            a2 = fma(v[u + 2], xv[u + 2], a2);
        }
    }
    return (a0 + a1) + a2;
}

// ---------------------------------------------------------------- reductions

// Sum of one value per consumer thread over the CTA, fixed order.  Valid in warp 0.
template <int W>
__device__ __forceinline__ double block_sum_w(double v, double* red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    consumer_sync<W>();                    // red may still be read from a previous call
    if (lane == 0) red[warp] = v;
    consumer_sync<W>();
    if (warp == 0) {
        v = lane < W ? red[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

// Fixed-order sum of G per-CTA partials from global memory (graph / stepwise kernels);
// every consumer thread gets the value.  Same order as grid_allreduce below.
template <int W>
__device__ __forceinline__ double sum_partials_w(const double* part, int G, double* red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    consumer_sync<W>();
    if (warp == 0) {
        double s = 0.0;
        for (int j = lane; j < G; j += 32) s += __ldcg(part + j);
        s = warp_sum(s);
        if (lane == 0) red[kRedTot] = s;
    }
    consumer_sync<W>();
    return red[kRedTot];
}

// ---------------------------------------------------------------- grid all-reduce == grid barrier
//
// Persistent kernel only (all CTAs co-resident, cooperative launch).  Push, then poll your
// own inbox: CTA c owns an inbox of 3 buffers x kBarVals values x G slots.  At barrier
// number `count` (buffer b = count mod 3) warp 0 of every CTA stores the CTA's NV block
// sums into slot c of EVERY CTA's inbox (lane l serves the destinations l, l + 32, ...),
// then polls its own inbox until none of its G slots holds the idle pattern.  Nobody polls
// a line another SM polls, so the round trip is one store latency plus one load latency.
// Every CTA adds the G values in the same fixed order (the order of sum_partials_w), so
// all CTAs hold bitwise the same totals: alpha and beta never exist in memory.
//
// Slot recycling: after its poll a CTA rewrites the slots it just read with the idle
// pattern (all-ones: a NaN no arithmetic produces, published NaNs are canonicalised, and
// cudaMemset(0xFF) arms the inboxes).  Source j writes that buffer again three all-reduces
// later.  FENCED all-reduces (the prologue's; with the fold, the one after K2 that publishes
// r and p) carry a gpu-scope fence before the push (release of everything the CTA wrote)
// and one after the reset (acquire; it also invalidates this SM's L1).  The others carry
// only their payload.  Between an all-reduce and the third one after it there is always
// either a fenced one or the counter barrier after K3 (grid_barrier_counter, fenced on both
// sides in every CTA), which is what orders a reset before the next write into the slot:
// reset -> my fence -> my later push or arrival -> j observes it -> j's fence -> j's write.
constexpr unsigned long long kIdle = 0xFFFFFFFFFFFFFFFFULL;
constexpr int kInboxStride = 3 * kBarVals * kBarGrid;     // u64 per CTA inbox

__device__ __forceinline__ void st_relaxed_u64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long publishable(double v) {
    return (v != v) ? 0x7FF8000000000000ULL : (unsigned long long)__double_as_longlong(v);
}

template <int W, int NV, bool FENCED>
__device__ __forceinline__ void grid_allreduce(const Params& P, double* red, unsigned& count,
                                               int cta, int G, double (&v)[NV],
                                               unsigned long long* dbg = nullptr) {
    static_assert(NV >= 1 && NV <= kBarVals && W <= 32, "slot layout");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double w[NV];
    if (dbg) dbg[0] = clock64();
#pragma unroll
    for (int i = 0; i < NV; ++i) w[i] = warp_sum(v[i]);
    consumer_sync<W>();
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) red[i * 32 + warp] = w[i];
    }
    consumer_sync<W>();                    // also: all phase stores of the CTA happen-before the fence below
    if (warp == 0) {
        if (dbg) dbg[1] = clock64();
#pragma unroll
        for (int i = 0; i < NV; ++i) w[i] = warp_sum(lane < W ? red[i * 32 + lane] : 0.0);
        unsigned long long* base = reinterpret_cast<unsigned long long*>(P.bslots);
        const unsigned b = count % 3u;
        if (FENCED) asm volatile("fence.acq_rel.gpu;" ::: "memory");
        // push into every inbox
#pragma unroll
        for (int m = 0; m < kBarM; ++m) {
            const int j = lane + 32 * m;
            if (j < G) {
                unsigned long long* dst = base + (size_t)j * kInboxStride + (b * kBarVals) * kBarGrid + cta;
#pragma unroll
                for (int i = 0; i < NV; ++i) st_relaxed_u64(dst + i * kBarGrid, publishable(w[i]));
            }
        }
        if (dbg) dbg[2] = clock64();
        // poll my inbox
        unsigned long long* mine = base + (size_t)cta * kInboxStride + (b * kBarVals) * kBarGrid;
        unsigned long long u[NV][kBarM];
        bool ready;
        do {
            ready = true;
#pragma unroll
            for (int i = 0; i < NV; ++i)
#pragma unroll
                for (int m = 0; m < kBarM; ++m) {
                    const int j = lane + 32 * m;
                    u[i][m] = (j < G) ? ld_relaxed_u64(mine + i * kBarGrid + j) : 0ULL;
                    ready = ready && (u[i][m] != kIdle);
                }
        } while (!ready);
        if (dbg) dbg[3] = clock64();
        // recycle the slots just read
#pragma unroll
        for (int i = 0; i < NV; ++i)
#pragma unroll
            for (int m = 0; m < kBarM; ++m) {
                const int j = lane + 32 * m;
                if (j < G) st_relaxed_u64(mine + i * kBarGrid + j, kIdle);
            }
        __syncwarp();
        if (dbg) dbg[4] = clock64();
        if (FENCED) asm volatile("fence.acq_rel.gpu;" ::: "memory");
        if (dbg) dbg[5] = clock64();
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            double tot = 0.0;
#pragma unroll
            for (int m = 0; m < kBarM; ++m)
                if (lane + 32 * m < G) tot += __longlong_as_double((long long)u[i][m]);
            tot = warp_sum(tot);
            if (lane == 0) red[kRedTot + i] = tot;
        }
    }
    if (dbg) dbg[6] = clock64();
    consumer_sync<W>();
    if (dbg) dbg[7] = clock64();
#pragma unroll
    for (int i = 0; i < NV; ++i) v[i] = red[kRedTot + i];
    ++count;
}

// Pure grid barrier (no payload), used after K3 to publish p: one relaxed atomic add on a
// counter and one poller per CTA, between a release fence and an acquire fence (the latter
// also invalidates this SM's L1 so the K1 gathers see the new p).  About half the latency of
// the push/poll exchange (1.5 k against 3.1 k cycles stand-alone): 148 atomics on one line
// and 148 polling threads instead of 21 904 stores.  The counter (Scal::bar) is zeroed per
// solve and only grows; `nbar` counts this CTA's arrivals.
template <int W>
__device__ __forceinline__ void grid_barrier_counter(const Params& P, unsigned long long& nbar, int G,
                                                     unsigned long long* dbg = nullptr) {
    if (dbg) dbg[0] = clock64();
    consumer_sync<W>();                    // all phase stores of the CTA happen-before the fence below
    if (threadIdx.x == 0) {
        if (dbg) dbg[1] = clock64();
        unsigned long long* ctr = &P.scal->bar;
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
        asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;" :: "l"(ctr), "l"(1ULL) : "memory");
        if (dbg) dbg[2] = clock64();
        const unsigned long long target = (++nbar) * (unsigned long long)G;
        while (ld_relaxed_u64(ctr) < target) { }
        if (dbg) dbg[3] = clock64();
        if (dbg) dbg[4] = dbg[3];
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
        if (dbg) { dbg[5] = clock64(); dbg[6] = dbg[5]; }
    }
    consumer_sync<W>();
    if (dbg) dbg[7] = clock64();
}

// ---------------------------------------------------------------- vector phases, vectors in global memory
// Same thread <-> row map as K1: warp w, trip k -> tile j = w + k W, row = 32 (tb + j) + lane.
// VU tiles are in flight per thread; the accumulation order is the tile order.

__device__ __forceinline__ double ld_cs_f64(const double* p) {
    double v;   // x is touched once per iteration: streaming (evict-first) accesses
    asm volatile("ld.global.cs.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_cs_f64(double* p, double v) {
    asm volatile("st.global.cs.f64 [%0], %1;" :: "l"(p), "d"(v) : "memory");
}

// Optional L2 residency hints for the big-system path (option "l2_hints", off by default).  q
// is written by K1 and read by K2 a whole matrix sweep (1.3 GB at config 4) later: its stores
// ask the L2 to keep the lines (evict_last), the one read in K2 releases them (evict_first).
// Measured at config 4: K2 55.6 k instead of 59.9 k cycles, but K3 28.2 k instead of 16.2 k
// (r and p lose their place in the L2): a net loss, hence off.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void st_hint_f64(double* p, double v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" :: "l"(p), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ double ld_hint_f64(const double* p, uint64_t pol) {
    double v;
    asm volatile("ld.global.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol) : "memory");
    return v;
}

constexpr int kVU = 4;

// Prologue: r = b - q (q = A x0); p = r (or D^-1 r); partials of r.r, b.b, r.z.
template <int W, bool PRE>
__device__ __forceinline__ void phase_init_tiles(const Params& P, long long tb, int Tc,
                                                 double& arr, double& abb, double& arz) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j0 = warp; j0 < Tc; j0 += W * kVU) {
        double bv[kVU], qv[kVU], dv[kVU];
        long long idx[kVU];
#pragma unroll
        for (int u = 0; u < kVU; ++u) {
            const int j = j0 + u * W;
            const long long i = (tb + j) * kTileRows + lane;
            idx[u] = (j < Tc && i < P.n) ? i : -1;
            if (idx[u] >= 0) { bv[u] = P.b[i]; qv[u] = ld_global_f64(P.q + i); if (PRE) dv[u] = P.dinv[i]; }
        }
#pragma unroll
        for (int u = 0; u < kVU; ++u) {
            if (idx[u] < 0) continue;
            const double ri = bv[u] - qv[u];
            P.r[idx[u]] = ri;
            abb = fma(bv[u], bv[u], abb);
            arr = fma(ri, ri, arr);
            if (PRE) {
                const double zi = dv[u] * ri;
                P.p[idx[u]] = zi;
                arz = fma(ri, zi, arz);
            } else {
                P.p[idx[u]] = ri;
            }
        }
    }
}

// K2: x += alpha p ; r -= alpha q ; partial r.r (and r.z with Jacobi).
template <int W, bool PRE>
__device__ __forceinline__ void phase_xr_tiles(const Params& P, double alpha, long long tb, int Tc,
                                               double& arr, double& arz) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const double na = -alpha;
    for (int j0 = warp; j0 < Tc; j0 += W * kVU) {
        double xv[kVU], rv[kVU], pv[kVU], qv[kVU], dv[kVU];
        long long idx[kVU];
#pragma unroll
        for (int u = 0; u < kVU; ++u) {
            const int j = j0 + u * W;
            const long long i = (tb + j) * kTileRows + lane;
            idx[u] = (j < Tc && i < P.n) ? i : -1;
            if (idx[u] >= 0) {
                xv[u] = ld_cs_f64(P.x + i); rv[u] = ld_global_f64(P.r + i);
                pv[u] = ld_global_f64(P.p + i);
                qv[u] = P.l2_stream ? ld_hint_f64(P.q + i, l2_policy_evict_first()) : ld_global_f64(P.q + i);
                if (PRE) dv[u] = P.dinv[i];
            }
        }
#pragma unroll
        for (int u = 0; u < kVU; ++u) {
            if (idx[u] < 0) continue;
            const double xi = fma(alpha, pv[u], xv[u]);
            const double ri = fma(na, qv[u], rv[u]);
            st_cs_f64(P.x + idx[u], xi);
            P.r[idx[u]] = ri;
            arr = fma(ri, ri, arr);
            if (PRE) arz = fma(ri, dv[u] * ri, arz);
        }
    }
}

// K3: p = r + beta p   (Jacobi: p = D^-1 r + beta p).
template <int W, bool PRE>
__device__ __forceinline__ void phase_p_tiles(const Params& P, double beta, long long tb, int Tc) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int VU = 2 * kVU;
    for (int j0 = warp; j0 < Tc; j0 += W * VU) {
        double rv[VU], pv[VU], dv[VU];
        long long idx[VU];
#pragma unroll
        for (int u = 0; u < VU; ++u) {
            const int j = j0 + u * W;
            const long long i = (tb + j) * kTileRows + lane;
            idx[u] = (j < Tc && i < P.n) ? i : -1;
            if (idx[u] >= 0) {
                rv[u] = ld_global_f64(P.r + i); pv[u] = ld_global_f64(P.p + i);
                if (PRE) dv[u] = P.dinv[i];
            }
        }
#pragma unroll
        for (int u = 0; u < VU; ++u) {
            if (idx[u] < 0) continue;
            const double zi = PRE ? rv[u] * dv[u] : rv[u];
            P.p[idx[u]] = fma(beta, pv[u], zi);
        }
    }
}

template <int W>
__device__ __forceinline__ void phase_zero_x_tiles(const Params& P, long long tb, int Tc) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j = warp; j < Tc; j += W) {
        const long long i = (tb + j) * kTileRows + lane;
        if (i < P.n) P.x[i] = 0.0;
    }
}

// K1 with vectors in global memory: y = A x over this CTA's tiles, for the pass that starts at
// ring position `pos`; returns this thread's partial of x.y when DOT.
template <int W, int U, bool DOT>
__device__ __forceinline__ double phase_spmv_tiles(const Params& P, const Ring& rg, const double* x,
                                                   double* y, long long tb, int Tc, RingPos pos) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double dot = 0.0;
    for (int j = warp; j < Tc; j += W) {
        const long long row = (tb + j) * kTileRows + lane;
        double xr = 0.0;
        if (DOT && row < P.n) xr = ld_global_f64(x + row);      // early: off the critical path
        const double acc = consume_tile<U>(rg, x, pos, j, lane);
        if (row < P.n) {
            if (P.l2_stream & 2) st_hint_f64(y + row, acc, l2_policy_evict_last());
            else y[row] = acc;
            if (DOT) dot = fma(acc, xr, dot);
        }
    }
    return dot;
}

}  // namespace cgs
