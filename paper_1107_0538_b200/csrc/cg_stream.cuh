// cg_stream.cuh -- the streamed CG path for sm_100a: warp-specialised bulk-async (TMA)
// producers, W consumer warps with one lane per row, grid all-reduce fused with the grid
// barrier, and (for systems small enough) x, r, p, q kept in registers for the whole solve.
//
// What is computed is unchanged ("DGEMV(sparse)" + the CG of
// PAPER.md:76): K1 q = A p with the p.q partials, K2 x += alpha p, r -= alpha q with the r.r
// partials, K3 p = r + beta p, scalars on the device.
//
// Work split.  The matrix is cut into tiles of 32 consecutive rows.  CTA c owns the
// contiguous tiles (cta_tiles below: T/G each, the left-over tiles at the two ends); inside a CTA tile j (0-based) belongs to consumer warp
// j mod W, lane l of that warp owns row 32*tile + l in EVERY phase.  The thread that
// computes q_i is therefore the thread that updates x_i, r_i, p_i, and all per-thread
// partial sums are accumulated in tile order: every loop mode (persistent with vectors in
// registers, persistent with vectors in global memory, graph, stepwise) performs the same
// floating-point operations in the same order and gives bitwise identical results.
//
// K1 data flow.  NP extra warps (the producers) walk the CTA's tiles in order and,
// for each, wait for a free ring slot and issue cp.async.bulk copies (SASS UBLKCP) into it.
// Two slot formats (template flag CMP):
//   plain CSR     the tile's contiguous vals span, its colind span and its 33 row pointers (36
//                 ints from a padded copy of rowptr): 12 B per entry, three copies;
//   compressed    (cg_compress_index) the vals span and ONE index record built at setup: 33
//                 relative row starts (u16) and one byte per entry that names the entry's column
//                 offset col - row in a table of <= 256 distinct offsets: 9 B per entry, two
//                 copies.  Entries keep their CSR order, so both formats give the same bits.
// Consumers wait on the slot's "full" mbarrier, copy their row bounds and entries from shared
// memory into registers, hand the slot back, then gather x through L1/L2.  No consumer ever
// waits on a row-pointer or matrix load from global memory; the only global loads in its loop
// are the x gathers.  In the persistent kernel the producers run ahead into the next
// iteration's tiles (the matrix does not change) while the consumers do K2/K3 and wait at the
// grid barriers, so K1 starts on a full ring.
//
// Alignment of the bulk copies: source, destination and size must be multiples of 16
// bytes.  A tile's span [s, e) is widened to [s & ~A, (e + A) & ~A) with A = 3 (plain: colind
// is the 4-byte array) or A = 1 (compressed: only vals come from the caller's arrays), clamped
// to nnz & ~A; the <= A entries of the whole matrix past that bound are written into the slot
// by the producer with ordinary loads/stores, so nothing outside the caller's arrays is touched.
//
// Every spin in this file is bounded (bounded_spin): after Params::spin_budget cycles the CTA
// raises Scal::abort, stops waiting and leaves the solve at the next collective point; the host
// then returns CG_ETIMEOUT instead of hanging the device.
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
constexpr int kRedTot = 96;          // red[0..95]: per-warp partials (3 values x 32 warps); red[96..98]: totals; red[99]: abort
constexpr int kRecHdr = 80;          // compressed index record: 33 u16 row starts, [33] = s & 1, padded to 80 bytes
constexpr int kMaxCodes = 256;       // distinct column offsets a compressed index can name
constexpr int kOffTabBytes = kMaxCodes * 4;
constexpr int kOffTabSmall = 32;     // with <= 32 codes (the stencils) the shared-memory copy of the table takes 128 bytes

// W consumer warps + NP producer warps per CTA; W + NP is a multiple of 4 so the warps spread
// evenly over the SM's four sub-partitions (their register files bound the registers per thread).
template <int W, int NP> struct Shape {
    static constexpr int kConsumers = W;
    static constexpr int kProducers = NP;
    static constexpr int kConsumerThreads = 32 * W;
    static constexpr int kThreads = 32 * (W + NP);
};

struct Ring {
    unsigned char* slots;
    uint64_t* full;
    uint64_t* empty;
    double* red;                      // 104 doubles of reduction scratch (see kRedTot)
    volatile int* ctl;                // [0] stop flag, [1] passes consumed (low), [2] (high), [3] passes started,
                                      // [4] a spin of this CTA ran out of budget (watchdog)
    volatile unsigned* tag;           // per slot: 1 + number (mod 2^32) of the tile last issued into it
    const int* offtab;                // compressed index: column offset per code (shared-memory copy)
    int S, slot_bytes, cap;
    int P, Q;                         // pinned slots [0, P) and streaming slots [P, P + Q), P + Q <= S
    int rec_words;                    // compressed index: 32-bit code words per lane in a record
    int n;                            // rows of the matrix
    int ncodes;                       // entries of the offset table in shared memory
    long long budget;                 // cycles a spin may last
    Scal* scal;
    unsigned long long* acc;          // optional: cycles this thread waited on full barriers (trace)
    __device__ __forceinline__ double* vals(int slot) const {
        return reinterpret_cast<double*>(slots + (size_t)slot * slot_bytes);
    }
    __device__ __forceinline__ int* cols(int slot) const {             // plain slots
        return reinterpret_cast<int*>(slots + (size_t)slot * slot_bytes + (size_t)cap * 8);
    }
    __device__ __forceinline__ int* rp(int slot) const {
        return reinterpret_cast<int*>(slots + (size_t)slot * slot_bytes + (size_t)cap * 12);
    }
    __device__ __forceinline__ unsigned char* rec(int slot) const {    // compressed slots
        return slots + (size_t)slot * slot_bytes + (size_t)cap * 8;
    }
};

__device__ __forceinline__ Ring ring_view(const Params& P, unsigned char* dyn) {
    Ring rg;
    rg.S = P.slots; rg.slot_bytes = P.slot_bytes; rg.cap = P.cap; rg.acc = nullptr;
    rg.P = P.pinned; rg.Q = P.stream_slots; rg.rec_words = (P.rec_stride - kRecHdr) / 128; rg.n = (int)P.n; rg.ncodes = P.ncodes_smem;
    rg.budget = P.spin_budget; rg.scal = P.scal;
    rg.slots = dyn;
    unsigned char* tail = dyn + (size_t)P.slots * P.slot_bytes;
    rg.full = reinterpret_cast<uint64_t*>(tail);
    rg.empty = rg.full + kMaxSlots;
    rg.red = reinterpret_cast<double*>(rg.empty + kMaxSlots);
    rg.ctl = reinterpret_cast<volatile int*>(rg.red + 104);
    rg.tag = reinterpret_cast<volatile unsigned*>(rg.ctl + 8);       // kMaxSlots entries
    rg.offtab = reinterpret_cast<const int*>(tail + kSmemTail);      // kOffTabBytes, only with a compressed index
    return rg;
}

// Called by every thread of the CTA (producer warps included) before anything else.
__device__ __forceinline__ void ring_init(const Params& P, const Ring& rg) {
    if ((int)threadIdx.x < rg.S) {
        mbar_init(&rg.full[threadIdx.x], 1);
        mbar_init(&rg.empty[threadIdx.x], 1);
        rg.tag[threadIdx.x] = 0u;
    }
    if (threadIdx.x < 8) rg.ctl[threadIdx.x] = 0;
    if (P.cmp && (int)threadIdx.x < P.ncodes_smem) const_cast<int*>(rg.offtab)[threadIdx.x] = P.idx_off[threadIdx.x];
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
}

// Barrier among the consumer warps only (the producers never join it).
template <int W> __device__ __forceinline__ void consumer_sync() {
    asm volatile("bar.sync 1, %0;" :: "n"(32 * W) : "memory");
}

// The CTA's contiguous tile range: floor(T / G) tiles each, and the T mod G tiles that are left over go to the
// CTAs at the two ENDS of the matrix (half to the first ones, half to the last ones).  On a grid in natural ordering
// those own the boundary planes, whose rows are shorter: at config 2 (4146 tiles = 148 x 28 + 2) the two 29-tile CTAs
// used to sit mid-matrix, where every row is full, and the grid waited for them at every all-reduce (K1 7.5 k
// against 7.0 k cycles).  For any other matrix the choice is as good as any.
__device__ __forceinline__ long long cta_tile_begin(long long ntiles, int cta, int G) {
    const long long q = ntiles / G, r = ntiles % G;
    const long long head = (r + 1) / 2, tail = r / 2;         // CTAs [0, head) and [G - tail, G) own q + 1 tiles
    const long long c = cta;
    return c * q + (c < head ? c : head) + (c > G - tail ? c - (G - tail) : 0);
}
__device__ __forceinline__ void cta_tiles(const Params& P, int cta, int G, long long& tb, int& Tc) {
    const long long ntiles = (P.n + kTileRows - 1) / kTileRows;
    tb = cta_tile_begin(ntiles, cta, G);
    Tc = (int)(cta_tile_begin(ntiles, cta + 1, G) - tb);
}

// ---------------------------------------------------------------- watchdog

// Spin until pred() holds.  Gives up (returns false) once the spin has lasted rg.budget cycles
// or another warp of this CTA has given up: it then raises the CTA's flag (ctl[4]) and the
// solve's (Scal::abort).  The clock is read once per 1024 polls, so the happy path costs nothing.
template <class Pred>
__device__ __forceinline__ bool bounded_spin(const Ring& rg, Pred pred) {
    if (pred()) return true;
    const long long t0 = clock64();
    for (unsigned n = 1;; ++n) {
        if (pred()) return true;
        if ((n & 0x3ffu) == 0u && (rg.ctl[4] != 0 || clock64() - t0 > rg.budget)) {
            rg.ctl[4] = 1;
            *reinterpret_cast<volatile int*>(&rg.scal->abort) = 1;
            return false;
        }
    }
}
__device__ __forceinline__ bool mbar_wait_bounded(const Ring& rg, uint64_t* bar, uint32_t parity) {
    return bounded_spin(rg, [&] { return mbar_try_wait(bar, parity); });
}

// ---------------------------------------------------------------- producer

// CHK (option "checked", cg_spmv only): every index is validated before it is used -- source
// ranges of the bulk copies against the arrays' lengths, slot offsets against the slot's size,
// codes against the table, gathered columns against n -- violations are counted in
// Scal::chk_errors and the access is clamped, so a checked run never touches memory it should not.
// This is the library's own stand-in for compute-sanitizer's memcheck (closed on this pool).
__device__ __forceinline__ void chk_fail(const Ring& rg) { atomicAdd(&rg.scal->chk_errors, 1); }

template <bool CMP, bool CHK = false>
__device__ __forceinline__ void producer_issue(const Params& P, const Ring& rg, int slot, long long t,
                                               int s, int e, uint64_t policy, unsigned tag, bool drop) {
    constexpr int A = CMP ? 1 : 3;                     // span alignment in entries (16 bytes of the narrowest array)
    if constexpr (CHK) {
        const long long ntiles = (P.n + kTileRows - 1) / kTileRows;
        const int lo = s & ~A;
        const bool bad = t < 0 || t >= ntiles || s < 0 || e < s || (long long)e > P.nnz || e - lo > rg.cap ||
                         slot < 0 || slot >= rg.S;
        if (bad) {                                     // announce nothing: complete the phase with a plain arrival
            chk_fail(rg);
            rg.tag[slot < 0 || slot >= rg.S ? 0 : slot] = tag;
            mbar_arrive(&rg.full[slot < 0 || slot >= rg.S ? 0 : slot]);
            return;
        }
    }
    const int s4 = s & ~A;
    const int lim = (int)(P.nnz & ~(long long)A);     // last entry reachable by bulk copies
    int e4 = (e + A) & ~A;
    if (e4 > lim) e4 = lim;
    const int cnt = e4 > s4 ? e4 - s4 : 0;            // multiple of A + 1
    double* sv = rg.vals(slot);
    if (e > lim) {                                    // the matrix's last <= A entries, by hand
        for (int k = (lim > s4 ? lim : s4); k < e; ++k) {
            sv[k - s4] = ld_stream_f64(P.vals + k);
            if (!CMP) rg.cols(slot)[k - s4] = ld_stream_s32(P.colind + k);
        }
    }
    uint64_t* bar = &rg.full[slot];
    rg.tag[slot] = tag;                               // before the arrive below (release): see consume_tile
    const uint32_t meta = CMP ? (uint32_t)P.rec_stride : (uint32_t)kRpInts * 4u;
    mbar_expect_tx(bar, (uint32_t)cnt * (CMP ? 8u : 12u) + meta);
    if (drop) return;                                 // fault injection (option "inject_fault"): the copies never come
    if (cnt > 0) {
        if (P.l2_stream) {
            bulk_g2s(sv, P.vals + s4, (uint32_t)cnt * 8u, bar, policy);
            if (!CMP) bulk_g2s(rg.cols(slot), P.colind + s4, (uint32_t)cnt * 4u, bar, policy);
        } else {
            bulk_g2s_plain(sv, P.vals + s4, (uint32_t)cnt * 8u, bar);
            if (!CMP) bulk_g2s_plain(rg.cols(slot), P.colind + s4, (uint32_t)cnt * 4u, bar);
        }
    }
    if (CMP) {
        const unsigned char* src = P.idx_rec + (size_t)t * (size_t)P.rec_stride;
        if (P.l2_stream) bulk_g2s(rg.rec(slot), src, meta, bar, policy);
        else             bulk_g2s_plain(rg.rec(slot), src, meta, bar);
    } else {
        bulk_g2s_plain(rg.rp(slot), P.rp_pad + t * kTileRows, meta, bar);
    }
}

// Pinned and streamed tiles.  The first P tiles of a CTA are PINNED: tile j < P is copied into
// slot j once, in the first pass, and stays there for the whole solve (no L2 traffic, no
// shared-memory write, no producer work for it in later iterations).  The other Ts = Tc - P
// tiles of a pass are STREAMED through the Q slots [P, P + Q): streamed tile number seq
// (counted over all passes) uses slot P + seq mod Q.  The host pins everything (P >= Tc) when
// the CTA's whole slice fits the ring and nothing otherwise; a mixed split (option "pin" >= 2)
// exists for tests and measurements.
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
// passes they have started).  Its waits end through the stop flag (ctl[0], raised by the
// consumers at the end of a persistent solve) or the CTA's watchdog flag (ctl[4]).
template <bool CMP, bool CHK = false>
__device__ __forceinline__ void producer_loop(const Params& P, const Ring& rg, long long tb, int Tc,
                                              long long passes, int q, int NP) {
    const int lane = threadIdx.x & 31;
    const uint64_t policy = l2_policy_evict_first();
    if (Tc <= 0) return;
    const int Pn = rg.P < Tc ? rg.P : Tc;                  // my CTA's pinned tiles: [0, Pn)
    const int Ts = Tc - Pn;                                 // streamed tiles per pass
    const int Q = rg.Q;
    // fault injection (tests): producer warp 0 of CTA 0 announces its `inject_fault`-th tile and never copies it
    const int fault_at = (P.inject_fault > 0 && blockIdx.x == 0 && q == 0) ? P.inject_fault : 0;
    int issued = 0;
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
            ++issued;
            if (lane == 0) producer_issue<CMP, CHK>(P, rg, j, tb + j, si, ei, policy, (unsigned)j + 1u, issued == fault_at);
        }
    }
    if (Ts <= 0 || Q <= 0) return;
    unsigned long long seq = (unsigned long long)q;        // next streamed tile number I issue
    long long pass = 0;
    int j = q;                                              // = seq - pass * Ts, index among the streamed tiles
    while (j >= Ts) { j -= Ts; ++pass; }
    unsigned slot = (unsigned)q, par = 0;                   // = seq mod Q, (seq / Q) & 1
    constexpr int B = 32;                                   // tile bounds are fetched 32 at a time, one per lane
    if (!cached) {                                          // bounds of my first batch
        const int jl = (int)(((long long)j + (long long)lane * NP) % Ts);
        s = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows);
        e = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows + kTileRows);
    }
    bool stopped = false;
    unsigned long long t_wait = 0;
    const long long t_begin = clock64();
    const bool timing = P.trace != nullptr;
    while (pass < passes && !stopped) {
        int s2 = 0, e2 = 0;
        if (!cached) {                     // bounds of the batch AFTER this one
            const int jl = (int)(((long long)j + (long long)(B + lane) * NP) % Ts);
            s2 = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows);
            e2 = ld_stream_s32(P.rp_pad + (tb + Pn + jl) * kTileRows + kTileRows);
        }
        for (int l = 0; l < B && pass < passes; ++l) {
            int ok = 1;
            if (lane == 0) {
                const long long t0 = timing ? clock64() : 0;
                if (passes > 1 && j >= P.lookahead) {
                    while ((long long)rg.ctl[3] <= pass) { if (rg.ctl[0] | rg.ctl[4]) { ok = 0; break; } }
                }
                while (ok && !mbar_try_wait(&rg.empty[Pn + slot], par ^ 1u)) {
                    if (rg.ctl[0] | rg.ctl[4]) ok = 0;
                }
                if (timing) t_wait += (unsigned long long)(clock64() - t0);
            }
            ok = __shfl_sync(0xffffffffu, ok, 0);
            if (!ok) { stopped = true; break; }
            const int src = cached ? Pn + j : l;
            const int si = __shfl_sync(0xffffffffu, s, src);
            const int ei = __shfl_sync(0xffffffffu, e, src);
            ++issued;
            if (lane == 0) producer_issue<CMP, CHK>(P, rg, Pn + (int)slot, tb + Pn + j, si, ei, policy, (unsigned)seq + 1u,
                                                    issued == fault_at);
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
    if (stopped && rg.ctl[4] == 0) {
        // Drain: my copies for tiles nobody will consume must land before the CTA exits.  The
        // consumers finished `done` whole passes, i.e. the streamed tiles below done * Ts.
        const unsigned long long done = (((unsigned long long)(unsigned)rg.ctl[2] << 32) | (unsigned)rg.ctl[1])
                                        * (unsigned long long)Ts;
        unsigned long long w = done + (((unsigned long long)q + (unsigned long long)NP
                                        - done % (unsigned long long)NP) % (unsigned long long)NP);
        for (; w < seq; w += (unsigned long long)NP)
            if (!mbar_wait_bounded(rg, &rg.full[Pn + (int)(w % (unsigned)Q)], (uint32_t)((w / (unsigned)Q) & 1ULL))) break;
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

__device__ __forceinline__ double2 ld_global_f64x2(const double2* p) {
    double2 v;
    asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

// The trip of a tile whose rows all have <= UU entries, compressed index, gather-first: UU gathers are
// issued back to back, the values are read from the slot while they fly, then the DFMAs run in CSR order
// into three accumulators.  The record pads short rows with the code of offset 0, so every padding
// gather reads x[row] (a valid address) and only the DFMA is predicated: ~10 instead of ~22
// instructions per entry -- the pinned kernel is bound by instruction issue and by the shared-memory
// datapath (ncu: 21 k warp instructions per SM and iteration through 4 schedulers in ~8 k cycles).
// sw: this lane's code words (word g at sw[32 g]); sr: the row's first value; len: its length.
template <int UU, bool CHK>
__device__ __forceinline__ void trip_issue(const Ring& rg, const double* x, const unsigned* sw, int gmax, int row,
                                           double (&xv)[UU]) {
    constexpr int NW = (UU + 3) / 4;
    unsigned cw[NW];
#pragma unroll
    for (int g = 0; g < NW; ++g) cw[g] = sw[32 * (g < gmax ? g : gmax)];
#pragma unroll
    for (int u = 0; u < UU; ++u) {
        unsigned code = __byte_perm(cw[u >> 2], 0u, 0x4440u | (unsigned)(u & 3));
        if constexpr (CHK) { if ((int)code >= rg.ncodes) { chk_fail(rg); code = 0; } }
        int col = row + rg.offtab[code];
        if constexpr (CHK) { if (col < 0 || col >= rg.n) { chk_fail(rg); col = 0; } }
        xv[u] = ld_global_f64(x + col);
    }
}
template <int UU>
__device__ __forceinline__ double trip_finish(const double* sr, int len, const double (&xv)[UU]) {
    static_assert(UU % 3 == 0, "three accumulators");
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
#pragma unroll
    for (int u = 0; u < UU; u += 3) {
        const double v0 = sr[u], v1 = sr[u + 1], v2 = sr[u + 2];
        if (u < len)     a0 = fma(v0, xv[u], a0);
        if (u + 1 < len) a1 = fma(v1, xv[u + 1], a1);
        if (u + 2 < len) a2 = fma(v2, xv[u + 2], a2);
    }
    return (a0 + a1) + a2;
}
template <int UU, bool CHK>
__device__ __forceinline__ double streamlined_trip(const Ring& rg, const double* x, const unsigned* sw, int gmax,
                                                   const double* sr, int len, int row) {
    double xv[UU];
    trip_issue<UU, CHK>(rg, x, sw, gmax, row, xv);
    return trip_finish<UU>(sr, len, xv);
}

// Short rows (every row of the tile has <= 9 entries: the 7-point Laplacian), tiles pinned: one tile's trip
// keeps only 9 gathers in flight and a warp that owns several tiles would pay one exposed L2 round trip per
// tile.  short_batch issues the gathers of NB <= 3 tiles (27 in flight, as a 27-point tile has) before it
// finishes any of them.  Per row the operations and their order are those of streamlined_trip<9>: same bits.
// Only for tiles that have landed and were checked by tiles_are_short (their "full" barrier is not waited
// on again: a pinned slot has one phase for the whole launch).
template <int NB, int W>
__device__ __forceinline__ void short_batch(const Ring& rg, const double* x, int warp, int kk0, int lane,
                                            long long tb, double* out) {
    // no branch in here: a gather result that is defined on one path only is merged through local memory,
    // and the store that does it waits for the gather (measured: the batch then runs slower than tile by tile)
    double xv[NB][9];
    const int row0 = (int)(tb * kTileRows) + lane;
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const int j = warp + (kk0 + b) * W;
        trip_issue<9, false>(rg, x, reinterpret_cast<const unsigned*>(rg.rec(j) + kRecHdr) + lane, rg.rec_words - 1,
                             row0 + j * kTileRows, xv[b]);
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const int j = warp + (kk0 + b) * W;
        const unsigned short* hd = reinterpret_cast<const unsigned short*>(rg.rec(j));
        const int ks = hd[lane], ke = hd[lane + 1];
        out[kk0 + b] = trip_finish<9>(rg.vals(j) + hd[33] + ks, ke - ks, xv[b]);
    }
}

// True (in every lane) when all tiles of this warp are pinned, complete (not the ragged last tile) and have
// only rows of <= 9 entries.  Call after a pass over the tiles (the slots' contents must have landed).
template <int W, int R>
__device__ __forceinline__ bool tiles_are_short(const Ring& rg, int warp, int lane, long long tb, int Tc) {
    bool ok = rg.P >= Tc;
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        if (ok && j < Tc) {
            const unsigned short* hd = reinterpret_cast<const unsigned short*>(rg.rec(j));
            const int tmax = __reduce_max_sync(0xffffffffu, (int)hd[lane + 1] - (int)hd[lane]);
            ok = tmax <= 9 && (tb + j) * kTileRows + (kTileRows - 1) < rg.n;
        }
    }
    return ok;
}

// One tile: wait for its slot, y_row = sum_k a_k x[col_k] for this lane's row.  U entries are
// in flight per lane and trip: their column indices and values are read from shared memory,
// then the U gathers are issued, then the FMAs go into three independent accumulators
// (27 = 3 x 9 for the stencil rows).  The trip count is made warp-uniform so that the slot
// can be handed back to the producer as soon as the LAST trip has copied its entries into
// registers -- before the gathers, which are the long-latency part: with U >= the row
// length a slot is held for a few hundred cycles only and nearly the whole ring is in
// flight.  Padding entries (k >= ke) use value 0 and column 0.
//
// CMP: the slot holds the compressed index record: row bounds are u16 relative to the tile,
// the codes of lane l's entries 4 g .. 4 g + 3 are the bytes of the 32-bit word [g * 32 + l]
// (transposed and packed at setup: one conflict-free load fetches four codes) and an entry's
// column is row + offtab[code].
//
// FOLD: the gathered operand is not stored anywhere yet: it is p_new[c] = fma(beta, p_old[c],
// r[c]), the very expression K3 evaluates for row c, recomputed here by every thread that
// needs it from the pair {p_old[c], r[c]} (one 16-byte gather; K2 stored r there).  Same
// operation, same operands, same bits as the owner's own update; it saves the third grid
// synchronisation of an iteration.  `x` then points at the double2 pairs.
template <int U, bool FOLD, bool CMP, bool GF, bool CHK = false>
__device__ __forceinline__ double consume_tile(const Ring& rg, const double* x, RingPos pos, int j,
                                               int lane, int row, double beta = 0.0) {
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
    bool ok = bounded_spin(rg, [&] { return rg.tag[slot] == at.seq + 1u; });
    if (rg.acc) {
        const long long t0 = clock64();
        ok = ok && mbar_wait_bounded(rg, &rg.full[slot], at.par);
        *rg.acc += (unsigned long long)(clock64() - t0);
    } else {
        ok = ok && mbar_wait_bounded(rg, &rg.full[slot], at.par);
    }
    if (!__all_sync(0xffffffffu, ok)) return 0.0;      // watchdog: the slot's contents are not to be trusted
    int ks, ke;
    const double* sv = rg.vals(slot);
    const int* sc = nullptr;
    const unsigned* sw = nullptr;
    int gmax = 0;
    if constexpr (CMP) {
        const unsigned short* hd = reinterpret_cast<const unsigned short*>(rg.rec(slot));
        ks = hd[lane]; ke = hd[lane + 1];
        sv += hd[33];                                  // the vals span starts at s & ~1
        sw = reinterpret_cast<const unsigned*>(rg.rec(slot) + kRecHdr) + lane;     // word g of this lane at sw[32 g]
        gmax = rg.rec_words - 1;
    } else {
        const int* rp = rg.rp(slot);
        const int base = rp[0] & ~3;
        ks = rp[lane] - base; ke = rp[lane + 1] - base;
        sc = rg.cols(slot);
    }
    if constexpr (CHK) {
        // row bounds inside the slot's value area (the streamlined trip also reads up to U values past a
        // short row's end, unpredicated: those must still lie inside the slot)
        const int shift = CMP ? (int)(sv - rg.vals(slot)) : 0;
        const int room = (rg.slot_bytes / 8) - shift;
        if (ks < 0 || ke < ks || ke + shift > rg.cap || ks + U > room) { chk_fail(rg); ks = 0; ke = 0; }
    }
    const int tmax = __reduce_max_sync(0xffffffffu, ke - ks);      // longest row of the tile (warp-uniform)
    const int trips = (tmax + U - 1) / U;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
    if constexpr (CMP && GF && !FOLD) {
        // Streamlined trip for the common case: every row of the tile fits one trip and the tile is not
        // the ragged last one (streamlined_trip below).  Its length follows the tile's longest row in steps
        // of 9 entries: a tile of 7-point rows issues 9 gathers, not 27, and the 18-entry rows of a boundary
        // plane (whose values sit 18 doubles apart: two-way bank conflicts) read 18 values, not 27.
        if (trips == 1 && row - lane + (kTileRows - 1) < rg.n) {
            double acc;
            if (U > 18 && tmax > 18)     acc = streamlined_trip<(U > 18 ? U : 9), CHK>(rg, x, sw, gmax, sv + ks, ke - ks, row);
            else if (U > 9 && tmax > 9)  acc = streamlined_trip<(U > 9 ? 18 : 9), CHK>(rg, x, sw, gmax, sv + ks, ke - ks, row);
            else                         acc = streamlined_trip<9, CHK>(rg, x, sw, gmax, sv + ks, ke - ks, row);
            if (!pinned) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&rg.empty[slot]);
            }
            return acc;
        }
    }
    if (trips == 0 && !pinned) {
        __syncwarp();
        if (lane == 0) mbar_arrive(&rg.empty[slot]);
    }
    for (int t = 0; t < trips; ++t) {
        const int k = ks + t * U;
        int c[U];
        double v[GF ? 1 : U], xv[U];
        // compressed index: the trip's U codes sit in (U + 6) / 4 consecutive 32-bit words of this
        // lane (four codes per word); entry u is byte (t U mod 4) + (u mod 4) of the word pair
        // {u / 4, u / 4 + 1}: one PRMT each, and 4 (U = 9) or 8 (U = 27) conflict-free loads per trip
        constexpr int NW = CMP ? (U + 6) / 4 : 1;
        unsigned cw[NW];
        unsigned cbase = 0;
        if constexpr (CMP) {
            const int g0 = (t * U) >> 2;
            cbase = (unsigned)(t * U) & 3u;
#pragma unroll
            for (int g = 0; g < NW; ++g) cw[g] = sw[32 * (g0 + g < gmax ? g0 + g : gmax)];
        }
        // a trip in which every lane still has U entries needs no per-entry predicates (a third of the
        // instructions): the interior tiles of the stencils, 57 % of config 4's
        const bool whole = !GF && !CHK && __all_sync(0xffffffffu, ke - k >= U);
        if (whole) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if constexpr (CMP) {
                    const unsigned code = __byte_perm(cw[u >> 2], cw[(u >> 2) + 1 < NW ? (u >> 2) + 1 : NW - 1], cbase + (u & 3)) & 0xffu;
                    c[u] = row + rg.offtab[code];
                } else {
                    c[u] = sc[k + u];
                }
                if constexpr (!GF) v[u] = sv[k + u];
            }
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const bool in = k + u < ke;
                const int kk = in ? k + u : 0;
                int cc;
                if constexpr (CMP) {
                    unsigned code = __byte_perm(cw[u >> 2], cw[(u >> 2) + 1 < NW ? (u >> 2) + 1 : NW - 1], cbase + (u & 3)) & 0xffu;
                    if constexpr (CHK) { if (in && (int)code >= rg.ncodes) { chk_fail(rg); code = 0; } }
                    cc = row + rg.offtab[in ? code : 0];
                } else {
                    cc = sc[kk];
                }
                if constexpr (CHK) { if (in && (cc < 0 || cc >= rg.n)) { chk_fail(rg); cc = 0; } }
                c[u] = in ? cc : 0;
                if constexpr (!GF) { const double vv = sv[kk]; v[u] = in ? vv : 0.0; }
            }
        }
        if (!GF && t == trips - 1 && !pinned) {
            __syncwarp();                  // every lane has its last entries in registers
            if (lane == 0) mbar_arrive(&rg.empty[slot]);
        }
        if constexpr (FOLD) {
            const double2* xp = reinterpret_cast<const double2*>(x);
            double2 pr[U];
#pragma unroll
            for (int u = 0; u < U; ++u) pr[u] = ld_global_f64x2(xp + c[u]);
#pragma unroll
            for (int u = 0; u < U; ++u) xv[u] = fma(beta, pr[u].x, pr[u].y);
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) xv[u] = ld_global_f64(x + c[u]);
        }
        if constexpr (GF) {
            // gather-first: the values are read from the slot while the gathers are in flight,
            // which keeps U of them in flight with U + few registers; the slot is held meanwhile
#pragma unroll
            for (int u = 0; u < U; u += 3) {
                const double v0 = k + u < ke ? sv[k + u] : 0.0;
                const double v1 = k + u + 1 < ke ? sv[k + u + 1] : 0.0;
                const double v2 = k + u + 2 < ke ? sv[k + u + 2] : 0.0;
                a0 = fma(v0, xv[u], a0);
                a1 = fma(v1, xv[u + 1], a1);
                a2 = fma(v2, xv[u + 2], a2);
            }
            if (t == trips - 1 && !pinned) {
                __syncwarp();
                if (lane == 0) mbar_arrive(&rg.empty[slot]);
            }
        } else {
#pragma unroll
            for (int u = 0; u < U; u += 3) {
                a0 = fma(v[u], xv[u], a0);
                a1 = fma(v[u + 1], xv[u + 1], a1);
                a2 = fma(v[u + 2], xv[u + 2], a2);
            }
        }
    }
    return (a0 + a1) + a2;
}

// Shapes without producer warps (NP = 0; only when every tile is pinned): consumer warp w copies
// its own tiles w, w + W, ... into their slots, once per kernel.
template <int W, bool CMP, bool CHK = false>
__device__ __forceinline__ void consumers_pin_tiles(const Params& P, const Ring& rg, long long tb, int Tc) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane != 0) return;
    const int Pn = rg.P < Tc ? rg.P : Tc;
    const uint64_t policy = l2_policy_evict_first();
    for (int j = warp; j < Pn; j += W) {
        const int s = ld_stream_s32(P.rp_pad + (tb + j) * kTileRows);
        const int e = ld_stream_s32(P.rp_pad + (tb + j) * kTileRows + kTileRows);
        producer_issue<CMP, CHK>(P, rg, j, tb + j, s, e, policy, (unsigned)j + 1u,
                                 P.inject_fault > 0 && blockIdx.x == 0 && j == P.inject_fault - 1);
    }
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
// later.  FENCED all-reduces carry a gpu-scope fence before the push (release of everything
// the CTA wrote) and one after the reset (acquire; it also invalidates this SM's L1).  The
// others carry only their payload.  Between an all-reduce and the third one after it there
// must be a fenced one or the counter barrier (grid_barrier_counter, fenced on both sides in
// every CTA), which is what orders a reset before the next write into the slot:
// reset -> my fence -> my later push or arrival -> j observes it -> j's fence -> j's write.
// The ONE place that fixes an iteration's sequence of synchronisations, and with it this
// invariant, is SyncPlan in cg_stream_kernels.cuh (checked there by a static_assert).
//
// Returns true when the watchdog tripped in this CTA (in any consumer warp before the call, or
// in the poll): the value is the same in every consumer thread of the CTA.
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
__device__ __forceinline__ bool grid_allreduce(const Params& P, const Ring& rg, unsigned& count,
                                               int cta, int G, double (&v)[NV],
                                               unsigned long long* dbg = nullptr) {
    static_assert(NV >= 1 && NV <= kBarVals && W <= 32, "slot layout");
    double* red = rg.red;
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
        bool ready, dead = false;
        unsigned rounds = 0;
        long long t0 = 0;
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
            if (!ready && (++rounds & 0xffu) == 0u) {          // watchdog, once per 256 poll rounds
                if (rounds == 0x100u) t0 = clock64();
                else if (rg.ctl[4] != 0 || clock64() - t0 > rg.budget) { dead = true; break; }
            }
        } while (!ready);
        dead = __any_sync(0xffffffffu, dead);
        if (dbg) dbg[3] = clock64();
        if (dead) {
            rg.ctl[4] = 1;
            *reinterpret_cast<volatile int*>(&P.scal->abort) = 1;
        } else {
            // recycle the slots just read
#pragma unroll
            for (int i = 0; i < NV; ++i)
#pragma unroll
                for (int m = 0; m < kBarM; ++m) {
                    const int j = lane + 32 * m;
                    if (j < G) st_relaxed_u64(mine + i * kBarGrid + j, kIdle);
                }
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
        if (lane == 0) red[kRedTot + kBarVals] = rg.ctl[4] != 0 ? 1.0 : 0.0;
    }
    if (dbg) dbg[6] = clock64();
    consumer_sync<W>();
    if (dbg) dbg[7] = clock64();
#pragma unroll
    for (int i = 0; i < NV; ++i) v[i] = red[kRedTot + i];
    ++count;
    return red[kRedTot + kBarVals] != 0.0;
}

// Pure grid barrier (no payload), used after K3 to publish p: one relaxed atomic add on a
// counter and one poller per CTA, after a release fence, polled with ACQUIRE loads (which
// also invalidates this SM's L1 so the K1 gathers see the new p).  About half the latency of
// the push/poll exchange (1.5 k against 3.1 k cycles stand-alone): 148 atomics on one line
// and 148 polling threads instead of 21 904 stores.  The counter (Scal::bar) is zeroed per
// solve and only grows; `nbar` counts this CTA's arrivals.  Returns true when the watchdog
// tripped (same value in every consumer thread).
template <int W>
__device__ __forceinline__ bool grid_barrier_counter(const Params& P, const Ring& rg, unsigned long long& nbar, int G,
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
        // the poll is an ACQUIRE load: it pairs with the other CTAs' {release fence, relaxed add} and invalidates
        // this SM's L1 (so the K1 gathers see the new p) without the full fence that used to follow the poll
        // (MEMBAR.ALL.GPU: ~750 cycles on the critical path of every iteration)
        bounded_spin(rg, [&] { return ld_acquire_u64(ctr) >= target; });
        if (dbg) dbg[3] = clock64();
        if (dbg) dbg[4] = dbg[3];
        if (dbg) { dbg[5] = clock64(); dbg[6] = dbg[5]; }
        rg.red[kRedTot + kBarVals] = rg.ctl[4] != 0 ? 1.0 : 0.0;
    }
    consumer_sync<W>();
    if (dbg) dbg[7] = clock64();
    return rg.red[kRedTot + kBarVals] != 0.0;
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

// q is read once in K2 a whole matrix sweep after K1 wrote it: when the matrix streams from HBM
// that read carries an evict-first hint so the lines leave the L2 to p and r.
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
template <int W, int U, bool DOT, bool CMP, bool GF, bool CHK = false>
__device__ __forceinline__ double phase_spmv_tiles(const Params& P, const Ring& rg, const double* x,
                                                   double* y, long long tb, int Tc, RingPos pos) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double dot = 0.0;
    for (int j = warp; j < Tc; j += W) {
        const long long row = (tb + j) * kTileRows + lane;
        double xr = 0.0;
        if (DOT && row < P.n) xr = ld_global_f64(x + row);      // early: off the critical path
        const double acc = consume_tile<U, false, CMP, GF, CHK>(rg, x, pos, j, lane, (int)row);
        if (row < P.n) {
            y[row] = acc;
            if (DOT) dot = fma(acc, xr, dot);
        }
    }
    return dot;
}

// The kernels instantiated gather-first with U = 9 are the short-row kernels (cg_variant.cu, CG_SHORT).
template <int U, bool GF, bool CMP, int R> struct ShortBatchKernel { static constexpr bool value = GF && CMP && U == 9 && R > 1; };

// K1 of a consumer thread that keeps its rows in registers: out[kk] = (A x)_row of tile warp + kk W
// (untouched when the warp has no such tile).  batch (warp-uniform, from tiles_are_short) selects short_batch.
template <int W, int U, int R, bool CMP, bool GF>
__device__ __forceinline__ void k1_resident_tiles(const Ring& rg, const double* x, RingPos pos, int warp, int lane,
                                                  long long tb, int Tc, bool batch, double (&out)[R]) {
    if constexpr (ShortBatchKernel<U, GF, CMP, R>::value) {
        if (batch) {
            // the warp's tiles are warp, warp + W, ...: cnt of them (warp-uniform); one branch-free batch per case
            const int cnt = Tc > warp ? (Tc - warp + W - 1) / W : 0;
            if (R >= 4 && cnt >= 4) {
                short_batch<2, W>(rg, x, warp, 0, lane, tb, out);
                short_batch<2, W>(rg, x, warp, 2, lane, tb, out);
            } else if (R >= 3 && cnt == 3) {
                short_batch<3, W>(rg, x, warp, 0, lane, tb, out);
            } else if (cnt == 2) {
                short_batch<2, W>(rg, x, warp, 0, lane, tb, out);
            } else if (cnt == 1) {
                short_batch<1, W>(rg, x, warp, 0, lane, tb, out);
            }
            return;
        }
    }
#pragma unroll
    for (int kk = 0; kk < R; ++kk) {
        const int j = warp + kk * W;
        if (j < Tc) out[kk] = consume_tile<U, false, CMP, GF>(rg, x, pos, j, lane, (int)((tb + j) * kTileRows + lane));
    }
}

}  // namespace cgs
