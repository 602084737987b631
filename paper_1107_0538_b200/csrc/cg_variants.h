// cg_variants.h -- the table of kernel entry points of one streamed kernel shape, filled by the
// translation units of cg_variant.cu (one per shape and slot format) and read by cg_api.cu.
#pragma once

// Streamed shapes: W consumer warps, NP producer warps, U entries in flight per lane, GF = gather-first
// consumer (cg_stream.cuh).  "spmv" option value = index + 2.  Every kernel that touches the slots exists
// for both slot formats ([cmp]: 0 plain CSR, 1 compressed index).
//   shape 0: 12 + 4 warps, U 9      shape 1: 11 + 5 warps, U 9      shape 2: 16 + 0 warps, U 27, gather-first
constexpr int kNumShapes = 3;
enum PersistentKind { kR0, kR0Jacobi, kR2, kR2Jacobi, kR2Fold, kR4, kR4Jacobi, kR4Fold, kNumPersistent };
struct StreamFns {
    int W, NP, U;
    const void* spmv[2];
    const void* spmv_checked[2];           // option "checked"
    const void* init_spmv[2]; const void* init_residual; const void* init_scalars;
    const void* k1[2]; const void* k2; const void* k3;
    const void* persistent[2][kNumPersistent];
    const void* cg1[2][2];                 // option "algo" = 1 (Chronopoulos-Gear): [cmp][R == 4]
    const void* pipe[2][2];                // option "algo" = 2 (pipelined CG); null for shape 0
    // Short-row kernels (shape 2, compressed index, no row longer than 9 entries, 4 rows per thread): U = 9 and
    // several tiles' gathers in flight per warp (cg_stream.cuh: short_batch).  Null for the other shapes.
    const void* short_persistent[2];       // [Jacobi]
    const void* short_cg1;
    const void* short_pipe;
};

void cg_fill_fns_0_0(StreamFns&); void cg_fill_fns_0_1(StreamFns&);
void cg_fill_fns_1_0(StreamFns&); void cg_fill_fns_1_1(StreamFns&);
void cg_fill_fns_2_0(StreamFns&); void cg_fill_fns_2_1(StreamFns&);
void cg_fill_fns_short(StreamFns&);      // cg_variant.cu compiled with -DCG_SHORT
