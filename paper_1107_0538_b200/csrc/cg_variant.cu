// cg_variant.cu -- instantiates the kernels of ONE streamed kernel shape and ONE slot format.
// Compiled six times (-DCG_SHAPE=0|1|2 -DCG_CMP=0|1) and once with -DCG_SHORT (the short-row kernels of
// shape 2) in parallel by build.py; nothing here but the table of entry points (cg_variants.h).  The
// kernels themselves are in cg_stream_kernels.cuh.
#include "cg_stream_kernels.cuh"
#include "cg_variants.h"

#if defined(CG_SHORT)

void cg_fill_fns_short(StreamFns& f) {
    f.short_persistent[0] = (const void*)cgs::ks_persistent<16, 0, 9, true, 4, false, false, true>;
    f.short_persistent[1] = (const void*)cgs::ks_persistent<16, 0, 9, true, 4, true, false, true>;
    f.short_cg1 = (const void*)cgs::ks_persistent_cg1<16, 0, 9, true, 4, true>;
    f.short_pipe = (const void*)cgs::ks_persistent_pipe<16, 0, 9, true, 4, true>;
}

#else

#if !defined(CG_SHAPE) || !defined(CG_CMP)
#error "compile with -DCG_SHAPE=0|1|2 -DCG_CMP=0|1, or -DCG_SHORT"
#endif

namespace {

template <int W, int NP, int U, bool GF, bool CMP> void fill(StreamFns& f) {
    constexpr int c = CMP ? 1 : 0;
    f.W = W; f.NP = NP; f.U = U;
    if constexpr (!CMP) {                  // kernels that never touch a slot: once per shape
        f.init_residual = (const void*)cgs::ks_init_residual<W, NP>;
        f.init_scalars = (const void*)cgs::ks_init_scalars<W, NP>;
        f.k2 = (const void*)cgs::ks2_update_xr<W, NP>;
        f.k3 = (const void*)cgs::ks3_update_p<W, NP>;
    }
    f.spmv[c] = (const void*)cgs::ks_spmv<W, NP, U, GF, CMP>;
    f.spmv_checked[c] = (const void*)cgs::ks_spmv<W, NP, U, GF, CMP, true>;
    f.init_spmv[c] = (const void*)cgs::ks_init_spmv<W, NP, U, GF, CMP>;
    f.k1[c] = (const void*)cgs::ks1_spmv_dot<W, NP, U, GF, CMP>;
    f.persistent[c][kR0]       = (const void*)cgs::ks_persistent<W, NP, U, GF, 0, false, false, CMP>;
    f.persistent[c][kR0Jacobi] = (const void*)cgs::ks_persistent<W, NP, U, GF, 0, true, false, CMP>;
    f.persistent[c][kR2]       = (const void*)cgs::ks_persistent<W, NP, U, GF, 2, false, false, CMP>;
    f.persistent[c][kR2Jacobi] = (const void*)cgs::ks_persistent<W, NP, U, GF, 2, true, false, CMP>;
    f.persistent[c][kR2Fold]   = (const void*)cgs::ks_persistent<W, NP, U, GF, 2, false, true, CMP>;
    f.persistent[c][kR4]       = (const void*)cgs::ks_persistent<W, NP, U, GF, 4, false, false, CMP>;
    f.persistent[c][kR4Jacobi] = (const void*)cgs::ks_persistent<W, NP, U, GF, 4, true, false, CMP>;
    f.persistent[c][kR4Fold]   = (const void*)cgs::ks_persistent<W, NP, U, GF, 4, false, true, CMP>;
    f.cg1[c][0] = (const void*)cgs::ks_persistent_cg1<W, NP, U, GF, 2, CMP>;
    f.cg1[c][1] = (const void*)cgs::ks_persistent_cg1<W, NP, U, GF, 4, CMP>;
    if constexpr (NP != 4) {               // the pipelined loop exists for shapes 1 and 2 only (build time)
        f.pipe[c][0] = (const void*)cgs::ks_persistent_pipe<W, NP, U, GF, 2, CMP>;
        f.pipe[c][1] = (const void*)cgs::ks_persistent_pipe<W, NP, U, GF, 4, CMP>;
    } else {
        f.pipe[c][0] = f.pipe[c][1] = nullptr;
    }
}

}  // namespace

#define CG_CAT3(a, b, c) a##b##_##c
#define CG_FILL_NAME(s, c) CG_CAT3(cg_fill_fns_, s, c)

void CG_FILL_NAME(CG_SHAPE, CG_CMP)(StreamFns& f) {
#if CG_SHAPE == 0
    fill<12, 4, 9, false, CG_CMP != 0>(f);
#elif CG_SHAPE == 1
    fill<11, 5, 9, false, CG_CMP != 0>(f);
#else
    fill<16, 0, 27, true, CG_CMP != 0>(f);
#endif
}

#endif  // CG_SHORT
