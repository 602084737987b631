/*
 * cg.h -- C ABI of libcg_b200: fp64 conjugate gradient on a CSR SPD matrix,
 * hand-written CUDA for sm_100a (one B200, no sharding, no collectives).
 *
 * The operation is the case study of arxiv 1107.0538 ("The conjugate
 * gradient (CG) method ... The matrix is stored in Compressed Sparse Row (CSR)
 * format having N=132651 and NNZ=3442951"; "DGEMV(sparse)", the CGLoop
 * with its continue-condition; PAPER.md:48 double precision; PAPER.md:60 TOL=1E-10).
 * Unlike the paper, which runs "scalar operations ... on CPU processor"
 * and loses its multi-GPU speed-up to "extra data transfers among cpu and devices"
 * (PAPER.md:50), alpha, beta and the stop test stay on the device: cg_solve makes
 * exactly one host synchronisation, at the end.
 *
 * Conventions:
 *  - d_* pointers are DEVICE memory owned by the caller (e.g. torch tensors),
 *    16-byte aligned; h_* pointers are HOST memory.  `cuda_stream` is a
 *    cudaStream_t passed as void* (0 = the legacy default stream).
 *  - The handle BORROWS rowptr/colind/vals and the workspace: they must outlive
 *    it and must not be written while a call is in flight.  The library never
 *    allocates or frees device memory (only the small host struct, 64 bytes of
 *    pinned host memory and, in graph mode, a CUDA graph).
 *  - CSR: 0-based int32 indices, rowptr[0] = 0, rowptr[n] = nnz, non-decreasing.
 *    Columns of a row need not be sorted or unique (duplicates add).
 *  - Return codes: 0 success / converged.  Positive = soft outcome: of cg_solve
 *    1 maxit reached, 2 breakdown (p.Ap <= 0 or not finite: A is not SPD); of
 *    cg_compress_index 3 (the index was left uncompressed); of cg_reorder 4 (the matrix
 *    was left in the caller's numbering).
 *    Negative = error: -1 invalid argument, -2 CUDA error (text via
 *    cg_strerror), -3 device not supported (needs compute capability 10.x),
 *    -4 device watchdog (a spin wait inside a solve ran out of its budget: a
 *    protocol error or a lost copy; the results of that call are void, the device
 *    is left usable), -5 out of host memory, -6 size beyond what cg_dot_static's fixed
 *    scratch can serve.
 *    Nothing is printed, thrown or aborted across this boundary.
 *  - The sparsity structure (rowptr, colind) is fixed for the life of the handle;
 *    vals may be rewritten between calls (then cg_set_option(h, "values_changed", 1)
 *    so that cg_solve_jacobi extracts the diagonal again).
 *  - One handle per stream; concurrent calls on one handle are undefined.
 */
#ifndef CG_B200_H
#define CG_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cg_handle cg_handle;

#define CG_OK             0
#define CG_MAXIT          1
#define CG_BREAKDOWN      2
#define CG_NOTCOMPRESSED  3
#define CG_NOTREORDERED   4
#define CG_EINVAL        -1
#define CG_ECUDA         -2
#define CG_EUNSUPPORTED  -3
#define CG_ETIMEOUT      -4
#define CG_ENOMEM        -5
#define CG_ETOOBIG       -6

/* Bytes of device workspace cg_create needs for an n-row system: the vectors
 * r, p, q, one spare and D^-1 (each n doubles, 256-byte aligned), a padded copy of rowptr
 * (n + 41 ints), the per-CTA reduction partials, a 16 MB reserve inside which the grid
 * all-reduce inboxes (1.8 MB) are placed, and the device-resident scalar state. */
size_t cg_workspace_bytes(int64_t n);

/* Bind a handle to a CSR matrix already resident on the device.
 * d_rowptr int32[n+1], d_colind int32[nnz], d_vals double[nnz].
 * d_workspace: >= cg_workspace_bytes(n) bytes, 256-byte aligned.
 * Reads the n+1 row pointers once (two stream-0 kernels: tile statistics, padded copy) to
 * pick the SpMV variant and the ring geometry, and times the grid synchronisation with the
 * all-reduce inboxes at 40 places of their reserve (which L2 slices their lines map to
 * changes its cost by a few per cent; ~30 ms; results never depend on the place).
 * Errors: CG_EINVAL on NULL/misaligned pointers, n <= 0, nnz < 0, n or nnz
 * >= 2^31, workspace too small; CG_EUNSUPPORTED off sm_100; CG_ECUDA. */
int cg_create(cg_handle** out, int64_t n, int64_t nnz,
              const int32_t* d_rowptr, const int32_t* d_colind, const double* d_vals,
              void* d_workspace, size_t workspace_bytes);

/* Optional compressed column index (the matrix comes "from
 * a FEM model", so col - row takes few distinct values).  When the matrix has at most 256
 * distinct offsets col - row, cg_compress_index builds, in caller-owned device memory, one
 * record per 32-row tile (33 16-bit row starts + one byte per entry naming its offset) and the
 * streamed kernels then move 9 instead of 12 bytes per entry: vals still come from the
 * caller's array, in CSR order, so every result keeps its bits.  At the paper's size this
 * makes each SM's slice of the matrix fit its shared memory for the whole solve.
 * cg_index_bytes: size the buffer needs (0: not worth compressing, e.g. very uneven rows).
 * cg_compress_index: d_index 256-byte aligned, borrowed until cg_destroy or the next call;
 * returns CG_OK (in use from now on), CG_NOTCOMPRESSED (more than 256 offsets: nothing
 * changes) or a negative error.  Synchronises the stream. */
size_t cg_index_bytes(cg_handle* h);
int cg_compress_index(cg_handle* h, void* d_index, size_t index_bytes, void* cuda_stream);

/* Optional renumbering for matrices whose rows arrive in no useful order (the
 * matrix comes from a FEM model of an electrical machine, numbered as the mesh generator left
 * it; BASELINE.json config 3).  When one warp-wide gather of the SpMV touches many 128-byte
 * lines (cg_get_info "lines_per_gather_x100"), K1 is bound by the 32-byte sectors the L2 has to
 * deliver for 8 useful bytes each.  cg_reorder computes a reverse Cuthill-McKee numbering on
 * the host (the pattern is copied there once; set-up work, like cg_create), builds the matrix
 * P A P^T in caller-owned device memory (entries of a row sorted by their new column) and binds
 * an inner handle to it.  From then on cg_solve / cg_solve_jacobi / cg_solve_host gather b and
 * x0 into the new numbering, run the SAME kernels on the renumbered matrix and scatter x back:
 * two small extra launches per solve, iterates equal to the caller's up to the rounding of a
 * different summation order (same parity bands in the tests).  cg_spmv, cg_dot and
 * cg_check_csr keep using the caller's matrix.  Options set later reach both handles;
 * "values_changed" drops the renumbered copy (call cg_reorder again); "reorder" = 0 / 1
 * switches its use off / on.
 * cg_reorder_bytes: size of d_buf (permutation, the renumbered CSR arrays, two vectors, the
 * inner handle's workspace).  cg_reorder: d_buf 256-byte aligned, borrowed until cg_destroy or
 * the next call; returns CG_OK (in use from now on), CG_NOTREORDERED (the new numbering
 * does not cut the lines per gather by at least a third: nothing changes) or a negative
 * error.  Synchronises the stream.
 * cg_rcm_host: the numbering alone, host arrays in, h_perm[new row] = old row out. */
size_t cg_reorder_bytes(int64_t n, int64_t nnz);
int cg_reorder(cg_handle* h, void* d_buf, size_t bytes, void* cuda_stream);
int cg_rcm_host(int64_t n, const int32_t* h_rowptr, const int32_t* h_colind, int32_t* h_perm);

/* Optional structural check of the bound CSR arrays on the device: rowptr[0] = 0,
 * rowptr[n] = nnz, non-decreasing, 0 <= colind < n.  Synchronises the stream.
 * Returns CG_OK or CG_EINVAL.  (Symmetry / definiteness are NOT checked:
 * PAPER.md:34 "should only be applied to" SPD systems; cg_solve reports
 * CG_BREAKDOWN instead.) */
int cg_check_csr(cg_handle* h, void* cuda_stream);

/* y = A x, the paper's "DGEMV(sparse)".  d_x, d_y: double[n],
 * distinct buffers.  Asynchronous on the stream. */
int cg_spmv(cg_handle* h, const double* d_x, double* d_y, void* cuda_stream);

/* *h_result = sum_i a_i b_i (the p.Ap / r.r reductions of the CG loop, which PAPER.md:44
 * counts among the "repetitive operations [that] run on GPU"), with a
 * fixed reduction order: bitwise reproducible run to run.  d_a, d_b: double[n].
 * Synchronises the stream once. */
int cg_dot(cg_handle* h, const double* d_a, const double* d_b,
           double* h_result, void* cuda_stream);

/* The same scalar product for callers that may not allocate (code under CUDA
 * graph capture, serving loops, harnesses that forbid cudaMalloc): no handle, no workspace, and
 * no cudaMalloc / cudaFree / cudaHostAlloc / malloc on its path.  The per-block partial sums
 * live in a fixed 32 KB __device__ array inside the library (held by every GPU that loads the
 * library until the process exits), which bounds the size: n <= cg_dot_static_max_n() =
 * 33 554 432; beyond that CG_ETOOBIG ("cg_dot_static: n exceeds ...").
 * d_a, d_b: device double[n]; d_result: DEVICE double[1], written on the stream.  Asynchronous:
 * nothing synchronises.  Blocks of 8192 elements, fixed-order sums: bitwise reproducible; the
 * grouping differs from cg_dot's, so the two agree to rounding (1e-15 sum|a_i b_i| log2 n).
 * Every call on a device shares the one scratch array: calls that may overlap on the GPU
 * (different streams) race; calls on one stream are ordered.  A call reads only the partials
 * it wrote itself, so nothing has to be cleared between calls.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress; make that
 * call outside stream capture).  Errors: CG_EINVAL (n < 0, NULL), CG_ETOOBIG, CG_ECUDA. */
int cg_dot_static(int64_t n, const double* d_a, const double* d_b, double* d_result, void* cuda_stream);
int64_t cg_dot_static_max_n(void);

/* Solve A x = b by unpreconditioned CG (readings in DESIGN.md):
 *   r = b - A x0; p = r; loop { q = A p; alpha = r.r / p.q; x += alpha p;
 *   r -= alpha q; beta = r'.r' / r.r; p = r + beta p } until
 *   ||r_k||_2 <= rtol ||b||_2 (tested before the first iteration and after
 *   every update) or k = maxit (the paper's CGLoop bound is N).
 * d_b double[n] (not modified); d_x double[n]: x0 on entry, x_k on return.
 * d_hist: device double[maxit+1] or NULL; d_hist[j] = ||r_j||_2 for j = 0..k.
 * *h_iters = k (number of in-loop SpMVs); *h_final_resnorm = ||r_k||_2.
 * b = 0 returns x = 0, k = 0, CG_OK.  Synchronises the stream once, at the end.
 * Returns CG_OK / CG_MAXIT / CG_BREAKDOWN or a negative error. */
int cg_solve(cg_handle* h, const double* d_b, double* d_x,
             double rtol, int64_t maxit, double* d_hist,
             int64_t* h_iters, double* h_final_resnorm, void* cuda_stream);

/* Jacobi-preconditioned variant (the paper's sequential
 * reference is Matlab's *p*cg): z = D^-1 r with D = diag(A) taken
 * from the CSR arrays; alpha = r.z / p.q, beta = r'.z' / r.z, p = z + beta p.
 * The stop test is still on ||r_k||_2.  Same arguments and returns as cg_solve;
 * CG_BREAKDOWN also when a diagonal entry is missing or not positive. */
int cg_solve_jacobi(cg_handle* h, const double* d_b, double* d_x,
                    double rtol, int64_t maxit, double* d_hist,
                    int64_t* h_iters, double* h_final_resnorm, void* cuda_stream);

/* End-to-end entry with HOST buffers: copies h_b and h_x (x0) to the device,
 * runs cg_solve, copies x and hist[0..k] back.  h_b, h_x double[n]; h_hist
 * double[maxit+1] or NULL.  d_scratch: device memory of at least
 * cg_host_scratch_bytes(n, maxit) bytes, 256-byte aligned.  Pinned host
 * buffers make the copies asynchronous; pageable ones also work. */
size_t cg_host_scratch_bytes(int64_t n, int64_t maxit);
int cg_solve_host(cg_handle* h, const double* h_b, double* h_x,
                  double rtol, int64_t maxit, double* h_hist,
                  int64_t* h_iters, double* h_final_resnorm,
                  void* d_scratch, size_t scratch_bytes, void* cuda_stream);

/* Tuning / diagnostics.  Options (name -> value):
 *   "loop"      0 = one cooperative persistent kernel (default)
 *               1 = CUDA graph of {K1, K2, K3} per iteration, replayed in chunks
 *                   with a device-side stop flag (the profilable twin)
 *               2 = plain per-iteration launches, same kernels as 1
 *   "spmv"      0 = auto; 1 = generic: sub-warp per row straight from global memory (any
 *               CSR matrix); 2, 3, 4 = streamed: 32-row tiles in shared-memory slots filled by
 *               bulk-async (TMA) copies, W consumer warps with one lane per row:
 *               2 = 12 consumer + 4 producer warps, 9 entries in flight per lane, slots handed
 *                   back to the producers before the gathers are issued;
 *               3 = 11 + 5, likewise;
 *               4 = 16 consumer warps and no producers (every warp copies its own tiles once),
 *                   27 gathers in flight per lane: only when every CTA's slice of the matrix is
 *                   pinned in shared memory (see "pin").
 *               Auto picks 4 when everything is pinned, else 3 when the matrix is re-streamed
 *               from the L2 every iteration or streams from HBM in compressed form, else 2.
 *               A request that cannot run (a 32-row tile does not fit a ring of 8 slots in the
 *               227 KB of shared memory; 4 without pinning) falls back to 1.
 *   "chunk"     iterations per graph replay in loop mode 1 (even, default 32)
 *   "resident"  1 (default) = the persistent streamed kernel keeps x, r, p, q in registers
 *               when every thread owns <= 4 rows; 0 = always in global memory
 *   "fold"      persistent streamed kernel with vectors in registers, no preconditioner:
 *               1 = fold K3 into the next K1 (every gathered p_j is recomputed on the fly as
 *               fma(beta, p_old_j, r_j) from one 16-byte {p_old, r} pair, the owner's own
 *               expression, so results keep their bits) and synchronise the grid twice
 *               instead of three times per iteration; 0 = off; 2 (default) = on when no row has
 *               more than 9 entries, a CTA gathers <= 500 entries per lane (tiles x mean row
 *               length) and the short-row kernels do not apply
 *   "sync_place" where the all-reduce inboxes sit in their reserve, in steps of 64 KB
 *               (0 .. cg_get_info "sync_places"); cg_create picks it by measurement
 *   "short_rows" 1 (default) = when no row has more than 9 entries (the 7-point Laplacian), every
 *               CTA's slice is pinned and a consumer warp owns several tiles, run the kernels
 *               that keep the gathers of 2-3 tiles in flight per warp instead of one tile's 9
 *               (same operations per row in the same order: same bits); 0 = off
 *   "pin"       1 (default) = when every CTA's slice of the matrix fits the shared memory (up
 *               to 64 tiles per SM) and the matrix would otherwise be re-read from the L2 every
 *               iteration, copy it there once per solve and keep it; 0 = stream everything
 *               every iteration; k >= 2 = pin k tiles per CTA and stream the rest (a mixed
 *               split, kept for tests and measurements)
 *   "algo"      0 (default) = the textbook recurrence of cg_solve above, three grid
 *               synchronisations per iteration.  1 = Chronopoulos-Gear single-reduction CG
 *               (SURVEY.md 8(f) rank 2): w = A r, ONE all-reduce of (r.r, w.r) and one barrier
 *               that publishes r per iteration; same iterates in exact arithmetic, different
 *               rounding (held to the same parity bands in the tests, never the default).
 *               2 = pipelined CG (Ghysels-Vanroose): w = A r, q = A w, ONE counter barrier per
 *               iteration; the partial sums of (r.r, w.r) are published by that barrier and read
 *               back after the SpMV, so the reduction needs no synchronisation of its own.  One
 *               more recurrence than 1 (more rounding); same status as 1.
 *               Both apply to loop 0 with the vectors in registers and no preconditioner (2 also
 *               needs kernel shape 3 or 4); otherwise the textbook path runs (cg_get_info "algo"
 *               tells which).  With 2 the SpMV of the next iteration is started before the stop
 *               test of the current one is known; iters still counts the updates of x.
 *   "compress"  1 (default) = use the compressed index once cg_compress_index has built it;
 *               0 = plain CSR slots
 *   "ring_slots" cap on the ring depth (8..64)
 *   "smem_cap_kb" cap (KB) on the shared memory a STREAMING ring may take; what is left of the
 *               SM's 256 KB array is L1, whose lines hold the outstanding gather misses.
 *               0 (default) = auto: 132 KB when gathers are irregular (> 8 lines per warp-wide
 *               gather), 164 KB when the matrix streams from HBM, else all of it
 *   "lookahead" tiles the producers may prefetch of an iteration the consumers have not
 *               started (default unlimited: the ring is refilled across the grid barriers)
 *   "tpr", "ctas_per_sm"  lanes per row and CTAs per SM of the generic variant
 *   "values_changed" (any value) the caller rewrote vals: cached D^-1 is dropped
 *   "checked"   1 = cg_spmv runs its checked twin: every index it forms (source ranges of the
 *               bulk copies, offsets inside a slot, index codes, gathered columns) is validated
 *               on the device before use and clamped when wrong; the call then synchronises and
 *               returns CG_ECUDA ("... out-of-range indices caught") if any was.  The library's
 *               own memcheck (compute-sanitizer is not available everywhere); default 0
 *   "spin_budget_ms" how long any device-side spin may last before the watchdog trips and
 *               the solve returns CG_ETIMEOUT (default 2000)
 *   "inject_fault" tests only: k > 0 makes producer warp 0 of CTA 0 announce its k-th tile
 *               and never copy it, which must end in CG_ETIMEOUT (default 0)
 * cg_get_info reads back: "loop", "spmv", "grid", "block", "smem", "launches" (kernels
 * launched by the last call), "sms", "tpr", "max_row_len", "max_tile_nnz", "stream_ok",
 * "consumer_warps", "producer_warps", "in_flight", "ring_slots", "pinned_tiles", "slot_bytes",
 * "sync_place", "sync_places", "reordered" (cg_reorder's numbering is in use), "resident_rows", "fold", "short_rows", "algo", "compressed", "index_codes", "from_hbm", "check_errors" (violations
 * counted by the last checked cg_spmv), "lines_per_gather_x100"
 * (cg_create statistic: 128-byte lines one warp-wide gather touches on average, times 100).
 * A name prefixed with "solve_" ("solve_spmv", "solve_ring_slots", ...) is answered by the handle
 * the solves run on: the renumbered one after cg_reorder, this one otherwise.
 * Unknown names return CG_EINVAL. */
int cg_set_option(cg_handle* h, const char* name, int64_t value);
int cg_get_info(cg_handle* h, const char* name, int64_t* value);

/* Read-bandwidth probe used by the bench for the L2 and HBM rooflines ("a
 * read-only streaming microbenchmark over a 40 MB buffer, repeated, on the same box"): reads
 * the `bytes` (>= 4096, 16-byte aligned) at d_buf `reps` times after one warm-up sweep, with
 * 16-byte loads from every SM, and returns bytes * reps / time in *h_gbs (GB/s, CUDA events).
 * A buffer smaller than the L2 measures L2 read bandwidth, a much larger one HBM read
 * bandwidth.  Synchronises the stream. */
int cg_probe_read_bandwidth(cg_handle* h, const void* d_buf, size_t bytes, int reps,
                            double* h_gbs, void* cuda_stream);

/* Grid-synchronisation probe (a profiling aid for DESIGN.md's latency figures): runs `reps`
 * synchronisations of one kind on the solve's own grid (one CTA of 512 threads per SM,
 * cooperative launch) with the very device functions cg_solve uses, and returns the mean cycles
 * per synchronisation over all CTAs in *h_cycles.  kind 0 = counter barrier (no payload; what
 * follows K3), 1 = push/poll all-reduce carrying only its payload (after K1 and K2; every third
 * one is replaced by a counter barrier, as the slot-recycling rule demands, so the figure is the
 * mean of two all-reduces and one barrier), 2 = all-reduce fenced on both sides (prologue, folded
 * loop).  Synchronises the stream.  CG_ETIMEOUT if the watchdog tripped. */
int cg_probe_grid_sync(cg_handle* h, int kind, int reps, double* h_cycles, void* cuda_stream);

/* Phase trace of the persistent loop (loop mode 0), a profiling aid: with a non-NULL
 * d_trace (device uint64[grid * (iters + 1) * 16], grid = cg_get_info "grid"), thread 0 of
 * every CTA stores clock64() at 8 points of each of the first `iters` iterations of later
 * solves: [0] iteration start, [1] K1 done, [2] past all-reduce 1, [3] K2 done, [4] past
 * all-reduce 2, [5] beta known, [6] K3 done, [7] past barrier 3; slots 8-15 detail that
 * barrier.  Layout [cta][iter][slot]; row `iters` of every CTA holds ring statistics
 * ([0] cycles producer warp 0 waited for free slots, [1] its lifetime, [2] tiles it issued,
 * [3] cycles consumer thread 0 waited for data).  NULL or iters = 0 switches it off (the
 * default).  The buffer is borrowed.  With cg_set_option "trace_clock" = 1 the streamed
 * persistent kernels stamp %globaltimer (nanoseconds, one clock for all SMs) instead, which
 * makes the stamps of different CTAs comparable: arrival and release skew at each grid
 * synchronisation. */
int cg_set_trace(cg_handle* h, uint64_t* d_trace, int64_t iters);

/* Frees the host struct (and any CUDA graph).  Device memory is the caller's. */
int cg_destroy(cg_handle* h);

/* Static text for a return code; for CG_ECUDA the last CUDA error string seen
 * by this thread. */
const char* cg_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* CG_B200_H */
