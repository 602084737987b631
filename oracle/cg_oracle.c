/*
 * cg_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, sequential fp64 implementation of what the hot path computes,
 * written from the paper and shared with nothing under paper_1107_0538_b200/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.
 *
 * What the paper fixes:
 *   PAPER.md:34  "The conjugate gradient (CG) method [5] ... systems that are
 *                symmetric or Hermitian positive definite ... Compressed
 *                Sparse Row (CSR) format having N=132651 and NNZ=3442951"
 *   PAPER.md:44  "Tasks, such as DGEMV(sparse), are repetitive"; "The CGLoop
 *                is a 132651 loop"; "A continue-condition ... so the loop can
 *                stop before running all iterations"; "scalar operations run
 *                on CPU processor, and repetitive operations run on GPU"
 *   PAPER.md:48  "four double-precision implementation versions"
 *   PAPER.md:60  "TOL=1E-10"
 *   PAPER.md:76  ref [5] Golub & Van Loan is the only source of the algorithm
 * Fig. 1 (the CG task graph) is a dangling image link, so the
 * iteration is textbook unpreconditioned Hestenes-Stiefel CG, with the readings
 * of SURVEY.md section 8(c) (listed in DESIGN.md "Readings"):
 *   - stop when ||r_k||_2 <= rtol * ||b||_2 (recurrence residual, Matlab pcg
 *     convention), tested before the first iteration and after every update;
 *   - an iteration = one SpMV inside the loop; hist[j] = ||r_j||_2, j = 0..k;
 *   - b = 0 returns x = 0, k = 0, converged;
 *   - breakdown (p.Ap <= 0 or not finite) returns status 2.
 *
 * Arithmetic rules: every sum is a left-to-right fp64 accumulation in index
 * order; build with -O2 -ffp-contract=off (no FMA contraction, no fast-math),
 * so each function is one well-defined function of its inputs.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_inputs.py): brute-force dense
 * mat-vec, row sums A*1 = 0.01*1, closed-form eigenpairs of the 7-point
 * Laplacian, finite termination on m eigenvectors, the hand-worked 2x2 case
 * in tests/golden/, dense Cholesky, recurrence-vs-true residual, A-orthogonality,
 * Lanczos/Ritz values, the kappa convergence bound and A-norm monotonicity.
 * Parity unpinned: the iteration COUNTS at the five configs (nothing external
 * fixes them; the paper's 116/117 belong to its own, missing matrix).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* y = A x.  Rows in order, entries of a row in stored order (PAPER.md:44
 * "DGEMV(sparse)"; CSR per PAPER.md:34). */
void oracle_spmv(int64_t n, const int32_t *rowptr, const int32_t *colind,
                 const double *vals, const double *x, double *y)
{
    for (int64_t i = 0; i < n; ++i) {
        double s = 0.0;
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
            s = s + vals[k] * x[colind[k]];
        y[i] = s;
    }
}

/* s = sum_i a_i b_i, left to right. */
double oracle_dot(int64_t n, const double *a, const double *b)
{
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i)
        s = s + a[i] * b[i];
    return s;
}

/* Diagnostics used only to attribute error: the same sums in
 * long double (x86 80-bit), and the SpMV error denominator (|A||x|)_i. */
void oracle_spmv_ld(int64_t n, const int32_t *rowptr, const int32_t *colind,
                    const double *vals, const double *x, double *y)
{
    for (int64_t i = 0; i < n; ++i) {
        long double s = 0.0L;
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
            s = s + (long double)vals[k] * (long double)x[colind[k]];
        y[i] = (double)s;
    }
}

double oracle_dot_ld(int64_t n, const double *a, const double *b)
{
    long double s = 0.0L;
    for (int64_t i = 0; i < n; ++i)
        s = s + (long double)a[i] * (long double)b[i];
    return (double)s;
}

void oracle_absrow(int64_t n, const int32_t *rowptr, const int32_t *colind,
                   const double *vals, const double *x, double *y)
{
    for (int64_t i = 0; i < n; ++i) {
        double s = 0.0;
        for (int64_t k = rowptr[i]; k < rowptr[i + 1]; ++k)
            s = s + fabs(vals[k]) * fabs(x[colind[k]]);
        y[i] = s;
    }
}

/*
 * Conjugate gradient, step by step in the order of SURVEY.md 8(c) / Golub &
 * Van Loan.  With dinv != NULL the same loop is the Jacobi-
 * preconditioned variant (z = D^-1 r, hinted by the
 * paper's baseline being Matlab's *p*cg); dinv == NULL is the
 * paper's path (M = I) and performs exactly the unpreconditioned arithmetic.
 *
 *   x      in: x0, out: x_k            hist   out: ||r_j||_2, j = 0..k (maxit+1)
 *   alpha_out, beta_out (may be NULL)  length maxit
 *   P_out, R_out, X_out (may be NULL)  keep x n row-major: p_j, r_j, x_j, j < keep
 * Returns status 0 converged, 1 maxit reached, 2 breakdown, -1 bad argument.
 */
int oracle_cg(int64_t n, const int32_t *rowptr, const int32_t *colind,
              const double *vals, const double *dinv, const double *b, double *x,
              double rtol, int64_t maxit, double *hist,
              int64_t *iters_out, double *resnorm_out,
              double *alpha_out, double *beta_out,
              double *P_out, double *R_out, double *X_out, int64_t keep)
{
    if (n <= 0 || maxit < 0 || !(rtol >= 0.0) || !hist) return -1;
    double *r = (double *)malloc(sizeof(double) * (size_t)n);
    double *p = (double *)malloc(sizeof(double) * (size_t)n);
    double *q = (double *)malloc(sizeof(double) * (size_t)n);
    double *z = dinv ? (double *)malloc(sizeof(double) * (size_t)n) : NULL;
    int status = 1;
    int64_t k = 0;

    double bb = oracle_dot(n, b, b);
    if (bb == 0.0) {                              /* reading 9: b = 0 */
        memset(x, 0, sizeof(double) * (size_t)n);
        hist[0] = 0.0;
        *iters_out = 0; *resnorm_out = 0.0;
        free(r); free(p); free(q); free(z);
        return 0;
    }
    /* r = b - A x0 */
    oracle_spmv(n, rowptr, colind, vals, x, q);
    for (int64_t i = 0; i < n; ++i) r[i] = b[i] - q[i];
    double rr = oracle_dot(n, r, r);              /* ||r||^2: the stopping norm */
    double rz;                                     /* r.z: equals rr when M = I */
    if (dinv) {
        for (int64_t i = 0; i < n; ++i) z[i] = dinv[i] * r[i];
        for (int64_t i = 0; i < n; ++i) p[i] = z[i];
        rz = oracle_dot(n, r, z);
    } else {
        for (int64_t i = 0; i < n; ++i) p[i] = r[i];
        rz = rr;
    }
    hist[0] = sqrt(rr);
    const double thresh = rtol * sqrt(bb);

    while (1) {
        if (k < keep) {
            if (P_out) memcpy(P_out + k * n, p, sizeof(double) * (size_t)n);
            if (R_out) memcpy(R_out + k * n, r, sizeof(double) * (size_t)n);
            if (X_out) memcpy(X_out + k * n, x, sizeof(double) * (size_t)n);
        }
        if (sqrt(rr) <= thresh) { status = 0; break; }   /* continue-condition */
        if (k >= maxit) { status = 1; break; }
        oracle_spmv(n, rowptr, colind, vals, p, q);      /* q = A p */
        double pq = oracle_dot(n, p, q);
        if (!(pq > 0.0) || !isfinite(pq)) { status = 2; break; }
        double alpha = rz / pq;
        for (int64_t i = 0; i < n; ++i) x[i] = x[i] + alpha * p[i];
        for (int64_t i = 0; i < n; ++i) r[i] = r[i] - alpha * q[i];
        double rr_new = oracle_dot(n, r, r);
        double rz_new;
        if (dinv) {
            for (int64_t i = 0; i < n; ++i) z[i] = dinv[i] * r[i];
            rz_new = oracle_dot(n, r, z);
        } else {
            rz_new = rr_new;
        }
        double beta = rz_new / rz;
        if (dinv) for (int64_t i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];
        else      for (int64_t i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
        if (alpha_out) alpha_out[k] = alpha;
        if (beta_out) beta_out[k] = beta;
        rr = rr_new; rz = rz_new;
        k = k + 1;
        hist[k] = sqrt(rr);
    }
    *iters_out = k;
    *resnorm_out = sqrt(rr);
    free(r); free(p); free(q); free(z);
    return status;
}
