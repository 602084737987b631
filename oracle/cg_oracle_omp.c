/*
 * cg_oracle_omp.c -- TEST / BASELINE INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * The loops of cg_oracle.c (same algorithm, same order of steps)
 * with row-parallel OpenMP on all host cores: the "CPU baseline on all cores" of SURVEY.md
 * section 8(d).  It is NOT the parity reference (its reductions are summed per thread, so
 * the rounding depends on the thread count); tests/test_oracle_pins.py checks it against the
 * sequential oracle with the same tolerances the GPU path has to meet.  Only tests/ and
 * bench.py's cpu legs may load it.  Build: gcc -O2 -ffp-contract=off -fopenmp.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <omp.h>

static void spmv(int64_t n, const int32_t *rp, const int32_t *ci, const double *va,
                 const double *x, double *y)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double s = 0.0;
        for (int64_t k = rp[i]; k < rp[i + 1]; ++k)
            s = s + va[k] * x[ci[k]];
        y[i] = s;
    }
}

static double dot(int64_t n, const double *a, const double *b)
{
    double s = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : s)
    for (int64_t i = 0; i < n; ++i)
        s = s + a[i] * b[i];
    return s;
}

int oracle_omp_threads(void) { return omp_get_max_threads(); }
void oracle_omp_set_threads(int t) { if (t > 0) omp_set_num_threads(t); }

/* Unpreconditioned CG; arguments and return value as oracle_cg (cg_oracle.c) without the
 * preconditioner and the diagnostics.  hist: maxit + 1 doubles. */
int oracle_cg_omp(int64_t n, const int32_t *rowptr, const int32_t *colind, const double *vals,
                  const double *b, double *x, double rtol, int64_t maxit, double *hist,
                  int64_t *iters_out, double *resnorm_out)
{
    if (n <= 0 || maxit < 0 || !(rtol >= 0.0) || !hist) return -1;
    double *r = (double *)malloc(sizeof(double) * (size_t)n);
    double *p = (double *)malloc(sizeof(double) * (size_t)n);
    double *q = (double *)malloc(sizeof(double) * (size_t)n);
    int status = 1;
    int64_t k = 0;
    double bb = dot(n, b, b);
    if (bb == 0.0) {
        memset(x, 0, sizeof(double) * (size_t)n);
        hist[0] = 0.0; *iters_out = 0; *resnorm_out = 0.0;
        free(r); free(p); free(q);
        return 0;
    }
    spmv(n, rowptr, colind, vals, x, q);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) { r[i] = b[i] - q[i]; p[i] = r[i]; }
    double rr = dot(n, r, r);
    hist[0] = sqrt(rr);
    const double thresh = rtol * sqrt(bb);
    while (1) {
        if (sqrt(rr) <= thresh) { status = 0; break; }
        if (k >= maxit) { status = 1; break; }
        spmv(n, rowptr, colind, vals, p, q);
        double pq = dot(n, p, q);
        if (!(pq > 0.0) || !isfinite(pq)) { status = 2; break; }
        double alpha = rr / pq;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) { x[i] = x[i] + alpha * p[i]; r[i] = r[i] - alpha * q[i]; }
        double rr_new = dot(n, r, r);
        double beta = rr_new / rr;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
        rr = rr_new;
        k = k + 1;
        hist[k] = sqrt(rr);
    }
    *iters_out = k;
    *resnorm_out = sqrt(rr);
    free(r); free(p); free(q);
    return status;
}
