/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * Plain, slow, obviously-correct CPU definition of what the hot path computes: for every
 * (i,k) line of an nx*ny*nz slab (x fastest, element (i,j,k) at i + nx*(j + ny*k)) the x with
 *
 *        a_j x_{j-1} + b_j x_j + c_j x_{j+1} = d_j ,   j = 0..ny-1,
 *
 * a = sub-, b = main, c = super-diagonal ("Problem: Ax = d (N times); Input
 * a,b,c,d; Output x").  a at j=0 and c at j=ny-1 are ignored.
 *
 * The method under test (divide-and-conquer partitions + reduced system + back-substitution,
 * PAPER.md:49-58) is a DIRECT solver: in exact arithmetic it returns this same x.  The oracle is
 * therefore the textbook sequential Thomas algorithm (ref [38]) applied to the whole
 * line, with NO partitioning, no blocking, no fusion:
 *
 *   c'_0 = c_0/b_0, d'_0 = d_0/b_0
 *   j=1..n-1: den = b_j - a_j c'_{j-1};  c'_j = c_j/den;  d'_j = (d_j - a_j d'_{j-1})/den
 *   x_{n-1} = d'_{n-1};  j=n-2..0: x_j = d'_j - c'_j x_{j+1}
 *
 * No pivoting: the inputs are diagonally dominant.  Each line is gathered into
 * contiguous temporaries, solved, and scattered back.  Two precisions of the same routine:
 * fp64 (the gate precision) and long double (reference for the weakly dominant Poisson lines,
 * SURVEY.md 8(c) G9).  Residuals are evaluated in long double.
 *
 * Shares no code with paper_2509_03933_b200/ (the CUDA path); neither includes the other.
 * Pins: tests/test_oracle_pins.py (dense LAPACK solve, manufactured solutions, Toeplitz closed
 * forms, banded LAPACK, degenerate cases).
 *
 * The loops over lines carry an OpenMP "parallel for" (lines are independent); this is how the
 * oracle "as it stands" is timed as the reported CPU baseline.  oracle_set_threads(1) gives the
 * single-core figure.
 */
#include <stddef.h>
#include <stdlib.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* One line, fp64.  cp, dp: work arrays of length n. */
static void thomas_line_f64(int n, const double *a, const double *b, const double *c,
                            const double *d, double *x, double *cp, double *dp)
{
    cp[0] = c[0] / b[0];
    dp[0] = d[0] / b[0];
    for (int j = 1; j < n; ++j) {
        double den = b[j] - a[j] * cp[j - 1];
        cp[j] = c[j] / den;
        dp[j] = (d[j] - a[j] * dp[j - 1]) / den;
    }
    x[n - 1] = dp[n - 1];
    for (int j = n - 2; j >= 0; --j) x[j] = dp[j] - cp[j] * x[j + 1];
}

/* One line, long double arithmetic on double inputs; result rounded once to double. */
static void thomas_line_ld(int n, const double *a, const double *b, const double *c,
                           const double *d, double *x, long double *cp, long double *dp)
{
    cp[0] = (long double)c[0] / (long double)b[0];
    dp[0] = (long double)d[0] / (long double)b[0];
    for (int j = 1; j < n; ++j) {
        long double den = (long double)b[j] - (long double)a[j] * cp[j - 1];
        cp[j] = (long double)c[j] / den;
        dp[j] = ((long double)d[j] - (long double)a[j] * dp[j - 1]) / den;
    }
    long double xn = dp[n - 1];
    x[n - 1] = (double)xn;
    for (int j = n - 2; j >= 0; --j) {
        xn = dp[j] - cp[j] * xn;
        x[j] = (double)xn;
    }
}

/* Solve every y-line of the slab.  use_ld = 0: fp64 Thomas; 1: long double Thomas.
 * Returns 0, or -1 on bad arguments / allocation failure. */
int oracle_solve_y(int nx, int ny, int nz, const double *a, const double *b, const double *c,
                   const double *d, double *x, int use_ld)
{
    if (nx < 1 || ny < 1 || nz < 1 || !a || !b || !c || !d || !x) return -1;
    int fail = 0;
    const long nlines = (long)nx * nz;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 5 * (size_t)ny);
        void *work = malloc((use_ld ? sizeof(long double) : sizeof(double)) * 2 * (size_t)ny);
        if (!buf || !work) {
#pragma omp atomic write
            fail = 1;
        }
        double *la = buf, *lb = buf + ny, *lc = buf + 2 * ny, *ld = buf + 3 * ny, *lx = buf + 4 * ny;
#pragma omp for schedule(static)
        for (long line = 0; line < nlines; ++line) {
            if (!buf || !work) continue;
            const long i = line % nx, k = line / nx;
            const size_t base = (size_t)i + (size_t)nx * (size_t)ny * (size_t)k;
            for (int j = 0; j < ny; ++j) {              /* gather the strided line */
                const size_t o = base + (size_t)nx * (size_t)j;
                la[j] = a[o]; lb[j] = b[o]; lc[j] = c[o]; ld[j] = d[o];
            }
            la[0] = 0.0;                                 /* ignored entries */
            lc[ny - 1] = 0.0;
            if (use_ld)
                thomas_line_ld(ny, la, lb, lc, ld, lx, (long double *)work, (long double *)work + ny);
            else
                thomas_line_f64(ny, la, lb, lc, ld, lx, (double *)work, (double *)work + ny);
            for (int j = 0; j < ny; ++j) x[base + (size_t)nx * (size_t)j] = lx[j];   /* scatter */
        }
        free(buf);
        free(work);
    }
    return fail ? -1 : 0;
}

/* Per-line residual report, evaluated in long double:
 *   res[line]  = || A x - d ||_inf
 *   dinf[line] = || d ||_inf,  xinf[line] = || x ||_inf,
 *   ainf[line] = || A ||_inf  (max row sum of |a|+|b|+|c|, with a_0 = c_{n-1} = 0).
 * Output arrays have nx*nz entries, line = i + nx*k. */
int oracle_residual_y(int nx, int ny, int nz, const double *a, const double *b, const double *c,
                      const double *d, const double *x, double *res, double *dinf, double *xinf,
                      double *ainf)
{
    if (nx < 1 || ny < 1 || nz < 1 || !a || !b || !c || !d || !x || !res || !dinf || !xinf || !ainf)
        return -1;
    const long nlines = (long)nx * nz;
#pragma omp parallel for schedule(static)
    for (long line = 0; line < nlines; ++line) {
        const long i = line % nx, k = line / nx;
        const size_t base = (size_t)i + (size_t)nx * (size_t)ny * (size_t)k;
        long double rmax = 0, dmax = 0, xmax = 0, amax = 0;
        for (int j = 0; j < ny; ++j) {
            const size_t o = base + (size_t)nx * (size_t)j;
            long double aj = (j == 0) ? 0.0L : (long double)a[o];
            long double cj = (j == ny - 1) ? 0.0L : (long double)c[o];
            long double r = (long double)b[o] * (long double)x[o] - (long double)d[o];
            if (j > 0) r += aj * (long double)x[o - (size_t)nx];
            if (j < ny - 1) r += cj * (long double)x[o + (size_t)nx];
            long double rowsum = fabsl(aj) + fabsl((long double)b[o]) + fabsl(cj);
            if (fabsl(r) > rmax) rmax = fabsl(r);
            if (fabsl((long double)d[o]) > dmax) dmax = fabsl((long double)d[o]);
            if (fabsl((long double)x[o]) > xmax) xmax = fabsl((long double)x[o]);
            if (rowsum > amax) amax = rowsum;
        }
        res[line] = (double)rmax; dinf[line] = (double)dmax;
        xinf[line] = (double)xmax; ainf[line] = (double)amax;
    }
    return 0;
}

/* d = A x evaluated in long double and rounded once (manufactured solutions, pin P2). */
int oracle_apply_y(int nx, int ny, int nz, const double *a, const double *b, const double *c,
                   const double *x, double *d)
{
    if (nx < 1 || ny < 1 || nz < 1 || !a || !b || !c || !d || !x) return -1;
    const long nlines = (long)nx * nz;
#pragma omp parallel for schedule(static)
    for (long line = 0; line < nlines; ++line) {
        const long i = line % nx, k = line / nx;
        const size_t base = (size_t)i + (size_t)nx * (size_t)ny * (size_t)k;
        for (int j = 0; j < ny; ++j) {
            const size_t o = base + (size_t)nx * (size_t)j;
            long double r = (long double)b[o] * (long double)x[o];
            if (j > 0) r += (long double)a[o] * (long double)x[o - (size_t)nx];
            if (j < ny - 1) r += (long double)c[o] * (long double)x[o + (size_t)nx];
            d[o] = (double)r;
        }
    }
    return 0;
}

/* Shared-coefficient lines.  The paper's own workload: the coefficient
 * matrix "depends solely on grid spacing", the FFT-reduced Poisson operator is
 * (d^2/dy^2 - k_l - k_m) and the fields are complex with real coefficients
 * (PAPER.md:377, 383).  So a, c and the y-part of the diagonal are 1-D arrays of length ny and
 * line (i,k) has
 *        a_j = a_y[j],   c_j = c_y[j],   b_j = b0_y[j] - (sx[i] + sz[k]),
 * the shift s = sx[i] + sz[k] being formed once per line, in fp64, before it is subtracted.
 * d and x hold ncomp (1 = real, 2 = complex, interleaved re/im) values per cell, element
 * (i,j,k,q) at q + ncomp*(i + nx*(j + ny*k)); every component is a separate right-hand side of
 * the same real matrix.  pin00 != 0: row 0 of line (0,0) is replaced by b = 1, c = 0 (the
 * singular mean mode pinned by x_0 = d_0, BASELINE cfg 2/3).  Still the plain Thomas algorithm
 * per line and component: nothing is shared between lines, nothing is precomputed. */
int oracle_solve_y_shared(int nx, int ny, int nz, int ncomp, const double *a_y, const double *b0_y,
                          const double *c_y, const double *sx, const double *sz, int pin00,
                          const double *d, double *x, int use_ld)
{
    if (nx < 1 || ny < 1 || nz < 1 || ncomp < 1 || ncomp > 2 || !a_y || !b0_y || !c_y || !sx || !sz || !d || !x)
        return -1;
    int fail = 0;
    const long nlines = (long)nx * nz;
#pragma omp parallel
    {
        double *buf = (double *)malloc(sizeof(double) * 5 * (size_t)ny);
        void *work = malloc((use_ld ? sizeof(long double) : sizeof(double)) * 2 * (size_t)ny);
        if (!buf || !work) {
#pragma omp atomic write
            fail = 1;
        }
        double *la = buf, *lb = buf + ny, *lc = buf + 2 * ny, *ld = buf + 3 * ny, *lx = buf + 4 * ny;
#pragma omp for schedule(static)
        for (long line = 0; line < nlines; ++line) {
            if (!buf || !work) continue;
            const long i = line % nx, k = line / nx;
            const double s = sx[i] + sz[k];
            for (int j = 0; j < ny; ++j) { la[j] = a_y[j]; lb[j] = b0_y[j] - s; lc[j] = c_y[j]; }
            la[0] = 0.0;
            lc[ny - 1] = 0.0;
            if (pin00 && i == 0 && k == 0) { lb[0] = 1.0; lc[0] = 0.0; }
            for (int q = 0; q < ncomp; ++q) {
                const size_t base = (size_t)q + (size_t)ncomp * ((size_t)i + (size_t)nx * (size_t)ny * (size_t)k);
                const size_t step = (size_t)ncomp * (size_t)nx;
                for (int j = 0; j < ny; ++j) ld[j] = d[base + step * (size_t)j];
                if (use_ld)
                    thomas_line_ld(ny, la, lb, lc, ld, lx, (long double *)work, (long double *)work + ny);
                else
                    thomas_line_f64(ny, la, lb, lc, ld, lx, (double *)work, (double *)work + ny);
                for (int j = 0; j < ny; ++j) x[base + step * (size_t)j] = lx[j];
            }
        }
        free(buf);
        free(work);
    }
    return fail ? -1 : 0;
}
