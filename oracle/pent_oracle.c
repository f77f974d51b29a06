/* pent_oracle.c -- CPU ORACLE for the batched pentadiagonal path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, link or call this file.  The CUDA product (paper_1807_07382_b200/) shares no
 * code with it and never falls back to it.
 *
 * What it is: a plain, serial, fp64 transcription of the extended Thomas algorithm of
 * PAPER.md section II.D (lines 148-244): factor A = L R (steps 1-14),
 * forward sweep L g = f, back substitution R x = g,
 * in the paper's order and with true divisions.  Build with
 *     gcc -O2 -ffp-contract=off -fPIC -shared [-fopenmp]
 * so that no FMA contraction changes the rounding (reading C-5).
 *
 * Index convention (reading C-1): the paper is 1-based with
 * a_3..a_N, b_2..b_N, c_1..c_N, d_1..d_{N-1}, e_1..e_{N-2}.  Here every diagonal is a
 * 0-based length-N array indexed by ROW: a[k]=A[k][k-2], b[k]=A[k][k-1], c[k]=A[k][k],
 * d[k]=A[k][k+1], e[k]=A[k][k+2]; paper index i is array index i-1.  Entries outside
 * the matrix are never read.
 *
 * Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"): dense Gaussian elimination with
 * partial pivoting (function below) and exact rational elimination on tiny N; L*R == A;
 * closed-form eigenpairs of I + sigma L^2 (Dirichlet sine modes, zero-flux cosine modes);
 * manufactured f = A x; reduction to the tridiagonal Thomas algorithm / diagonal scaling;
 * LAPACK dgbsv through scipy.linalg.solve_banded; LDL^T invariants of symmetric A;
 * Toeplitz-interior fixed point of the factor recurrences; mean conservation of the
 * zero-flux Cahn-Hilliard step.  The paper prints no worked numerical example of a solve,
 * so no pin is a number printed in the paper (said so in DESIGN.md).
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static int bad_pivot(double alpha) { return alpha == 0.0 || !isfinite(alpha); }

/* ---------------------------------------------------------------------------------------
 * Factor A = L R.  PAPER.md:167-221, steps 1-14.  Outputs: eps, beta, alpha (bands of L)
 * and gamma, delta (bands of unit-upper R), length N each.  Entries the paper never
 * defines (beta_1, eps_1, eps_2, gamma_N, delta_{N-1}, delta_N) are stored as 0
 * (reading C-3).  Returns 0, or k+1 where k is the first 0-based row whose
 * pivot alpha_k is zero or non-finite (no pivoting is attempted).
 * ------------------------------------------------------------------------------------- */
int pent_oracle_factor(int N, const double *a, const double *b, const double *c,
                       const double *d, const double *e,
                       double *eps, double *beta, double *alpha, double *gamma, double *delta)
{
    int i;
    if (N < 1) return -1;
    for (i = 0; i < N; ++i) { eps[i] = beta[i] = alpha[i] = gamma[i] = delta[i] = 0.0; }

    if (N < 4) {
        /* The paper's step list special-cases rows 1,2 and N-1,N and so needs N >= 4.
         * For N = 1,2,3 use the same recurrences (steps 8.1-8.4) with every out-of-range
         * term dropped (reading C-4). */
        for (i = 0; i < N; ++i) {
            double g2 = i >= 2 ? gamma[i - 2] : 0.0, d2 = i >= 2 ? delta[i - 2] : 0.0;
            double g1 = i >= 1 ? gamma[i - 1] : 0.0, d1 = i >= 1 ? delta[i - 1] : 0.0;
            double ai = i >= 2 ? a[i] : 0.0, bi = i >= 1 ? b[i] : 0.0;
            double di = i + 1 < N ? d[i] : 0.0, ei = i + 2 < N ? e[i] : 0.0;
            beta[i] = bi - ai * g2;
            alpha[i] = c[i] - ai * d2 - beta[i] * g1;
            if (bad_pivot(alpha[i])) return i + 1;
            gamma[i] = (di - beta[i] * d1) / alpha[i];
            delta[i] = ei / alpha[i];
            eps[i] = ai;
        }
        return 0;
    }

    /* step 1-3 (paper row 1 = index 0) */
    alpha[0] = c[0];
    if (bad_pivot(alpha[0])) return 1;
    gamma[0] = d[0] / alpha[0];
    delta[0] = e[0] / alpha[0];
    /* step 4-7 (paper row 2 = index 1) */
    beta[1] = b[1];
    alpha[1] = c[1] - beta[1] * gamma[0];
    if (bad_pivot(alpha[1])) return 2;
    gamma[1] = (d[1] - beta[1] * delta[0]) / alpha[1];
    delta[1] = e[1] / alpha[1];
    /* step 8: paper i = 3..N-2  ->  index 2..N-3 */
    for (i = 2; i <= N - 3; ++i) {
        beta[i] = b[i] - a[i] * gamma[i - 2];                               /* 8.1 */
        alpha[i] = c[i] - a[i] * delta[i - 2] - beta[i] * gamma[i - 1];     /* 8.2 */
        if (bad_pivot(alpha[i])) return i + 1;
        gamma[i] = (d[i] - beta[i] * delta[i - 1]) / alpha[i];              /* 8.3 */
        delta[i] = e[i] / alpha[i];                                         /* 8.4 */
    }
    /* step 9-11 (paper row N-1 = index N-2) */
    i = N - 2;
    beta[i] = b[i] - a[i] * gamma[i - 2];
    alpha[i] = c[i] - a[i] * delta[i - 2] - beta[i] * gamma[i - 1];
    if (bad_pivot(alpha[i])) return i + 1;
    gamma[i] = (d[i] - beta[i] * delta[i - 1]) / alpha[i];
    /* step 12-13 (paper row N = index N-1) */
    i = N - 1;
    beta[i] = b[i] - a[i] * gamma[i - 2];
    alpha[i] = c[i] - a[i] * delta[i - 2] - beta[i] * gamma[i - 1];
    if (bad_pivot(alpha[i])) return i + 1;
    /* step 14: eps_i = a_i for all i (a_1, a_2 do not exist -> 0) */
    for (i = 2; i < N; ++i) eps[i] = a[i];
    return 0;
}

/* ---------------------------------------------------------------------------------------
 * Solve one system (contiguous f, x of length N; x may alias f).
 * Forward sweep PAPER.md:223-231, back substitution PAPER.md:233-242.
 * g is held in x (the paper overwrites the right-hand side).
 * ------------------------------------------------------------------------------------- */
void pent_oracle_solve(int N, const double *eps, const double *beta, const double *alpha,
                       const double *gamma, const double *delta, const double *f, double *x)
{
    int i;
    double *g = x;
    /* forward 1. */
    g[0] = f[0] / alpha[0];
    if (N == 1) return;
    /* forward 2. */
    g[1] = (f[1] - beta[1] * g[0]) / alpha[1];
    /* forward 3. */
    for (i = 2; i < N; ++i)
        g[i] = (f[i] - eps[i] * g[i - 2] - beta[i] * g[i - 1]) / alpha[i];
    /* back 1. x_N = g_N (already in place) */
    /* back 2. */
    x[N - 2] = g[N - 2] - gamma[N - 2] * x[N - 1];
    /* back 3. */
    for (i = N - 3; i >= 0; --i)
        x[i] = g[i] - gamma[i] * x[i + 1] - delta[i] * x[i + 2];
}

/* ---------------------------------------------------------------------------------------
 * Batch drivers.  Layout is the paper's SERIAL layout, "one system per row"
 * (PAPER.md:349): F and X are M x N row-major, system i occupies F[i*N .. i*N+N-1].
 * The Python wrapper transposes from / to the interleaved layout outside this file.
 * nthreads > 1 parallelises the loop over systems exactly as the paper's OpenMP variant
 * (PAPER.md:369); the arithmetic of each system is unchanged.
 * ------------------------------------------------------------------------------------- */
void pent_oracle_solve_rows(int N, long M, const double *eps, const double *beta,
                            const double *alpha, const double *gamma, const double *delta,
                            const double *F, double *X, int nthreads)
{
    long i;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i)
        pent_oracle_solve(N, eps, beta, alpha, gamma, delta, F + (size_t)i * N, X + (size_t)i * N);
}

/* Per-system matrices ("Rewrite" mode): every diagonal is M x N row-major.
 * info[i] = 0 or (first bad row + 1); X of a failed system is left untouched. */
void pent_oracle_factor_solve_rows(int N, long M, const double *a, const double *b,
                                   const double *c, const double *d, const double *e,
                                   const double *F, double *X, int *info, int nthreads)
{
    long i;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i) {
        double *w = (double *)malloc((size_t)5 * N * sizeof(double));
        size_t o = (size_t)i * N;
        int rc = pent_oracle_factor(N, a + o, b + o, c + o, d + o, e + o,
                                    w, w + N, w + 2 * N, w + 3 * N, w + 4 * N);
        info[i] = rc;
        if (rc == 0)
            pent_oracle_solve(N, w, w + N, w + 2 * N, w + 3 * N, w + 4 * N, F + o, X + o);
        free(w);
    }
}

/* ---------------------------------------------------------------------------------------
 * Second, independent oracle: dense Gaussian elimination with partial pivoting on the
 * full N x N matrix (row-major A, destroyed; f destroyed; x out).  Exists only to pin the
 * banded algorithm on tiny N (north_star).  Returns 0, or 1 if A is singular.
 * ------------------------------------------------------------------------------------- */
int pent_oracle_dense_ge(int N, double *A, double *f, double *x)
{
    int i, j, k;
    for (k = 0; k < N; ++k) {
        int p = k;
        double big = fabs(A[(size_t)k * N + k]);
        for (i = k + 1; i < N; ++i)
            if (fabs(A[(size_t)i * N + k]) > big) { big = fabs(A[(size_t)i * N + k]); p = i; }
        if (big == 0.0) return 1;
        if (p != k) {
            for (j = 0; j < N; ++j) {
                double t = A[(size_t)k * N + j];
                A[(size_t)k * N + j] = A[(size_t)p * N + j];
                A[(size_t)p * N + j] = t;
            }
            { double t = f[k]; f[k] = f[p]; f[p] = t; }
        }
        for (i = k + 1; i < N; ++i) {
            double m = A[(size_t)i * N + k] / A[(size_t)k * N + k];
            if (m != 0.0) {
                for (j = k; j < N; ++j) A[(size_t)i * N + j] -= m * A[(size_t)k * N + j];
                f[i] -= m * f[k];
            }
        }
    }
    for (i = N - 1; i >= 0; --i) {
        double s = f[i];
        for (j = i + 1; j < N; ++j) s -= A[(size_t)i * N + j] * x[j];
        x[i] = s / A[(size_t)i * N + i];
    }
    return 0;
}
