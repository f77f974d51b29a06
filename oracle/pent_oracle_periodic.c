/* pent_oracle_periodic.c -- CPU ORACLE for the PERIODIC (cyclic) pentadiagonal solve and the
 * periodic hyperdiffusion time step.  TEST INFRASTRUCTURE ONLY (same rules as pent_oracle.c:
 * only tests/, smoke() and bench.py's CPU legs may use it; the CUDA product shares no code).
 *
 * What it follows: PAPER.md section II.C (lines 104-146), the reduction the paper takes from
 * Navon: the N x N periodic matrix of Eq. 7a is split into the strictly pentadiagonal
 * (N-2) x (N-2) block E (Eq. 8), the two last columns k and the two last rows h^T (Eq. 9) and the
 * 2 x 2 corner block; then, in the paper's order,
 *     (x_{N-1}, x_N)^T = [ C2 - h^T E^{-1} k ]^{-1} [ (f_{N-1}, f_N)^T - h^T E^{-1} f^ ]     (Eq. 12)
 *     X^ = E^{-1} [ f^ - k (x_{N-1}, x_N)^T ]                                                (Eq. 11)
 * with h^T E^{-1} and the inverted 2 x 2 matrix computed once and stored.
 *
 * Readings:
 *  C-21  The paper writes the matrix with constant a..e (Eq. 7a).  Here every diagonal is a
 *        length-N array indexed by ROW, wrapped cyclically: a[k] = A[k][(k-2) mod N],
 *        b[k] = A[k][(k-1) mod N], c[k] = A[k][k], d[k] = A[k][(k+1) mod N],
 *        e[k] = A[k][(k+2) mod N]; ALL N entries of every array are used.  N >= 6 so that the
 *        corner entries do not overlap the band.  With constant arrays this is Eq. 7a/9 exactly:
 *        k = (a b; 0 a; 0 0; ...; e 0; d e), h = (e d; 0 e; 0 0; ...; a 0; b a).
 *  C-20  "(E^{-1})^T h = h^T E^{-1}" is read as: the stored quantity is
 *        Y = E^{-T} h, i.e. two solves with E TRANSPOSED (for the symmetric E of the paper the
 *        same factorisation serves).  E^T is pentadiagonal with the diagonals mirrored, and is
 *        factored by the same routine.
 *
 * The periodic hyperdiffusion step is Eq. 6 / 7c: A c+ = (2I - A) c with
 * the cyclic A, evaluated row by row from the original diagonals.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int pent_oracle_factor(int N, const double *a, const double *b, const double *c,
                       const double *d, const double *e,
                       double *eps, double *beta, double *alpha, double *gamma, double *delta);
void pent_oracle_solve(int N, const double *eps, const double *beta, const double *alpha,
                       const double *gamma, const double *delta, const double *f, double *x);

/* Set-up.  Outputs: facE = 5*(N-2) doubles (eps,beta,alpha,gamma,delta of E), Y = 2*(N-2)
 * doubles (row j = column j of E^{-T} h, i.e. row j of h^T E^{-1}), kk = 2*(N-2) doubles (the two
 * columns of k, kept for Eq. 11), s2inv = 4 doubles (row-major inverse of C2 - h^T E^{-1} k).
 * Returns 0; r+1 if row r of E (or of E^T) has a bad pivot; N-1 (+0) style code N if the 2x2
 * Schur complement is singular (reported as row N-2, i.e. return value N-1). */
int pent_oracle_periodic_setup(int N, const double *a, const double *b, const double *c,
                               const double *d, const double *e,
                               double *facE, double *Y, double *kk, double *s2inv)
{
    const int n = N - 2;
    int i, j, rc;
    double *w, *ta, *tb, *tc, *td, *te, *facT, *h;
    double s00, s01, s10, s11, det;
    if (N < 6) return -1;
    /* E: rows/columns 0..N-3 of A: the band entries that stay inside the block (Eq. 8) */
    rc = pent_oracle_factor(n, a, b, c, d, e, facE, facE + n, facE + 2 * n, facE + 3 * n, facE + 4 * n);
    if (rc != 0) return rc;
    /* E^T: (E^T)[k][k-2] = E[k-2][k] = e[k-2], (E^T)[k][k-1] = d[k-1], (E^T)[k][k+1] = b[k+1],
     * (E^T)[k][k+2] = a[k+2] */
    w = (double *)calloc((size_t)12 * n, sizeof(double));
    if (!w) return -2;
    ta = w; tb = w + n; tc = w + 2 * n; td = w + 3 * n; te = w + 4 * n; facT = w + 5 * n; h = w + 10 * n;
    for (i = 0; i < n; ++i) {
        ta[i] = i >= 2 ? e[i - 2] : 0.0;
        tb[i] = i >= 1 ? d[i - 1] : 0.0;
        tc[i] = c[i];
        td[i] = i + 1 < n ? b[i + 1] : 0.0;
        te[i] = i + 2 < n ? a[i + 2] : 0.0;
    }
    rc = pent_oracle_factor(n, ta, tb, tc, td, te, facT, facT + n, facT + 2 * n, facT + 3 * n, facT + 4 * n);
    if (rc != 0) { free(w); return rc; }
    /* h (Eq. 9), column 0 = row N-2 of A restricted to columns 0..N-3, column 1 = row N-1 */
    for (i = 0; i < 2 * n; ++i) h[i] = 0.0;
    h[0] = e[N - 2];            /* A[N-2][0]   */
    h[n - 2] = a[N - 2];        /* A[N-2][N-4] */
    h[n - 1] = b[N - 2];        /* A[N-2][N-3] */
    h[n + 0] = d[N - 1];        /* A[N-1][0]   */
    h[n + 1] = e[N - 1];        /* A[N-1][1]   */
    h[n + n - 1] = a[N - 1];    /* A[N-1][N-3] */
    for (j = 0; j < 2; ++j)
        pent_oracle_solve(n, facT, facT + n, facT + 2 * n, facT + 3 * n, facT + 4 * n, h + j * n, Y + j * n);
    /* k (Eq. 9), column 0 = column N-2 of A restricted to rows 0..N-3, column 1 = column N-1 */
    for (i = 0; i < 2 * n; ++i) kk[i] = 0.0;
    kk[0] = a[0];               /* A[0][N-2]   */
    kk[n - 2] = e[N - 4];       /* A[N-4][N-2] */
    kk[n - 1] = d[N - 3];       /* A[N-3][N-2] */
    kk[n + 0] = b[0];           /* A[0][N-1]   */
    kk[n + 1] = a[1];           /* A[1][N-1]   */
    kk[n + n - 1] = e[N - 3];   /* A[N-3][N-1] */
    /* S2 = C2 - h^T E^{-1} k, C2 = (c_{N-1} d_{N-1}; b_N c_N) in the paper's 1-based notation */
    s00 = c[N - 2]; s01 = d[N - 2]; s10 = b[N - 1]; s11 = c[N - 1];
    for (i = 0; i < n; ++i) {
        s00 -= Y[i] * kk[i];     s01 -= Y[i] * kk[n + i];
        s10 -= Y[n + i] * kk[i]; s11 -= Y[n + i] * kk[n + i];
    }
    free(w);
    det = s00 * s11 - s01 * s10;
    if (det == 0.0 || !isfinite(det)) return N - 1;
    s2inv[0] = s11 / det; s2inv[1] = -s01 / det; s2inv[2] = -s10 / det; s2inv[3] = s00 / det;
    return 0;
}

/* One system, contiguous f and x of length N (x must not alias f). */
void pent_oracle_periodic_solve(int N, const double *facE, const double *Y, const double *kk,
                                const double *s2inv, const double *f, double *x)
{
    const int n = N - 2;
    int i;
    double r0 = f[N - 2], r1 = f[N - 1], t0, t1;
    double *rhs = (double *)malloc((size_t)n * sizeof(double));
    /* Eq. 12 */
    for (i = 0; i < n; ++i) { r0 -= Y[i] * f[i]; r1 -= Y[n + i] * f[i]; }
    t0 = s2inv[0] * r0 + s2inv[1] * r1;
    t1 = s2inv[2] * r0 + s2inv[3] * r1;
    /* Eq. 11 */
    for (i = 0; i < n; ++i) rhs[i] = f[i] - kk[i] * t0 - kk[n + i] * t1;
    pent_oracle_solve(n, facE, facE + n, facE + 2 * n, facE + 3 * n, facE + 4 * n, rhs, x);
    x[N - 2] = t0;
    x[N - 1] = t1;
    free(rhs);
}

void pent_oracle_periodic_solve_rows(int N, long M, const double *facE, const double *Y,
                                     const double *kk, const double *s2inv, const double *F,
                                     double *X, int nthreads)
{
    long i;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i)
        pent_oracle_periodic_solve(N, facE, Y, kk, s2inv, F + (size_t)i * N, X + (size_t)i * N);
}

/* y = (2I - A) v with the cyclic A (Eq. 7c generalised to row-indexed diagonals); y != v */
void pent_oracle_periodic_rhs(int N, const double *a, const double *b, const double *c,
                              const double *d, const double *e, const double *v, double *y)
{
    int k;
    for (k = 0; k < N; ++k) {
        double s = c[k] * v[k];
        s += b[k] * v[(k + N - 1) % N];
        s += a[k] * v[(k + N - 2) % N];
        s += d[k] * v[(k + 1) % N];
        s += e[k] * v[(k + 2) % N];
        y[k] = 2.0 * v[k] - s;
    }
}

/* nsteps Crank-Nicolson steps A c+ = (2I - A) c on M systems in the serial layout (M x N). */
void pent_oracle_periodic_step_rows(int N, long M, const double *a, const double *b,
                                    const double *c, const double *d, const double *e,
                                    const double *facE, const double *Y, const double *kk,
                                    const double *s2inv, double *C, int nsteps, int nthreads)
{
    long i;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i) {
        double *rhs = (double *)malloc((size_t)N * sizeof(double));
        double *ci = C + (size_t)i * N;
        int s;
        for (s = 0; s < nsteps; ++s) {
            pent_oracle_periodic_rhs(N, a, b, c, d, e, ci, rhs);
            pent_oracle_periodic_solve(N, facE, Y, kk, s2inv, rhs, ci);
        }
        free(rhs);
    }
}
