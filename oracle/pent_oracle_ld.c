/* pent_oracle_ld.c -- the CPU ORACLE once more, in `long double` (x87 80-bit, 64-bit significand,
 * unit round-off 5.4e-20).  TEST INFRASTRUCTURE ONLY (same rules as pent_oracle.c).
 *
 * Why it exists (SURVEY.md section 8(c) reading C-7 allows long double on the host): for stiff
 * matrices (sigma ~ 1.1e4, cond(A) ~ 1.8e5) two CORRECT fp64 evaluations of A^{-1} f differ by
 * ~cond(A) * 2^-53 ~ 2e-11, which is above the 1e-11 parity bar of north_star.  This file gives the
 * tests a "truth" (error ~cond * 5e-20, then rounded once to fp64) against which BOTH the fp64
 * oracle and the GPU result are measured, so that the parity tolerance on those inputs is
 *     err(GPU, truth) <= max(1e-11, 2 * err(fp64 oracle, truth))
 * -- a measured quantity, not a fitted constant (reading C-15).
 *
 * It is the SAME literal transcription as pent_oracle.c / pent_oracle_step.c /
 * pent_oracle_periodic.c: factor = steps 1-14 of PAPER.md:167-221, forward sweep PAPER.md:223-231,
 * back substitution PAPER.md:233-242, periodic reduction Eqs. 8-12 (Eq. 12 then
 * Eq. 11), right-hand sides of Eq. 2 and Eq. 7c; only the arithmetic
 * type differs.  Inputs and outputs are fp64 arrays; every intermediate is long double.
 *
 * Pins (tests/test_oracle_ld_pins.py, -m "not gpu"): exact rational (fractions.Fraction) solves on
 * tiny N to 1e-18 (which the fp64 oracle cannot meet: proves the extra precision is real); the
 * closed-form eigenpairs at sigma = 1.1e4 evaluated in exact rational arithmetic times a
 * high-precision sine; agreement with the fp64 oracle to cond * 2^-53 on every function.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double R;

static int bad_pivot_ld(R alpha) { return alpha == 0.0L || !isfinite((double)alpha); }

/* PAPER.md:167-221, steps 1-14; same branches as pent_oracle_factor (reading C-4 for N < 4). */
static int factor_ld(int N, const R *a, const R *b, const R *c, const R *d, const R *e,
                     R *eps, R *beta, R *alpha, R *gamma, R *delta)
{
    int i;
    if (N < 1) return -1;
    for (i = 0; i < N; ++i) eps[i] = beta[i] = alpha[i] = gamma[i] = delta[i] = 0.0L;
    if (N < 4) {
        for (i = 0; i < N; ++i) {
            R g2 = i >= 2 ? gamma[i - 2] : 0.0L, d2 = i >= 2 ? delta[i - 2] : 0.0L;
            R g1 = i >= 1 ? gamma[i - 1] : 0.0L, d1 = i >= 1 ? delta[i - 1] : 0.0L;
            R ai = i >= 2 ? a[i] : 0.0L, bi = i >= 1 ? b[i] : 0.0L;
            R di = i + 1 < N ? d[i] : 0.0L, ei = i + 2 < N ? e[i] : 0.0L;
            beta[i] = bi - ai * g2;
            alpha[i] = c[i] - ai * d2 - beta[i] * g1;
            if (bad_pivot_ld(alpha[i])) return i + 1;
            gamma[i] = (di - beta[i] * d1) / alpha[i];
            delta[i] = ei / alpha[i];
            eps[i] = ai;
        }
        return 0;
    }
    alpha[0] = c[0];                                                        /* 1 */
    if (bad_pivot_ld(alpha[0])) return 1;
    gamma[0] = d[0] / alpha[0];                                             /* 2 */
    delta[0] = e[0] / alpha[0];                                             /* 3 */
    beta[1] = b[1];                                                         /* 4 */
    alpha[1] = c[1] - beta[1] * gamma[0];                                   /* 5 */
    if (bad_pivot_ld(alpha[1])) return 2;
    gamma[1] = (d[1] - beta[1] * delta[0]) / alpha[1];                      /* 6 */
    delta[1] = e[1] / alpha[1];                                             /* 7 */
    for (i = 2; i <= N - 3; ++i) {                                          /* 8 */
        beta[i] = b[i] - a[i] * gamma[i - 2];
        alpha[i] = c[i] - a[i] * delta[i - 2] - beta[i] * gamma[i - 1];
        if (bad_pivot_ld(alpha[i])) return i + 1;
        gamma[i] = (d[i] - beta[i] * delta[i - 1]) / alpha[i];
        delta[i] = e[i] / alpha[i];
    }
    i = N - 2;                                                              /* 9-11 */
    beta[i] = b[i] - a[i] * gamma[i - 2];
    alpha[i] = c[i] - a[i] * delta[i - 2] - beta[i] * gamma[i - 1];
    if (bad_pivot_ld(alpha[i])) return i + 1;
    gamma[i] = (d[i] - beta[i] * delta[i - 1]) / alpha[i];
    i = N - 1;                                                              /* 12-13 */
    beta[i] = b[i] - a[i] * gamma[i - 2];
    alpha[i] = c[i] - a[i] * delta[i - 2] - beta[i] * gamma[i - 1];
    if (bad_pivot_ld(alpha[i])) return i + 1;
    for (i = 2; i < N; ++i) eps[i] = a[i];                                  /* 14 */
    return 0;
}

/* PAPER.md:223-242; x may alias f */
static void solve_ld(int N, const R *eps, const R *beta, const R *alpha, const R *gamma, const R *delta,
                     const R *f, R *x)
{
    int i;
    R *g = x;
    g[0] = f[0] / alpha[0];
    if (N == 1) return;
    g[1] = (f[1] - beta[1] * g[0]) / alpha[1];
    for (i = 2; i < N; ++i) g[i] = (f[i] - eps[i] * g[i - 2] - beta[i] * g[i - 1]) / alpha[i];
    x[N - 2] = g[N - 2] - gamma[N - 2] * x[N - 1];
    for (i = N - 3; i >= 0; --i) x[i] = g[i] - gamma[i] * x[i + 1] - delta[i] * x[i + 2];
}

/* fp64 diagonals -> long double copies (5N) followed by the factors (5N); returns NULL on failure.
 * *rc receives the factor's return code. */
static R *widen_and_factor(int N, const double *a, const double *b, const double *c, const double *d,
                           const double *e, int *rc)
{
    R *w = (R *)malloc((size_t)10 * N * sizeof(R));
    int i;
    if (!w) { *rc = -2; return NULL; }
    for (i = 0; i < N; ++i) {
        w[i] = a[i]; w[N + i] = b[i]; w[2 * N + i] = c[i]; w[3 * N + i] = d[i]; w[4 * N + i] = e[i];
    }
    *rc = factor_ld(N, w, w + N, w + 2 * N, w + 3 * N, w + 4 * N, w + 5 * N, w + 6 * N, w + 7 * N,
                    w + 8 * N, w + 9 * N);
    return w;
}

/* Shared A, serial layout (M x N row-major F, X; X may alias F).  Returns the factor's code. */
int pent_oracle_ld_solve_rows(int N, long M, const double *a, const double *b, const double *c,
                              const double *d, const double *e, const double *F, double *X, int nthreads)
{
    int rc;
    long i;
    R *w = widen_and_factor(N, a, b, c, d, e, &rc);
    (void)nthreads;
    if (!w || rc != 0) { free(w); return rc; }
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i) {
        R *v = (R *)malloc((size_t)N * sizeof(R));
        int k;
        for (k = 0; k < N; ++k) v[k] = F[(size_t)i * N + k];
        solve_ld(N, w + 5 * N, w + 6 * N, w + 7 * N, w + 8 * N, w + 9 * N, v, v);
        for (k = 0; k < N; ++k) X[(size_t)i * N + k] = (double)v[k];
        free(v);
    }
    free(w);
    return 0;
}

/* Per-system matrices, every diagonal M x N row-major; info[i] as pent_oracle. */
void pent_oracle_ld_factor_solve_rows(int N, long M, const double *a, const double *b, const double *c,
                                      const double *d, const double *e, const double *F, double *X,
                                      int *info, int nthreads)
{
    long i;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i) {
        size_t o = (size_t)i * N;
        int rc, k;
        R *w = widen_and_factor(N, a + o, b + o, c + o, d + o, e + o, &rc);
        info[i] = rc;
        if (w && rc == 0) {
            R *v = (R *)malloc((size_t)N * sizeof(R));
            for (k = 0; k < N; ++k) v[k] = F[o + k];
            solve_ld(N, w + 5 * N, w + 6 * N, w + 7 * N, w + 8 * N, w + 9 * N, v, v);
            for (k = 0; k < N; ++k) X[o + k] = (double)v[k];
            free(v);
        }
        free(w);
    }
}

/* ---- time step (pent_oracle_step.c in long double) ------------------------------------------ */
static void apply_L_ld(int N, int bc, const R *w, R *y)
{
    int k;
    for (k = 0; k < N; ++k) {
        R diag = -2.0L, s;
        if (bc == 1 && (k == 0 || k == N - 1)) diag = -1.0L;
        s = diag * w[k];
        if (k > 0) s += w[k - 1];
        if (k + 1 < N) s += w[k + 1];
        y[k] = s;
    }
}

static void rhs_ld(int N, int kind, int bc, int form, R r, R sigma, const R *dg, const R *C, R *out, R *work)
{
    const R *a = dg, *b = dg + N, *c = dg + 2 * N, *d = dg + 3 * N, *e = dg + 4 * N;
    R *w = work, *t = work + N;
    int k;
    if (kind == 1) {
        for (k = 0; k < N; ++k) {
            R s = c[k] * C[k];
            if (k >= 1) s += b[k] * C[k - 1];
            if (k >= 2) s += a[k] * C[k - 2];
            if (k + 1 < N) s += d[k] * C[k + 1];
            if (k + 2 < N) s += e[k] * C[k + 2];
            out[k] = 2.0L * C[k] - s;
        }
        return;
    }
    for (k = 0; k < N; ++k) w[k] = C[k] * C[k] * C[k] - C[k];
    if (form == 0) {
        apply_L_ld(N, bc, w, t);
        for (k = 0; k < N; ++k) out[k] = C[k] + r * t[k];
    } else {
        apply_L_ld(N, bc, C, t);
        for (k = 0; k < N; ++k) w[k] = r * w[k] - sigma * t[k];
        apply_L_ld(N, bc, w, out);
    }
}

/* nsteps steps, state kept in long double between steps, rounded to fp64 at the end.
 * r and sigma are the fp64 values the caller passes to the library (widened exactly). */
int pent_oracle_ld_step_rows(int N, long M, int kind, int bc, int form, double r, double sigma,
                             const double *a, const double *b, const double *c, const double *d,
                             const double *e, double *C, int nsteps, int nthreads)
{
    int rc;
    long i;
    R *w = widen_and_factor(N, a, b, c, d, e, &rc);
    (void)nthreads;
    if (!w || rc != 0) { free(w); return rc; }
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i) {
        R *buf = (R *)malloc((size_t)5 * N * sizeof(R));
        R *ci = buf, *rhs = buf + N, *sol = buf + 2 * N, *work = buf + 3 * N;
        int s, k;
        for (k = 0; k < N; ++k) ci[k] = C[(size_t)i * N + k];
        for (s = 0; s < nsteps; ++s) {
            rhs_ld(N, kind, bc, form, (R)r, (R)sigma, w, ci, rhs, work);
            solve_ld(N, w + 5 * N, w + 6 * N, w + 7 * N, w + 8 * N, w + 9 * N, rhs, sol);
            if (kind == 0 && form == 1)
                for (k = 0; k < N; ++k) ci[k] = ci[k] + sol[k];
            else
                for (k = 0; k < N; ++k) ci[k] = sol[k];
        }
        for (k = 0; k < N; ++k) C[(size_t)i * N + k] = (double)ci[k];
        free(buf);
    }
    free(w);
    return 0;
}

/* ---- periodic solve (pent_oracle_periodic.c in long double): set-up + Eq. 12 + Eq. 11 ---------- */
int pent_oracle_ld_periodic_solve_rows(int N, long M, const double *a, const double *b, const double *c,
                                       const double *d, const double *e, const double *F, double *X,
                                       int nthreads)
{
    const int n = N - 2;
    int i, j, rc;
    long s;
    R *w, *da, *db, *dc, *dd, *de, *facE, *facT, *ta, *tb, *tc, *td, *te, *h, *Y, *kk;
    R s00, s01, s10, s11, det, inv[4];
    (void)nthreads;
    if (N < 6) return -1;
    w = (R *)calloc((size_t)5 * N + (size_t)21 * n, sizeof(R));
    if (!w) return -2;
    da = w; db = da + N; dc = db + N; dd = dc + N; de = dd + N;
    facE = de + N; facT = facE + 5 * n; ta = facT + 5 * n; tb = ta + n; tc = tb + n; td = tc + n; te = td + n;
    h = te + n; Y = h + 2 * n; kk = Y + 2 * n;
    for (i = 0; i < N; ++i) { da[i] = a[i]; db[i] = b[i]; dc[i] = c[i]; dd[i] = d[i]; de[i] = e[i]; }
    rc = factor_ld(n, da, db, dc, dd, de, facE, facE + n, facE + 2 * n, facE + 3 * n, facE + 4 * n);
    if (rc != 0) { free(w); return rc; }
    for (i = 0; i < n; ++i) {          /* E^T (reading C-20) */
        ta[i] = i >= 2 ? de[i - 2] : 0.0L;
        tb[i] = i >= 1 ? dd[i - 1] : 0.0L;
        tc[i] = dc[i];
        td[i] = i + 1 < n ? db[i + 1] : 0.0L;
        te[i] = i + 2 < n ? da[i + 2] : 0.0L;
    }
    rc = factor_ld(n, ta, tb, tc, td, te, facT, facT + n, facT + 2 * n, facT + 3 * n, facT + 4 * n);
    if (rc != 0) { free(w); return rc; }
    h[0] = de[N - 2]; h[n - 2] = da[N - 2]; h[n - 1] = db[N - 2];                 /* Eq. 9 */
    h[n + 0] = dd[N - 1]; h[n + 1] = de[N - 1]; h[n + n - 1] = da[N - 1];
    for (j = 0; j < 2; ++j)
        solve_ld(n, facT, facT + n, facT + 2 * n, facT + 3 * n, facT + 4 * n, h + j * n, Y + j * n);
    kk[0] = da[0]; kk[n - 2] = de[N - 4]; kk[n - 1] = dd[N - 3];
    kk[n + 0] = db[0]; kk[n + 1] += da[1]; kk[n + n - 1] = de[N - 3];
    s00 = dc[N - 2]; s01 = dd[N - 2]; s10 = db[N - 1]; s11 = dc[N - 1];
    for (i = 0; i < n; ++i) {
        s00 -= Y[i] * kk[i];     s01 -= Y[i] * kk[n + i];
        s10 -= Y[n + i] * kk[i]; s11 -= Y[n + i] * kk[n + i];
    }
    det = s00 * s11 - s01 * s10;
    if (det == 0.0L || !isfinite((double)det)) { free(w); return N - 1; }
    inv[0] = s11 / det; inv[1] = -s01 / det; inv[2] = -s10 / det; inv[3] = s00 / det;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (s = 0; s < M; ++s) {
        const double *f = F + (size_t)s * N;
        R *rhs = (R *)malloc((size_t)n * sizeof(R));
        R r0 = f[N - 2], r1 = f[N - 1], t0, t1;
        int k;
        for (k = 0; k < n; ++k) { r0 -= Y[k] * f[k]; r1 -= Y[n + k] * f[k]; }          /* Eq. 12 */
        t0 = inv[0] * r0 + inv[1] * r1;
        t1 = inv[2] * r0 + inv[3] * r1;
        for (k = 0; k < n; ++k) rhs[k] = f[k] - kk[k] * t0 - kk[n + k] * t1;            /* Eq. 11 */
        solve_ld(n, facE, facE + n, facE + 2 * n, facE + 3 * n, facE + 4 * n, rhs, rhs);
        for (k = 0; k < n; ++k) X[(size_t)s * N + k] = (double)rhs[k];
        X[(size_t)s * N + N - 2] = (double)t0;
        X[(size_t)s * N + N - 1] = (double)t1;
        free(rhs);
    }
    free(w);
    return 0;
}
