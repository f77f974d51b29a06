/* pent_oracle_step.c -- CPU ORACLE for the fused time-step path.  TEST INFRASTRUCTURE ONLY
 * (same rules as pent_oracle.c: only tests/, smoke() and bench.py's CPU legs may use it).
 *
 * One step = build the explicit right-hand side from the state, then one pentadiagonal
 * solve with the shared, already factored A (pent_oracle_solve).
 *
 *   kind 0, Cahn-Hilliard, PAPER.md:53 (Eq. 2, read with C^{n+1} on the left, reading C-19):
 *       (C+ - C)/dt = D d_xx (C^3 - C)  -  gamma D d_xxxx C+ ,  D = 1 (reading C-17)
 *     discretised with the second-difference matrix L (d_xx ~ L/dx^2, d_xxxx ~ L^2/dx^4):
 *       A C+ = C + r L w,   w = C^3 - C,   r = dt/dx^2,   A = I + sigma L^2,
 *       sigma = gamma dt/dx^4                                   ("direct form", form 0)
 *     and the algebraically identical increment form (reading C-14), form 1:
 *       q = r w - sigma L C ;   A delta = L q ;   C+ = C + delta
 *     (identity: C + r L w - A C = L (r w - sigma L C)).
 *   kind 1, hyperdiffusion Crank-Nicolson, PAPER.md:81-92 (Eqs. 5-6) and :117 (Eq. 7c):
 *       A C+ = (2I - A) C, evaluated row by row with the ORIGINAL diagonals of A
 *       (reading C-18: same boundary rows as A; the paper's matrix is periodic).
 *
 * L (reading C-13): (L w)_k = w_{k-1} - 2 w_k + w_{k+1}, neighbours outside 0..N-1 dropped;
 *   bc 0 (Dirichlet): nothing else;  bc 1 (zero-flux): the diagonal entry of rows 0 and N-1
 *   is -1 instead of -2, so that the column sums of L vanish and mean(C) is invariant.
 */
#include <stddef.h>
#include <stdlib.h>

void pent_oracle_solve(int N, const double *eps, const double *beta, const double *alpha,
                       const double *gamma, const double *delta, const double *f, double *x);

/* y = L w (length N, y must not alias w) */
void pent_oracle_apply_L(int N, int bc, const double *w, double *y)
{
    int k;
    for (k = 0; k < N; ++k) {
        double diag = -2.0;
        double s;
        if (bc == 1 && (k == 0 || k == N - 1)) diag = -1.0;
        s = diag * w[k];
        if (k > 0) s += w[k - 1];
        if (k + 1 < N) s += w[k + 1];
        y[k] = s;
    }
}

/* Right-hand side of one step for ONE system.  out has length N.  work: 2N doubles.
 * kind 0 form 0: out = C + r L (C^3 - C)
 * kind 0 form 1: out = L (r (C^3 - C) - sigma L C)           (the increment's RHS)
 * kind 1       : out = 2 C - A C   (original diagonals a..e, row-indexed)            */
void pent_oracle_rhs(int N, int kind, int bc, int form, double r, double sigma,
                     const double *a, const double *b, const double *c, const double *d,
                     const double *e, const double *C, double *out, double *work)
{
    int k;
    double *w = work, *t = work + N;
    if (kind == 1) {
        for (k = 0; k < N; ++k) {
            double s = c[k] * C[k];
            if (k >= 1) s += b[k] * C[k - 1];
            if (k >= 2) s += a[k] * C[k - 2];
            if (k + 1 < N) s += d[k] * C[k + 1];
            if (k + 2 < N) s += e[k] * C[k + 2];
            out[k] = 2.0 * C[k] - s;
        }
        return;
    }
    for (k = 0; k < N; ++k) w[k] = C[k] * C[k] * C[k] - C[k];
    if (form == 0) {
        pent_oracle_apply_L(N, bc, w, t);
        for (k = 0; k < N; ++k) out[k] = C[k] + r * t[k];
    } else {
        pent_oracle_apply_L(N, bc, C, t);
        for (k = 0; k < N; ++k) w[k] = r * w[k] - sigma * t[k];      /* q */
        pent_oracle_apply_L(N, bc, w, out);
    }
}

/* nsteps steps on a batch in the serial layout (M x N row-major, in place). */
void pent_oracle_step_rows(int N, long M, int kind, int bc, int form, double r, double sigma,
                           const double *a, const double *b, const double *c, const double *d,
                           const double *e,
                           const double *eps, const double *beta, const double *alpha,
                           const double *gamma, const double *delta,
                           double *C, int nsteps, int nthreads)
{
    long i;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i) {
        double *buf = (double *)malloc((size_t)4 * N * sizeof(double));
        double *rhs = buf, *sol = buf + N, *work = buf + 2 * N;
        double *Ci = C + (size_t)i * N;
        int s, k;
        for (s = 0; s < nsteps; ++s) {
            pent_oracle_rhs(N, kind, bc, form, r, sigma, a, b, c, d, e, Ci, rhs, work);
            pent_oracle_solve(N, eps, beta, alpha, gamma, delta, rhs, sol);
            if (kind == 0 && form == 1)
                for (k = 0; k < N; ++k) Ci[k] = Ci[k] + sol[k];
            else
                for (k = 0; k < N; ++k) Ci[k] = sol[k];
        }
        free(buf);
    }
}

/* ---------------------------------------------------------------------------------------
 * Forced Cahn-Hilliard, PAPER.md:63-67 (Remark 1, Eq. 3): dC/dt = [Eq. 1a] + Phi(x, t, mu_1, mu_2, ...),
 * "a parameter study based on the model (3) provides the motivation for batch programming in this
 * work": every system i of the batch has its own parameters (mu_1[i], mu_2[i]).
 * The paper specifies no Phi.  Reading C-22: a zero-mean travelling wave
 *     Phi(x, t; mu_1, mu_2) = mu_1 cos(2 pi (x - mu_2 t)),     x_k = (k + 1/2) / N  (cell centres, L = 1),
 * treated explicitly like the other bracketed term of Eq. 2 (evaluated at t_n = t0 + n dt):
 *     (C+ - C)/dt = [D d_xx (C^3 - C)]^n - gamma D d_xxxx C+ + Phi^n
 *  => form 0:  A C+ = C + r L w + dt Phi^n ;     form 1:  A delta = L q + dt Phi^n,  C+ = C + delta.
 * sum_k Phi(x_k) = 0 on this grid, so the zero-flux scheme still conserves mean(C).
 * ------------------------------------------------------------------------------------- */
#include <math.h>

void pent_oracle_forcing(int N, double t, double mu1, double mu2, double *phi)
{
    const double two_pi = 6.283185307179586476925286766559;
    int k;
    for (k = 0; k < N; ++k) {
        double x = ((double)k + 0.5) / (double)N;
        phi[k] = mu1 * cos(two_pi * (x - mu2 * t));
    }
}

/* nsteps forced steps (kind 0 only) on a batch in the serial layout (M x N row-major, in place);
 * mu1, mu2: M per-system parameters; step n of the call is taken at t_n = t0 + n dt. */
void pent_oracle_step_forced_rows(int N, long M, int bc, int form, double r, double sigma,
                                  double dt, double t0, const double *mu1, const double *mu2,
                                  const double *a, const double *b, const double *c, const double *d,
                                  const double *e,
                                  const double *eps, const double *beta, const double *alpha,
                                  const double *gamma, const double *delta,
                                  double *C, int nsteps, int nthreads)
{
    long i;
    (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
    for (i = 0; i < M; ++i) {
        double *buf = (double *)malloc((size_t)5 * N * sizeof(double));
        double *rhs = buf, *sol = buf + N, *work = buf + 2 * N, *phi = buf + 4 * N;
        double *Ci = C + (size_t)i * N;
        int s, k;
        for (s = 0; s < nsteps; ++s) {
            double t = t0 + (double)s * dt;
            pent_oracle_rhs(N, 0, bc, form, r, sigma, a, b, c, d, e, Ci, rhs, work);
            pent_oracle_forcing(N, t, mu1[i], mu2[i], phi);
            for (k = 0; k < N; ++k) rhs[k] = rhs[k] + dt * phi[k];
            pent_oracle_solve(N, eps, beta, alpha, gamma, delta, rhs, sol);
            if (form == 1)
                for (k = 0; k < N; ++k) Ci[k] = Ci[k] + sol[k];
            else
                for (k = 0; k < N; ++k) Ci[k] = sol[k];
        }
        free(buf);
    }
}
