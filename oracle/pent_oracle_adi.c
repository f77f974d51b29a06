/* pent_oracle_adi.c -- CPU ORACLE for a 2-D alternating-direction-implicit (ADI) time step built on the
 * pentadiagonal solver.  TEST INFRASTRUCTURE ONLY (same rules as pent_oracle.c).
 *
 * PAPER.md:379 (section IV): "solving parabolic numerical PDEs in two and three dimensions ... The resulting
 * matrix to be inverted at each time step can be reduced to a series of one-dimensional problems using the
 * alternating-direction-implicit (ADI) technique.  In this scenario, the present pentadiagonal batch solver may
 * prove useful".  The paper gives no scheme.  Reading C-23: the Peaceman-Rachford splitting of
 *     u_t = D_x u + D_y u,        A_x = I - (dt/2) D_x,    A_y = I - (dt/2) D_y
 * (each A pentadiagonal along its own axis, e.g. the Remark-3 heat matrix of PAPER.md:96 or the hyperdiffusion
 * matrix of Eq. 7b without the cross term), one time step =
 *     half step 1:   A_x u*      = (2I - A_y) u^n      explicit along y, implicit along x
 *     half step 2:   A_y u^{n+1} = (2I - A_x) u*       explicit along x, implicit along y
 * i.e. every half step is "(2I - A) c" along one axis (Eq. 7c's form) followed by a batch of
 * 1-D pentadiagonal solves along the other.  Because (I (x) A_x) and (A_y (x) I) commute,
 * the step equals  (A_y (x) A_x)^{-1} ((2I - A_y) (x) (2I - A_x)) u^n  exactly (the pin of the tests).
 *
 * Field layout: U is Ny x Nx row-major, U[y*Nx + x]; rows are x-lines (systems of length Nx, "one system per
 * row"), columns are y-lines (an interleaved batch of Nx systems of length Ny).
 */
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

void pent_oracle_solve(int N, const double *eps, const double *beta, const double *alpha,
                       const double *gamma, const double *delta, const double *f, double *x);

/* out_k = 2 v_k - (A v)_k along a strided line of length N (row-indexed diagonals a..e of A) */
static void two_i_minus_a(int N, const double *a, const double *b, const double *c, const double *d,
                          const double *e, const double *v, size_t stride, double *out)
{
    int k;
    for (k = 0; k < N; ++k) {
        double s = c[k] * v[(size_t)k * stride];
        if (k >= 1) s += b[k] * v[(size_t)(k - 1) * stride];
        if (k >= 2) s += a[k] * v[(size_t)(k - 2) * stride];
        if (k + 1 < N) s += d[k] * v[(size_t)(k + 1) * stride];
        if (k + 2 < N) s += e[k] * v[(size_t)(k + 2) * stride];
        out[k] = 2.0 * v[(size_t)k * stride] - s;
    }
}

/* dx, dy: 5*N diagonals (a,b,c,d,e) of A_x (N = Nx) and A_y (N = Ny); fx, fy: their 5*N factors
 * (eps,beta,alpha,gamma,delta) from pent_oracle_factor.  U: Ny x Nx, updated in place; W: Ny x Nx work array. */
void pent_oracle_adi_steps(int Nx, int Ny, const double *dx, const double *fx, const double *dy,
                           const double *fy, double *U, double *W, int nsteps, int nthreads)
{
    int s;
    (void)nthreads;
    for (s = 0; s < nsteps; ++s) {
        long x, y;
        /* half step 1, explicit part along y: W[:, x] = (2I - A_y) U[:, x] for every column x */
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
        for (x = 0; x < Nx; ++x) {
            double *col = (double *)malloc((size_t)Ny * sizeof(double));
            int k;
            two_i_minus_a(Ny, dy, dy + Ny, dy + 2 * Ny, dy + 3 * Ny, dy + 4 * Ny, U + x, (size_t)Nx, col);
            for (k = 0; k < Ny; ++k) W[(size_t)k * Nx + x] = col[k];
            free(col);
        }
        /* half step 1, implicit part along x: A_x U*[y, :] = W[y, :] for every row y; then the explicit
         * part of half step 2 along x: W[y, :] = (2I - A_x) U*[y, :] */
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
        for (y = 0; y < Ny; ++y) {
            double *row = U + (size_t)y * Nx;
            pent_oracle_solve(Nx, fx, fx + Nx, fx + 2 * Nx, fx + 3 * Nx, fx + 4 * Nx, W + (size_t)y * Nx, row);
            two_i_minus_a(Nx, dx, dx + Nx, dx + 2 * Nx, dx + 3 * Nx, dx + 4 * Nx, row, 1, W + (size_t)y * Nx);
        }
        /* half step 2, implicit part along y: A_y U[:, x] = W[:, x] for every column x */
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads > 0 ? nthreads : 1)
#endif
        for (x = 0; x < Nx; ++x) {
            double *col = (double *)malloc((size_t)2 * Ny * sizeof(double));
            int k;
            for (k = 0; k < Ny; ++k) col[k] = W[(size_t)k * Nx + x];
            pent_oracle_solve(Ny, fy, fy + Ny, fy + 2 * Ny, fy + 3 * Ny, fy + 4 * Ny, col, col + Ny);
            for (k = 0; k < Ny; ++k) U[(size_t)k * Nx + x] = col[Ny + k];
            free(col);
        }
    }
}
