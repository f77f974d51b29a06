// pent_step.cu -- fused time step: explicit right-hand side + pentadiagonal solve in ONE kernel
// (BASELINE.json configs[3]; the paper runs the RHS as a separate stencil kernel).
//
//  kind 0  Cahn-Hilliard, PAPER.md:53 (Eq. 2):  A c+ = c + r L (c^3 - c)           (form 0)
//          increment form:  q = r (c^3 - c) - sigma L c ;  A delta = L q ;  c+ = c + delta  (form 1)
//  kind 1  hyperdiffusion Crank-Nicolson, PAPER.md:87-89 (Eq. 6), :117 (Eq. 7c):  A c+ = (2I - A) c
//  L = second-difference matrix: (L v)_k = v_{k-1} + dg_k v_k + v_{k+1}, out-of-range terms
//  dropped, dg_k = -2 except dg_0 = dg_{N-1} = -1 when bc = 1 (zero-flux).
//
// This file: the thread-per-system version (one launch per step, 4 passes) used when the tile does
// not fit on chip; the default path is the on-chip kernel of pent_step_chunked.cu.  The state is read through a sliding window of rows held in
// registers (each c_k is loaded exactly once in the forward sweep), the right-hand side of
// row k is formed in registers and consumed at once by the forward recurrence; g goes to
// `scratch`; the back substitution writes the new state in place.
#include <cmath>
#include "pent_internal.h"

namespace pent {

template <typename T>
struct StepCoef {
    int kind, bc, form;
    T r, sigma;
    // forcing (reading C-22): rhs_k += dt mu1_i cos(2 pi (x_k - mu2_i t)); mu1 == nullptr: none
    const T* mu1;
    const T* mu2;
    double dt, t;
};

template <typename T>
__device__ __forceinline__ T Ldiag(int k, int N, int bc)
{
    return (bc == 1 && (k == 0 || k == N - 1)) ? (T)-1 : (T)-2;
}

template <typename T>
__global__ void __launch_bounds__(128)
step_tps_kernel(int N, int64_t M, const typename Vec<T>::T4* __restrict__ fw,
                const typename Vec<T>::T2* __restrict__ bw, const T* __restrict__ dgt,
                StepCoef<T> p, T* c, T* __restrict__ scratch)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    T* ci = c + i;
    T* gi = scratch + i;
    // window: cm2 = c_{k-2}, cm1 = c_{k-1}, c0 = c_k, cp1 = c_{k+1}, cp2 = c_{k+2}
    T cm2 = 0, cm1 = 0;
    T c0 = ci[0];
    T cp1 = (N > 1) ? ci[M] : (T)0;
    T cp2 = (N > 2) ? ci[2 * M] : (T)0;
    // kind 0 carries: w_{k-1}, w_k (form 0) or q_{k-1}, q_k (form 1)
    T um1 = 0, u0 = 0;
    if (p.kind == 0) {
        T w0 = c0 * c0 * c0 - c0;
        if (p.form == 0) u0 = w0;
        else u0 = fma(-p.sigma, fma(Ldiag<T>(0, N, p.bc), c0, cp1), p.r * w0);   // q_0
    }
    // forcing amplitudes of this system at this step: dt mu1 (cos, sin)(2 pi mu2 t); the space factors
    // cos / sin(2 pi x_k) sit in slots 5, 6 of the dg table
    T fa = 0, fb = 0;
    if (p.mu1) {
        double sn, cs;
        sincospi(2.0 * (double)p.mu2[i] * p.t, &sn, &cs);
        const double am = p.dt * (double)p.mu1[i];
        fa = (T)(am * cs); fb = (T)(am * sn);
    }
    T g1 = 0, g2 = 0;
    for (int k = 0; k < N; ++k) {
        T cn = (k + 3 < N) ? __ldcs(ci + (int64_t)(k + 3) * M) : (T)0;   // c_{k+3}, prefetch
        T rhs;
        if (p.kind == 1) {
            const T* dk = dgt + 8 * k;
            T s = __ldg(dk + 2) * c0;
            s = fma(__ldg(dk + 1), cm1, s);
            s = fma(__ldg(dk + 0), cm2, s);
            s = fma(__ldg(dk + 3), cp1, s);
            s = fma(__ldg(dk + 4), cp2, s);
            rhs = (T)2 * c0 - s;
        } else {
            // u_{k+1}: w_{k+1} or q_{k+1} (zero beyond the last row)
            T up1 = 0;
            if (k + 1 < N) {
                T w1 = cp1 * cp1 * cp1 - cp1;
                if (p.form == 0) up1 = w1;
                else up1 = fma(-p.sigma, c0 + fma(Ldiag<T>(k + 1, N, p.bc), cp1, cp2), p.r * w1);
            }
            T Lu = um1 + fma(Ldiag<T>(k, N, p.bc), u0, up1);
            rhs = (p.form == 0) ? fma(p.r, Lu, c0) : Lu;
            if (p.mu1) rhs = fma(fa, __ldg(dgt + 8 * k + 5), fma(fb, __ldg(dgt + 8 * k + 6), rhs));
            um1 = u0; u0 = up1;
        }
        typename Vec<T>::T4 cf = ldg4(fw + k);
        T g = fma(-cf.z, g1, fma(-cf.y, g2, cf.x * rhs));
        gi[(int64_t)k * M] = g;
        g2 = g1; g1 = g;
        cm2 = cm1; cm1 = c0; c0 = cp1; cp1 = cp2; cp2 = cn;
    }
    T x1 = 0, x2 = 0;
    const bool incr = (p.kind == 0 && p.form == 1);
    for (int k = N - 1; k >= 0; --k) {
        typename Vec<T>::T2 cb = ldg2(bw + k);
        T xv = fma(-cb.y, x2, fma(-cb.x, x1, gi[(int64_t)k * M]));
        T out = incr ? ci[(int64_t)k * M] + xv : xv;
        ci[(int64_t)k * M] = out;
        x2 = x1; x1 = xv;
    }
}

template <typename T>
static int step_impl(const pent_handle* h, const pent_step_params* p, const pent_forcing* fg, int64_t M, void* c,
                     void* scratch, int nsteps, cudaStream_t s)
{
    T* sc = (T*)scratch;
    bool own = false;
    if (!sc) {
        cudaError_t er = cudaMallocAsync((void**)&sc, (size_t)h->N * (size_t)M * sizeof(T), s);
        if (er == cudaErrorMemoryAllocation) { cudaGetLastError(); return PENT_ERR_ALLOC; }
        PENT_CUDA(er);
        own = true;
    }
    StepCoef<T> sp{p->kind, p->bc, p->form, (T)p->r, (T)p->sigma, nullptr, nullptr, 0.0, 0.0};
    if (fg && fg->kind == 1) { sp.mu1 = (const T*)fg->mu1; sp.mu2 = (const T*)fg->mu2; sp.dt = fg->dt; }
    const int tb = 128;
    unsigned nb = (unsigned)((M + tb - 1) / tb);
    cudaError_t le = cudaSuccess;
    for (int it = 0; it < nsteps && le == cudaSuccess; ++it) {
        if (sp.mu1) sp.t = fg->t0 + (double)it * fg->dt;
        step_tps_kernel<T><<<nb, tb, 0, s>>>(h->N, M, (const typename Vec<T>::T4*)h->fw,
                                             (const typename Vec<T>::T2*)h->bw, (const T*)h->dg,
                                             sp, (T*)c, sc);
        count_launch();
        le = cudaGetLastError();
    }
    if (own) cudaFreeAsync(sc, s);
    if (le != cudaSuccess) return cuda_fail(le);
    return PENT_OK;
}
}  // namespace pent

extern "C" int pent_step_batch_forced_v(const pent_handle* h, const pent_step_params* p, const pent_forcing* g,
                                        int64_t M, void* c_inout, void* scratch, int nsteps, void* stream, int kernel)
{
    if (!h || h->kind != 0 || !p || M < 0 || nsteps < 0 || !c_inout) return PENT_ERR_ARG;
    if (p->kind != 0 && p->kind != 1) return PENT_ERR_ARG;
    if (p->kind == 0 && ((p->bc != 0 && p->bc != 1) || (p->form != 0 && p->form != 1)))
        return PENT_ERR_ARG;
    if (kernel != PENT_KERNEL_AUTO && kernel != PENT_KERNEL_THREAD_PER_SYSTEM && kernel != PENT_KERNEL_CHUNKED)
        return PENT_ERR_ARG;
    if (g) {
        if (g->kind != 0 && g->kind != 1) return PENT_ERR_ARG;
        if (g->kind == 1 && (p->kind != 0 || !g->mu1 || !g->mu2)) return PENT_ERR_ARG;   // Eq. 3 forces Eq. 1 only
        if (g->kind == 0) g = nullptr;
    }
    if (M == 0 || nsteps == 0) return PENT_OK;
    if (!pent::on_handle_device(h)) return PENT_ERR_ARG;
    // the increment form is the scheme of Eq. 2 only if the handle's A IS I + sigma L^2 for this sigma and bc
    // (checked against what pent_factor detected; the direct form uses neither sigma nor the form of A)
    if (p->kind == 0 && p->form == 1) {
        const double tol = (h->dtype == PENT_F64 ? 1e-12 : 1e-6) * fabs(p->sigma);
        if (h->periodic || h->l2_bc != p->bc || !(fabs(h->l2_sigma - p->sigma) <= tol)) return PENT_ERR_ARG;
    }
    cudaStream_t s = (cudaStream_t)stream;
    if (h->periodic) {       // the paper's own loop: periodic hyperdiffusion, Eq. 6 / 7c
        if (p->kind != 1 || kernel != PENT_KERNEL_AUTO) return PENT_ERR_ARG;
        return pent::step_periodic(h, M, c_inout, scratch, nsteps, s);
    }
    const bool on_chip = pent::step_chunked_supported(h, M, c_inout);
    if (kernel == PENT_KERNEL_CHUNKED && !on_chip) return PENT_ERR_ARG;
    if (kernel != PENT_KERNEL_THREAD_PER_SYSTEM && on_chip)
        return pent::launch_step_chunked(h, p, g, M, c_inout, nsteps, s);
    // Crank-Nicolson hyperdiffusion whose state does not fit on chip (N > 1024): A c+ = (2I - A) c  <=>  c+ = 2 A^{-1} c - c,
    // i.e. ONE chunked solve with the "2x - f" epilogue per step, in place: 2 passes over the state per step instead of the
    // 4 passes of the thread-per-system step kernel (pent_solve_chunked_epi.cu; pentadiagonal tables)
    if (kernel == PENT_KERNEL_AUTO && p->kind == 1) {
        int rc = PENT_OK;
        for (int it = 0; it < nsteps && rc == PENT_OK; ++it) {
            rc = pent::launch_solve_chunked_epi(h, M, c_inout, c_inout, s);
            if (rc == pent::PENT_UNSUPPORTED && it > 0) rc = PENT_ERR_ARG;      // (cannot happen: the plan does not depend on the step)
        }
        if (rc != pent::PENT_UNSUPPORTED) return rc;
    }
    if (h->dtype == PENT_F64) return pent::step_impl<double>(h, p, g, M, c_inout, scratch, nsteps, s);
    return pent::step_impl<float>(h, p, g, M, c_inout, scratch, nsteps, s);
}

extern "C" int pent_step_batch_forced(const pent_handle* h, const pent_step_params* p, const pent_forcing* g,
                                      int64_t M, void* c_inout, void* scratch, int nsteps, void* stream)
{
    return pent_step_batch_forced_v(h, p, g, M, c_inout, scratch, nsteps, stream, PENT_KERNEL_AUTO);
}

extern "C" int pent_step_batch_v(const pent_handle* h, const pent_step_params* p, int64_t M,
                                 void* c_inout, void* scratch, int nsteps, void* stream, int kernel)
{
    return pent_step_batch_forced_v(h, p, nullptr, M, c_inout, scratch, nsteps, stream, kernel);
}

extern "C" int pent_step_batch(const pent_handle* h, const pent_step_params* p, int64_t M,
                               void* c_inout, void* scratch, int nsteps, void* stream)
{
    return pent_step_batch_forced_v(h, p, nullptr, M, c_inout, scratch, nsteps, stream, PENT_KERNEL_AUTO);
}

extern "C" int pent_step_kernel_choice(const pent_handle* h, int64_t M)
{
    if (!h || h->kind != 0) return -1;
    if (h->periodic) return pent::step_chunked_periodic_supported(h, M, nullptr) ? PENT_KERNEL_CHUNKED : PENT_KERNEL_THREAD_PER_SYSTEM;
    return pent::step_chunked_supported(h, M, nullptr) ? PENT_KERNEL_CHUNKED : PENT_KERNEL_THREAD_PER_SYSTEM;
}
