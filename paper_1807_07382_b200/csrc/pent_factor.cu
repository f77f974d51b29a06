// pent_factor.cu -- shared-A factorisation A = L R on the device and the
// derived, sweep-ready coefficient tables kept in the handle.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include "pent_internal.h"

namespace pent {
thread_local int g_last_cuda_error = 0;
thread_local int64_t g_launches = 0;

// Widen the caller's diagonals to fp64 and zero the entries that lie outside the matrix
// (they are never read from the caller's arrays: include/pent.h).  layout out: a,b,c,d,e.
template <typename T>
__global__ void widen_diagonals(int N, const T* __restrict__ a, const T* __restrict__ b,
                                const T* __restrict__ c, const T* __restrict__ d,
                                const T* __restrict__ e, double* __restrict__ out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    out[0 * N + k] = (k >= 2) ? (double)a[k] : 0.0;
    out[1 * N + k] = (k >= 1) ? (double)b[k] : 0.0;
    out[2 * N + k] = (double)c[k];
    out[3 * N + k] = (k + 1 < N) ? (double)d[k] : 0.0;
    out[4 * N + k] = (k + 2 < N) ? (double)e[k] : 0.0;
}

// The factor recurrence is strictly serial in k: one thread.  With out-of-matrix entries
// zeroed, the paper's steps 1-14 are the single recurrence (steps 8.1-8.4)
//   beta_k = b_k - a_k gamma_{k-2};  alpha_k = c_k - a_k delta_{k-2} - beta_k gamma_{k-1};
//   gamma_k = (d_k - beta_k delta_{k-1}) / alpha_k;  delta_k = e_k / alpha_k;  eps_k = a_k
// evaluated for k = 0..N-1 with gamma_{-1} = gamma_{-2} = delta_{-1} = delta_{-2} = 0.
// No FMA contraction here (__dmul_rn/__dsub_rn): same rounding as a plain C evaluation.
// status[0] = -1, or the first row with a zero / non-finite pivot.
__global__ void factor_shared(int N, const double* __restrict__ dg, double* __restrict__ fac,
                              int* __restrict__ status)
{
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    const double *a = dg, *b = dg + N, *c = dg + 2 * N, *d = dg + 3 * N, *e = dg + 4 * N;
    double *eps = fac, *beta = fac + N, *alpha = fac + 2 * N, *gamma = fac + 3 * N,
           *delta = fac + 4 * N;
    double g1 = 0.0, g2 = 0.0, d1 = 0.0, d2 = 0.0;   // gamma_{k-1}, gamma_{k-2}, delta_{k-1}, delta_{k-2}
    int bad = -1;
    for (int k = 0; k < N; ++k) {
        double ak = a[k];
        double be = __dsub_rn(b[k], __dmul_rn(ak, g2));
        double al = __dsub_rn(__dsub_rn(c[k], __dmul_rn(ak, d2)), __dmul_rn(be, g1));
        if (bad < 0 && (al == 0.0 || !isfinite(al))) bad = k;
        double ga = __ddiv_rn(__dsub_rn(d[k], __dmul_rn(be, d1)), al);
        double de = __ddiv_rn(e[k], al);
        eps[k] = ak; beta[k] = be; alpha[k] = al; gamma[k] = ga; delta[k] = de;
        g2 = g1; g1 = ga; d2 = d1; d1 = de;
    }
    status[0] = bad;
}

// Sweep-ready tables (one thread per row):
//   fw[k] = {1/alpha, eps/alpha, beta/alpha, 0}:  g_k = fw.x f_k - fw.y g_{k-2} - fw.z g_{k-1}
//   bw[k] = {gamma, delta}:                        x_k = g_k - bw.x x_{k+1} - bw.y x_{k+2}
//   dgT[k] = {a,b,c,d,e, cos(2 pi x_k), sin(2 pi x_k), 0} in T: the original diagonals (for the (2I-A)c
//            right-hand side) and the space factors of the travelling-wave forcing at x_k = (k + 1/2)/N
// All divisions of the solve are done here, once (fp64 division is a long software sequence
// on the GPU); the per-unknown work of the sweeps is then 1 mul + 4 fma.
template <typename T>
__global__ void derive_tables(int N, const double* __restrict__ dg, const double* __restrict__ fac,
                              typename Vec<T>::T4* __restrict__ fw,
                              typename Vec<T>::T2* __restrict__ bw, T* __restrict__ dgT)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    double al = fac[2 * N + k];
    typename Vec<T>::T4 w;
    w.x = (T)(1.0 / al); w.y = (T)(fac[k] / al); w.z = (T)(fac[N + k] / al); w.w = (T)0;
    fw[k] = w;
    typename Vec<T>::T2 v;
    v.x = (T)fac[3 * N + k]; v.y = (T)fac[4 * N + k];
    bw[k] = v;
    for (int j = 0; j < 5; ++j) dgT[8 * k + j] = (T)dg[j * N + k];
    double sx, cx;
    sincospi((2.0 * k + 1.0) / (double)N, &sx, &cx);
    dgT[8 * k + 5] = (T)cx; dgT[8 * k + 6] = (T)sx; dgT[8 * k + 7] = (T)0;
}

int build_chunk_tables(pent_handle* h, cudaStream_t s);   // pent_solve_chunked.cu

static bool is_device_ptr(const void* p)
{
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// Is the matrix I + sigma L^2 for the second-difference matrix L with boundary bc (0 Dirichlet, 1 zero-flux)?
// (L^2)[k][k] = dg_k^2 + [k > 0] + [k < N-1], (L^2)[k][k+-1] = dg_k + dg_{k+-1}, (L^2)[k][k+-2] = 1, with
// dg = -2 except dg_0 = dg_{N-1} = -1 for bc = 1.  dg5 = the widened diagonals a,b,c,d,e (host copy).
// tol: relative, on the scale of 1 + 6 sigma (fp32 handles hold rounded entries).
static void detect_l2_form(pent_handle* h, const double* dg5, double tol)
{
    const int N = h->N;
    h->l2_bc = -1; h->l2_sigma = 0.0;
    if (N < 3) return;
    const double* a = dg5; const double* b = dg5 + N; const double* c = dg5 + 2 * (size_t)N;
    const double* d = dg5 + 3 * (size_t)N; const double* e = dg5 + 4 * (size_t)N;
    const double sigma = a[2];
    if (!(sigma > 0.0)) return;
    const double scale = tol * (1.0 + 6.0 * sigma);
    for (int bc = 0; bc < 2; ++bc) {
        auto dgL = [&](int k) { return (bc == 1 && (k == 0 || k == N - 1)) ? -1.0 : -2.0; };
        bool ok = true;
        for (int k = 0; k < N && ok; ++k) {
            const double cc = 1.0 + sigma * (dgL(k) * dgL(k) + (k > 0 ? 1.0 : 0.0) + (k < N - 1 ? 1.0 : 0.0));
            ok = fabs(c[k] - cc) <= scale;
            if (ok && k >= 1) ok = fabs(b[k] - sigma * (dgL(k) + dgL(k - 1))) <= scale;
            if (ok && k + 1 < N) ok = fabs(d[k] - sigma * (dgL(k) + dgL(k + 1))) <= scale;
            if (ok && k >= 2) ok = fabs(a[k] - sigma) <= scale;
            if (ok && k + 2 < N) ok = fabs(e[k] - sigma) <= scale;
        }
        if (ok) { h->l2_bc = bc; h->l2_sigma = sigma; return; }
    }
}

// Everything on the PRIVATE stream `s` (non-blocking): no other stream of the process is stalled, and the
// host waits for `s` only.  Temporaries are stream-ordered allocations on `s`.
template <typename T>
int factor_on_stream(int N, const void* const src[5], pent_dtype dtype, pent_handle** out, int* bad_row,
                     cudaStream_t s)
{
    pent_handle* h = new (std::nothrow) pent_handle();
    if (!h) return PENT_ERR_ALLOC;
    std::memset(h, 0, sizeof(*h));
    h->kind = 0; h->N = N; h->dtype = dtype; h->l2_bc = -1; h->band = 2;
    if (cudaGetDevice(&h->device) != cudaSuccess) { delete h; return cuda_fail(cudaGetLastError()); }
    T* stage = nullptr;
    int* status = nullptr;
    double* hostdg = (double*)std::malloc(sizeof(double) * 5 * (size_t)N);
    int rc = PENT_OK;
    auto fail = [&](int code) {
        if (stage) cudaFreeAsync(stage, s);
        if (status) cudaFreeAsync(status, s);
        cudaStreamSynchronize(s);
        std::free(hostdg);
        pent_destroy(h);
        return code;
    };
    if (!hostdg) return fail(PENT_ERR_ALLOC);
    auto chk = [&](cudaError_t e) { if (e != cudaSuccess) { rc = cuda_fail(e); return false; } return true; };
    auto alloc = [&](void** p, size_t bytes) {
        cudaError_t e = cudaMalloc(p, bytes);
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); rc = PENT_ERR_ALLOC; return false; }
        return chk(e);
    };
    auto alloc_tmp = [&](void** p, size_t bytes) {
        cudaError_t e = cudaMallocAsync(p, bytes, s);
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); rc = PENT_ERR_ALLOC; return false; }
        return chk(e);
    };
    if (!alloc_tmp((void**)&stage, sizeof(T) * 5 * (size_t)N) || !alloc_tmp((void**)&status, 2 * sizeof(int)) ||
        !alloc((void**)&h->diag, sizeof(double) * 5 * (size_t)N) ||
        !alloc((void**)&h->fac, sizeof(double) * 5 * (size_t)N) ||
        !alloc(&h->fw, sizeof(T) * 4 * (size_t)N) || !alloc(&h->bw, sizeof(T) * 2 * (size_t)N) ||
        !alloc(&h->dg, sizeof(T) * 8 * (size_t)N))
        return fail(rc);

    // order of src: a, b, c, d, e
    for (int j = 0; j < 5; ++j) {
        cudaMemcpyKind kind = is_device_ptr(src[j]) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        if (!chk(cudaMemcpyAsync(stage + (size_t)j * N, src[j], sizeof(T) * (size_t)N, kind, s))) return fail(rc);
    }
    int tb = 128, nb = (N + tb - 1) / tb;
    widen_diagonals<T><<<nb, tb, 0, s>>>(N, stage, stage + N, stage + 2 * (size_t)N, stage + 3 * (size_t)N,
                                         stage + 4 * (size_t)N, h->diag);
    factor_shared<<<1, 32, 0, s>>>(N, h->diag, h->fac, status);
    derive_tables<T><<<nb, tb, 0, s>>>(N, h->diag, h->fac, (typename Vec<T>::T4*)h->fw,
                                       (typename Vec<T>::T2*)h->bw, (T*)h->dg);
    count_launch(3);
    if (!chk(cudaGetLastError())) return fail(rc);
    int bad = -1;
    if (!chk(cudaMemcpyAsync(&bad, status, sizeof(int), cudaMemcpyDeviceToHost, s)) ||
        !chk(cudaMemcpyAsync(hostdg, h->diag, sizeof(double) * 5 * (size_t)N, cudaMemcpyDeviceToHost, s)) ||
        !chk(cudaStreamSynchronize(s)))
        return fail(rc);
    if (bad_row) *bad_row = bad;
    if (bad >= 0) return fail(PENT_ERR_PIVOT);
    detect_l2_form(h, hostdg, sizeof(T) == 8 ? 1e-13 : 1e-6);
    {   // tridiagonal matrix (a == e == 0 inside the matrix)?  cuThomasBatch's case
        bool tri = true;
        for (int k = 0; k < N && tri; ++k) tri = hostdg[k] == 0.0 && hostdg[4 * (size_t)N + k] == 0.0;
        h->band = (tri && !std::getenv("PENT_AB_NO_TRI")) ? 1 : 2;   // A/B: run a tridiagonal A through the BAND = 2 kernel
    }
    rc = build_chunk_tables(h, s);
    if (rc != PENT_OK) return fail(rc);
    cudaFreeAsync(stage, s); cudaFreeAsync(status, s);
    stage = nullptr; status = nullptr;
    if (!chk(cudaStreamSynchronize(s))) return fail(rc);
    std::free(hostdg);
    *out = h;
    return PENT_OK;
}
template int factor_on_stream<double>(int, const void* const*, pent_dtype, pent_handle**, int*, cudaStream_t);
template int factor_on_stream<float>(int, const void* const*, pent_dtype, pent_handle**, int*, cudaStream_t);
}  // namespace pent

// ------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------
extern "C" int pent_factor(int N, const void* e, const void* c, const void* d, const void* a,
                           const void* b, pent_dtype dtype, pent_handle** out, int* bad_row)
{
    if (bad_row) *bad_row = -1;
    if (!out) return PENT_ERR_ARG;
    *out = nullptr;
    if (N < 1 || !e || !c || !d || !a || !b) return PENT_ERR_ARG;
    if (dtype != PENT_F64 && dtype != PENT_F32) return PENT_ERR_ARG;
    const void* src[5] = {a, b, c, d, e};
    cudaStream_t s = nullptr;
    PENT_CUDA(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
    const int rc = dtype == PENT_F64 ? pent::factor_on_stream<double>(N, src, dtype, out, bad_row, s)
                                     : pent::factor_on_stream<float>(N, src, dtype, out, bad_row, s);
    cudaStreamDestroy(s);
    return rc;
}

extern "C" void pent_destroy(pent_handle* h)
{
    if (!h) return;
    cudaFree(h->diag); cudaFree(h->fac); cudaFree(h->fw); cudaFree(h->bw);
    for (int j = 0; j < PENT_NQ; ++j) { cudaFree(h->cf[j]); cudaFree(h->cf1[j]); }
    cudaFree(h->dg); cudaFree(h->ms); cudaFree(h->Zt); cudaFree(h->dgp); cudaFree(h->pfold); cudaFree(h->pzedge);
    pent_destroy(h->inner);
    delete h;
}

extern "C" int pent_handle_n(const pent_handle* h) { return h ? h->N : -1; }
extern "C" int pent_handle_dtype(const pent_handle* h) { return h ? (int)h->dtype : -1; }
extern "C" int64_t pent_handle_m(const pent_handle* h) { return h ? h->M : -1; }
extern "C" int pent_handle_device(const pent_handle* h) { return h ? h->device : -1; }
extern "C" int pent_handle_growth(const pent_handle* h, double* out3)
{
    if (!h || h->kind != 0 || !out3) return PENT_ERR_ARG;
    const pent_handle* g = h->periodic ? h->inner : h;
    for (int j = 0; j < 3; ++j) out3[j] = g->growth[j];
    return PENT_OK;
}
extern "C" int pent_handle_band(const pent_handle* h) { return (h && h->kind == 0) ? (h->periodic ? 2 : h->band) : -1; }
extern "C" int pent_handle_exchange_depth(const pent_handle* h, int Q)
{
    if (!h || h->kind != 0) return -1;
    if (h->periodic) return pent_handle_exchange_depth(h->inner, Q) < 0 ? -1 : (Q > 1 ? Q - 1 : 1);   // the fused periodic kernel exchanges with every rank
    int j = 0;
    while ((1 << j) < Q) ++j;
    if ((1 << j) != Q || j >= PENT_NQ || !h->cf[j]) return -1;
    return h->band == 1 ? h->xdepth1[j] : h->xdepth[j];
}

extern "C" int pent_handle_factors(const pent_handle* h, double* eps, double* beta, double* alpha,
                                   double* gamma, double* delta)
{
    if (!h || h->kind != 0 || !pent::on_handle_device(h)) return PENT_ERR_ARG;
    if (h->periodic) return pent_handle_factors(h->inner, eps, beta, alpha, gamma, delta);   // factors of E
    double* dst[5] = {eps, beta, alpha, gamma, delta};
    for (int j = 0; j < 5; ++j)
        if (dst[j])
            PENT_CUDA(cudaMemcpy(dst[j], h->fac + (size_t)j * h->N, sizeof(double) * h->N,
                                 cudaMemcpyDeviceToHost));
    return PENT_OK;
}

extern "C" int pent_last_cuda_error(void) { return pent::g_last_cuda_error; }

extern "C" int64_t pent_launch_count(int reset)
{
    int64_t v = pent::g_launches;
    if (reset) pent::g_launches = 0;
    return v;
}

extern "C" int pent_handle_periodic(const pent_handle* h) { return h ? h->periodic : -1; }

extern "C" const char* pent_version(void) { return "pent 0.3 (sm_100a)"; }
