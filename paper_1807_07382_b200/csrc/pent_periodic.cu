// pent_periodic.cu -- periodic (cyclic) pentadiagonal systems, section II.C (Eqs. 7a-12):
// the matrix the paper actually benchmarks.  Reduction (the paper takes it from Navon): strip the
// last two rows and columns,
//     E X^ + k t = f^,      h^T X^ + C2 t = (f_{N-2}, f_{N-1})^T,      t = (x_{N-2}, x_{N-1})^T
// (0-based; Eq. 10).  Set-up, once per handle: factor E (the shared-A path of pent_factor),
// Z = E^{-1} k (two fp64 solves), S2 = C2 - h^T Z and its inverse ("computed and
// stored at the start").  Per batch:
//     y = E^{-1} f^                          the chunked solve kernel on the first N-2 rows
//     t = S2^{-1} [ (f_{N-2}, f_{N-1}) - h^T y ]      h has six non-zero entries (Eq. 9)
//     X^ = y - Z t                           rank-2 update
// which is Eq. 11-12 with E^{-1} applied to f^ first: h^T E^{-1} f^ = h^T y, E^{-1} k = Z.
// In the interleaved layout the first N-2 rows of a batch ARE an interleaved (N-2) x M batch,
// so the inner solve needs no copy.
#include <cstdlib>
#include <new>
#include "pent_chunk_common.cuh"

namespace pent {

// thread j < 2: z_j = E^{-1} k_j by the paper's sweeps (true divisions, fp64); then thread 0:
// S2 = C2 - h^T Z, out[0..5] = h entries, out[6..9] = S2^{-1} row-major, status = 0 / 1 (singular)
// G (2 x n): the forward-sweep intermediates g = L^{-1} k of the two solves (the chunk states of the Z solve, needed by
// the on-chip periodic time step)
__global__ void periodic_setup_kernel(int N, const double* __restrict__ fac, const double* __restrict__ dg,
                                      double* __restrict__ Z, double* __restrict__ G, double* __restrict__ out,
                                      int* __restrict__ status)
{
    const int n = N - 2, j = threadIdx.x;
    const double *a = dg, *b = dg + N, *c = dg + 2 * N, *d = dg + 3 * N, *e = dg + 4 * N;
    const double *eps = fac, *beta = fac + n, *alpha = fac + 2 * n, *gamma = fac + 3 * n, *delta = fac + 4 * n;
    if (j < 2) {
        double* z = Z + (size_t)j * n;
        // k (Eq. 9): column j = column N-2+j of A restricted to rows 0..N-3
        for (int i = 0; i < n; ++i) z[i] = 0.0;
        if (j == 0) { z[0] = a[0]; z[n - 2] = e[N - 4]; z[n - 1] = d[N - 3]; }
        else        { z[0] = b[0]; z[1] += a[1]; z[n - 1] = e[N - 3]; }
        double g1 = 0.0, g2 = 0.0;
        for (int i = 0; i < n; ++i) {
            double g = __ddiv_rn(z[i] - eps[i] * g2 - beta[i] * g1, alpha[i]);
            z[i] = g; G[(size_t)j * n + i] = g; g2 = g1; g1 = g;
        }
        double x1 = 0.0, x2 = 0.0;
        for (int i = n - 1; i >= 0; --i) {
            double xv = z[i] - gamma[i] * x1 - delta[i] * x2;
            z[i] = xv; x2 = x1; x1 = xv;
        }
    }
    __syncthreads();
    if (j == 0) {
        const double h00 = e[N - 2], h0a = a[N - 2], h0b = b[N - 2];      // row N-2: cols 0, N-4, N-3
        const double h10 = d[N - 1], h11 = e[N - 1], h1a = a[N - 1];      // row N-1: cols 0, 1,   N-3
        const double *z0 = Z, *z1 = Z + n;
        double s00 = c[N - 2] - (h00 * z0[0] + h0a * z0[n - 2] + h0b * z0[n - 1]);
        double s01 = d[N - 2] - (h00 * z1[0] + h0a * z1[n - 2] + h0b * z1[n - 1]);
        double s10 = b[N - 1] - (h10 * z0[0] + h11 * z0[1] + h1a * z0[n - 1]);
        double s11 = c[N - 1] - (h10 * z1[0] + h11 * z1[1] + h1a * z1[n - 1]);
        double det = s00 * s11 - s01 * s10;
        status[0] = (det == 0.0 || !isfinite(det)) ? 1 : 0;
        out[0] = h00; out[1] = h0a; out[2] = h0b; out[3] = h10; out[4] = h11; out[5] = h1a;
        out[6] = s11 / det; out[7] = -s01 / det; out[8] = -s10 / det; out[9] = s00 / det;
    }
}

template <typename T>
__global__ void periodic_tables_kernel(int N, const T* __restrict__ stage, const double* __restrict__ Z,
                                       typename Vec<T>::T2* __restrict__ Zt, T* __restrict__ dgp,
                                       double* __restrict__ dg64)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int n = N - 2;
    for (int j = 0; j < 5; ++j) {
        T v = stage[(size_t)j * N + k];
        dgp[8 * (size_t)k + j] = v;
        if (dg64) dg64[(size_t)j * N + k] = (double)v;
    }
    for (int j = 5; j < 8; ++j) dgp[8 * (size_t)k + j] = (T)0;
    if (Z && k < n) { typename Vec<T>::T2 z; z.x = (T)Z[k]; z.y = (T)Z[n + k]; Zt[k] = z; }
}

// x^ = y - Z t without the rows of Z in shared memory (the fused periodic solve and the on-chip periodic time step).
// Inside a chunk that holds no non-zero row of k, Z is a homogeneous solution of the two recurrences,
// Z_rows = chi F^Z_{p-1} + psi B^Z_{p+1}, so  y - Z t  is the usual correction with the chunk states F - F^Z t, B - B^Z t.
// fold[p] = {g^Z_0, g^Z_1 of row s-2 | of row s-1 | Z_0, Z_1 of row e+1 | of row e+2} (s = pC, e = s+C-1; zero outside
// 0..n-1).  The chunks that hold the non-zero rows of k (rows 0, 1 and n-2, n-1: chunk 0 and the chunks of rows n-2 and
// n-1) get fold = 0 and subtract their explicit rows of Z instead: zedge[0] = chunk 0, zedge[1] = the chunk of row n-2,
// zedge[2] = the chunk of row n-1 (C rows x {z0, z1} each).  Pt >= the number of chunks: entries beyond it are zero.
template <typename T>
__global__ void periodic_fold_kernel(int n, int Pt, const double* __restrict__ Z, const double* __restrict__ G,
                                     T* __restrict__ fold, typename Vec<T>::T2* __restrict__ zedge)
{
    constexpr int C = ChunkCfg<T>::C;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int ga = (n - 2) / C, gb = (n - 1) / C;
    if (p < Pt) {
        const int s = p * C, e = s + C - 1;
        const bool edge = p == 0 || p == ga || p == gb || s >= n;
        auto at = [&](const double* v, int col, int k) -> T { return (!edge && k >= 0 && k < n) ? (T)v[(size_t)col * n + k] : (T)0; };
        T* o = fold + 8 * (size_t)p;
        o[0] = at(G, 0, s - 2); o[1] = at(G, 1, s - 2); o[2] = at(G, 0, s - 1); o[3] = at(G, 1, s - 1);
        o[4] = at(Z, 0, e + 1); o[5] = at(Z, 1, e + 1); o[6] = at(Z, 0, e + 2); o[7] = at(Z, 1, e + 2);
    }
    if (p < 3 * C) {
        const int which = p / C, j = p % C, k = (which == 0 ? 0 : which == 1 ? ga : gb) * C + j;
        typename Vec<T>::T2 z;
        z.x = k < n ? (T)Z[k] : (T)0;
        z.y = k < n ? (T)Z[(size_t)n + k] : (T)0;
        zedge[p] = z;
    }
}

template <typename T>
struct PeriodicCoef { T h00, h0a, h0b, h10, h11, h1a, i00, i01, i10, i11; };

// t = S2^{-1} [ (f_{N-2}, f_{N-1}) - h^T y ]; one thread per system; y is in x (rows 0..N-3)
template <typename T>
__global__ void periodic_tail_kernel(int N, int64_t M, PeriodicCoef<T> pc, const T* f, T* x)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    const T y0 = x[i], y1 = x[M + i], ya = x[(int64_t)(N - 4) * M + i], yb = x[(int64_t)(N - 3) * M + i];
    const T r0 = f[(int64_t)(N - 2) * M + i] - fma(pc.h0b, yb, fma(pc.h0a, ya, pc.h00 * y0));
    const T r1 = f[(int64_t)(N - 1) * M + i] - fma(pc.h1a, yb, fma(pc.h11, y1, pc.h10 * y0));
    x[(int64_t)(N - 2) * M + i] = fma(pc.i01, r1, pc.i00 * r0);
    x[(int64_t)(N - 1) * M + i] = fma(pc.i11, r1, pc.i10 * r0);
}

// X^ = y - Z t, in place on rows 0..N-3; a block covers ROWS rows x blockDim.x systems
template <typename T, int ROWS>
__global__ void periodic_update_kernel(int N, int64_t M, const typename Vec<T>::T2* __restrict__ Zt, T* x)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    const int n = N - 2, k0 = blockIdx.y * ROWS;
    const T t0 = x[(int64_t)(N - 2) * M + i], t1 = x[(int64_t)(N - 1) * M + i];
    T v[ROWS];
#pragma unroll
    for (int r = 0; r < ROWS; ++r) v[r] = (k0 + r < n) ? __ldcs(x + (int64_t)(k0 + r) * M + i) : (T)0;
#pragma unroll
    for (int r = 0; r < ROWS; ++r)
        if (k0 + r < n) {
            typename Vec<T>::T2 z = ldg2(Zt + k0 + r);
            x[(int64_t)(k0 + r) * M + i] = fma(-z.y, t1, fma(-z.x, t0, v[r]));
        }
}

// out = (2I - A) c with the cyclic A (Eq. 7c); a block covers ROWS rows x blockDim.x systems
template <typename T, int ROWS>
__global__ void periodic_rhs_kernel(int N, int64_t M, const T* __restrict__ dgp, const T* __restrict__ c,
                                    T* __restrict__ out)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    const int k0 = blockIdx.y * ROWS;
    auto ld = [&](int k) -> T { k = k < 0 ? k + N : (k >= N ? k - N : k); return c[(int64_t)k * M + i]; };
    T w[ROWS + 4];
#pragma unroll
    for (int r = 0; r < ROWS + 4; ++r) w[r] = (k0 + r - 2 < N + 2) ? ld(k0 + r - 2) : (T)0;
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
        const int k = k0 + r;
        if (k < N) {
            const T* dk = dgp + 8 * (size_t)k;
            T s = __ldg(dk + 2) * w[r + 2];
            s = fma(__ldg(dk + 1), w[r + 1], s);
            s = fma(__ldg(dk + 0), w[r], s);
            s = fma(__ldg(dk + 3), w[r + 3], s);
            s = fma(__ldg(dk + 4), w[r + 4], s);
            out[(int64_t)k * M + i] = (T)2 * w[r + 2] - s;
        }
    }
}

template <typename T>
static PeriodicCoef<T> coef_of(const pent_handle* h)
{
    PeriodicCoef<T> pc;
    pc.h00 = (T)h->pc[0]; pc.h0a = (T)h->pc[1]; pc.h0b = (T)h->pc[2];
    pc.h10 = (T)h->pc[3]; pc.h11 = (T)h->pc[4]; pc.h1a = (T)h->pc[5];
    pc.i00 = (T)h->pc[6]; pc.i01 = (T)h->pc[7]; pc.i10 = (T)h->pc[8]; pc.i11 = (T)h->pc[9];
    return pc;
}

template <typename T>
static int solve_periodic_t(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s, int kernel)
{
    if (kernel == PENT_KERNEL_AUTO && periodic_fused_supported(h, M, f)) {
        const int rc = launch_solve_chunked_periodic(h, M, f, x, s);  // one kernel, 2 passes
        if (rc != PENT_UNSUPPORTED) return rc;                         // (cluster size not schedulable on this device: unfused)
    }
    if ((kernel & 0xff) == PENT_KERNEL_CHUNKED && kernel != PENT_KERNEL_CHUNKED) return PENT_ERR_ARG;
    // unfused: inner solve (chunked when kernel == PENT_KERNEL_CHUNKED or AUTO) + tail + rank-2 update
    int rc = pent_solve_batch_v(h->inner, M, f, x, (void*)s, kernel == PENT_KERNEL_CHUNKED ? PENT_KERNEL_AUTO : kernel);
    if (rc != PENT_OK) return rc;
    const int tb = 128;
    const unsigned nb = (unsigned)((M + tb - 1) / tb);
    periodic_tail_kernel<T><<<nb, tb, 0, s>>>(h->N, M, coef_of<T>(h), (const T*)f, (T*)x);
    constexpr int ROWS = 8;
    dim3 grid(nb, (unsigned)((h->N - 2 + ROWS - 1) / ROWS));
    periodic_update_kernel<T, ROWS><<<grid, tb, 0, s>>>(h->N, M, (const typename Vec<T>::T2*)h->Zt, (T*)x);
    count_launch(2);
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}

int solve_periodic(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s, int kernel)
{
    if (h->dtype == PENT_F64) return solve_periodic_t<double>(h, M, f, x, s, kernel);
    return solve_periodic_t<float>(h, M, f, x, s, kernel);
}

template <typename T>
static int step_periodic_t(const pent_handle* h, int64_t M, void* c, void* scratch, int nsteps, cudaStream_t s)
{
    T* sc = (T*)scratch;
    bool own = false;
    if (!sc) {
        cudaError_t er = cudaMallocAsync((void**)&sc, (size_t)h->N * (size_t)M * sizeof(T), s);
        if (er == cudaErrorMemoryAllocation) { cudaGetLastError(); return PENT_ERR_ALLOC; }
        PENT_CUDA(er);
        own = true;
    }
    const int tb = 128;
    constexpr int ROWS = 8;
    dim3 grid((unsigned)((M + tb - 1) / tb), (unsigned)((h->N + ROWS - 1) / ROWS));
    int rc = PENT_OK;
    for (int it = 0; it < nsteps && rc == PENT_OK; ++it) {
        periodic_rhs_kernel<T, ROWS><<<grid, tb, 0, s>>>(h->N, M, (const T*)h->dgp, (const T*)c, sc);
        count_launch();
        cudaError_t le = cudaGetLastError();
        if (le != cudaSuccess) { rc = cuda_fail(le); break; }
        rc = solve_periodic_t<T>(h, M, sc, c, s, PENT_KERNEL_AUTO);
    }
    if (own) cudaFreeAsync(sc, s);
    return rc;
}

int step_periodic(const pent_handle* h, int64_t M, void* c, void* scratch, int nsteps, cudaStream_t s)
{
    // default: the whole loop in ONE launch with the state on chip (pent_step_chunked.cu); otherwise one right-hand-side
    // kernel and one fused periodic solve per step
    static const int two_kernels = []() { const char* e = std::getenv("PENT_AB_PERIODIC_STEP_UNFUSED"); return e ? std::atoi(e) : 0; }();
    if (!two_kernels && step_chunked_periodic_supported(h, M, c)) return launch_step_chunked_periodic(h, M, c, nsteps, s);
    if (h->dtype == PENT_F64) return step_periodic_t<double>(h, M, c, scratch, nsteps, s);
    return step_periodic_t<float>(h, M, c, scratch, nsteps, s);
}

static bool is_dev(const void* p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

template <typename T>
static int factor_periodic_t(int N, const void* const src[5], pent_dtype dtype, pent_handle** out, int* bad_row,
                             cudaStream_t s)
{
    // Everything runs on the private non-blocking stream `s`; temporaries are stream-ordered allocations.
    const int n = N - 2;
    T* stage = nullptr;
    double *dg64 = nullptr, *Z = nullptr, *G = nullptr, *coef = nullptr;
    int* status = nullptr;
    pent_handle* h = new (std::nothrow) pent_handle();
    if (!h) return PENT_ERR_ALLOC;
    *h = pent_handle{};
    h->kind = 0; h->periodic = 1; h->N = N; h->dtype = dtype; h->l2_bc = -1; h->band = 2;
    if (cudaGetDevice(&h->device) != cudaSuccess) { delete h; return cuda_fail(cudaGetLastError()); }
    int rc = PENT_OK;
    auto done = [&](int code) {
        if (stage) cudaFreeAsync(stage, s);
        if (dg64) cudaFreeAsync(dg64, s);
        if (Z) cudaFreeAsync(Z, s);
        if (G) cudaFreeAsync(G, s);
        if (coef) cudaFreeAsync(coef, s);
        if (status) cudaFreeAsync(status, s);
        cudaStreamSynchronize(s);
        if (code != PENT_OK) pent_destroy(h);
        return code;
    };
    auto alloc = [&](void** p, size_t bytes) {
        cudaError_t e = cudaMalloc(p, bytes);
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); rc = PENT_ERR_ALLOC; return false; }
        if (e != cudaSuccess) { rc = cuda_fail(e); return false; }
        return true;
    };
    auto alloc_tmp = [&](void** p, size_t bytes) {
        cudaError_t e = cudaMallocAsync(p, bytes, s);
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); rc = PENT_ERR_ALLOC; return false; }
        if (e != cudaSuccess) { rc = cuda_fail(e); return false; }
        return true;
    };
    if (!alloc_tmp((void**)&stage, sizeof(T) * 5 * (size_t)N) || !alloc_tmp((void**)&dg64, sizeof(double) * 5 * (size_t)N) ||
        !alloc_tmp((void**)&Z, sizeof(double) * 2 * (size_t)n) || !alloc_tmp((void**)&G, sizeof(double) * 2 * (size_t)n) || !alloc_tmp((void**)&coef, sizeof(double) * 10) ||
        !alloc_tmp((void**)&status, sizeof(int)) || !alloc(&h->Zt, sizeof(T) * 2 * (size_t)n) ||
        !alloc(&h->dgp, sizeof(T) * 8 * (size_t)N))
        return done(rc);
    for (int j = 0; j < 5; ++j) {     // order of src: a, b, c, d, e
        cudaError_t e = cudaMemcpyAsync(stage + (size_t)j * N, src[j], sizeof(T) * (size_t)N,
                                        is_dev(src[j]) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) return done(cuda_fail(e));
    }
    // E = leading (N-2) x (N-2) block: the shared-A factorisation of the first N-2 entries of each array
    const void* inner_src[5] = {stage, stage + (size_t)N, stage + 2 * (size_t)N, stage + 3 * (size_t)N,
                                stage + 4 * (size_t)N};
    rc = factor_on_stream<T>(n, inner_src, dtype, &h->inner, bad_row, s);
    if (rc != PENT_OK) return done(rc);
    h->inner->band = 2;               // the fused periodic kernel reads the pentadiagonal tables
    const int tb = 128, nb = (N + tb - 1) / tb;
    periodic_tables_kernel<T><<<nb, tb, 0, s>>>(N, stage, nullptr, nullptr, (T*)h->dgp, dg64);
    periodic_setup_kernel<<<1, 32, 0, s>>>(N, h->inner->fac, dg64, Z, G, coef, status);
    periodic_tables_kernel<T><<<nb, tb, 0, s>>>(N, stage, Z, (typename Vec<T>::T2*)h->Zt, (T*)h->dgp, nullptr);
    count_launch(3);
    {       // chunk states of the Z solve + explicit edge rows (fused periodic solve, on-chip time step)
        constexpr int C = ChunkCfg<T>::C;
        const int Pt = (n + C - 1) / C + PENT_MAXQ, C3 = 3 * C, nt = Pt > C3 ? Pt : C3;   // any rank's slice stays inside
        if (!alloc(&h->pfold, sizeof(T) * 8 * (size_t)Pt) || !alloc(&h->pzedge, sizeof(T) * 2 * (size_t)C3)) return done(rc);
        periodic_fold_kernel<T><<<(nt + tb - 1) / tb, tb, 0, s>>>(n, Pt, Z, G, (T*)h->pfold, (typename Vec<T>::T2*)h->pzedge);
        count_launch();
    }
    cudaError_t le = cudaGetLastError();
    int st = 0;
    if (le == cudaSuccess) le = cudaMemcpyAsync(&st, status, sizeof(int), cudaMemcpyDeviceToHost, s);
    if (le == cudaSuccess) le = cudaMemcpyAsync(h->pc, coef, sizeof(double) * 10, cudaMemcpyDeviceToHost, s);
    if (le == cudaSuccess) le = cudaStreamSynchronize(s);
    if (le != cudaSuccess) return done(cuda_fail(le));
    if (st != 0) { if (bad_row) *bad_row = N - 2; return done(PENT_ERR_PIVOT); }
    *out = h;
    return done(PENT_OK);
}
}  // namespace pent

extern "C" int pent_periodic_fused(const pent_handle* h, int64_t M)
{
    if (!h || !h->periodic) return -1;
    return pent::periodic_fused_supported(h, M, nullptr) ? 1 : 0;
}

extern "C" int pent_factor_periodic(int N, const void* e, const void* c, const void* d, const void* a,
                                    const void* b, pent_dtype dtype, pent_handle** out, int* bad_row)
{
    if (bad_row) *bad_row = -1;
    if (!out) return PENT_ERR_ARG;
    *out = nullptr;
    if (N < 6 || !e || !c || !d || !a || !b) return PENT_ERR_ARG;
    if (dtype != PENT_F64 && dtype != PENT_F32) return PENT_ERR_ARG;
    const void* src[5] = {a, b, c, d, e};
    cudaStream_t s = nullptr;
    PENT_CUDA(cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
    const int rc = dtype == PENT_F64 ? pent::factor_periodic_t<double>(N, src, dtype, out, bad_row, s)
                                     : pent::factor_periodic_t<float>(N, src, dtype, out, bad_row, s);
    cudaStreamDestroy(s);
    return rc;
}
