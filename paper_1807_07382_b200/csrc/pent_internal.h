// pent_internal.h -- private declarations shared by the .cu files of libpent (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include "pent.h"

// Cluster sizes (CTAs along k) the chunked kernel has tables for: Q = 1 << j, j < PENT_NQ.  Q = 16 is a
// non-portable cluster size (cudaFuncAttributeNonPortableClusterSizeAllowed); PENT_MAXQ sizes the block-product table.
#define PENT_NQ 5
#define PENT_MAXQ 16

struct pent_handle {
    int kind;            // 0 = shared A, 1 = per-system factors
    int N;
    pent_dtype dtype;
    int64_t M;           // per-system only
    int device;          // CUDA device ordinal the handle's memory lives on (every call checks it)
    // shared A: set at factor time when the matrix is I + sigma L^2 for the Dirichlet (0) or zero-flux (1)
    // second-difference matrix L (what pent_step_batch(kind 0) requires of its handle); -1 otherwise
    int l2_bc;
    double l2_sigma;
    double growth[3];    // shared A: max |Phi|, |X|, |Psi| inside a chunk (stability guard of the chunk stitching)
    int band;            // shared A: 1 if a == e == 0 inside the matrix (tridiagonal), else 2
    // ---- shared A, all device memory ----
    double* diag;        // 5*N: a,b,c,d,e widened to fp64, out-of-matrix entries zeroed
    double* fac;         // 5*N: eps,beta,alpha,gamma,delta (Eq. 13), fp64
    void* fw;            // N x {1/alpha, eps/alpha, beta/alpha, 0}   in T (T4)
    void* bw;            // N x {gamma, delta}                        in T (T2)
    void* dg;            // N x {a,b,c,d,e,0,0,0} in T, for the (2I-A)c right-hand side
    // chunked kernel (pent_solve_chunked.cu): for cluster size Q = 1 << j, Q per-rank coefficient
    // tables in T, laid out as they sit in shared memory; cfP[j] = chunks per CTA (0: not built)
    void* cf[PENT_NQ];
    int cfP[PENT_NQ];
    int lev_f[PENT_NQ], lev_b[PENT_NQ];   // Kogge-Stone levels the chunk-state scans need
    // cluster exchange depth: how many neighbouring ranks on each side a CTA exchanges block aggregates with: 1 when
    // every block transfer product is below 1e-25 (diagonally dominant matrices: the state entering a block of >= 32
    // chunks has decayed to nothing by its end), else Q - 1 (every rank); xdepth1: the tridiagonal tables
    int xdepth[PENT_NQ], xdepth1[PENT_NQ];
    // the same for the tridiagonal instantiation (band == 1 only): 5-word coefficient rows, scalar transfers
    void* cf1[PENT_NQ];
    int lev_f1[PENT_NQ], lev_b1[PENT_NQ];
    // ---- periodic (cyclic) A, Eqs. 7a-12 (pent_periodic.cu): N is the full size, `inner`
    // is the shared-A handle of the (N-2) x (N-2) block E, Zt = E^{-1} k as (N-2) x {z0, z1} in T,
    // dgp = N x {a,b,c,d,e,0,0,0} in T with the wrapped entries kept, pc = the six entries of h
    // (row N-2: cols 0, N-4, N-3; row N-1: cols 0, 1, N-3) and the inverted 2x2 Schur complement
    int periodic;
    pent_handle* inner;
    void* Zt;
    void* dgp;
    double pc[10];
    // x^ = y - Z t without the rows of Z on chip (fused periodic solve, on-chip periodic time step): per chunk of C rows
    // the chunk states of the Z solve, [chunks + PENT_MAXQ][8] in T = {g^Z of rows s-2, s-1 | Z of rows e+1, e+2} x 2
    // columns (zero for the chunks that hold the non-zero rows of k), and the explicit rows of Z of those chunks,
    // [3][C] x {z0, z1} in T: chunk 0, the chunk of row n-2, the chunk of row n-1 (periodic_fold_kernel)
    void* pfold;
    void* pzedge;
    // ---- per-system factors, device, interleaved, in T ----
    void* ms;            // 5*N*M: ia, en, bn, gamma, delta
};

namespace pent {

constexpr int PENT_UNSUPPORTED = -100;      // internal: no on-chip plan for this shape (never crosses the C ABI)

extern thread_local int g_last_cuda_error;
extern thread_local int64_t g_launches;

inline int cuda_fail(cudaError_t e) { g_last_cuda_error = (int)e; return PENT_ERR_CUDA; }
inline void count_launch(int n = 1) { g_launches += n; }

// cudaFuncAttributeMaxDynamicSharedMemorySize is a PROCESS-wide property of (kernel instance, device), and
// cudaFuncSetAttribute sets it (it can lower it).  So it is raised exactly once per kernel instance and
// device, to the largest value any launch of this library uses (SMEM_OPTIN), and never touched again:
// `mask` is a `static SmemOnce` at the launch site (one per template instance), bit d = done on device d.
// Two threads racing on the first launch both set the same value, which is harmless.
constexpr size_t SMEM_OPTIN = 232448;       // 227 KB, the sm_100 per-CTA limit
struct SmemOnce { std::atomic<uint32_t> mask{0}; };
template <typename K>
inline cudaError_t ensure_dynamic_smem(SmemOnce& once, K kernel, size_t bytes)
{
    if (bytes > SMEM_OPTIN) return cudaErrorInvalidValue;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const uint32_t bit = 1u << (dev & 31);
    if (!(once.mask.load(std::memory_order_acquire) & bit)) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_OPTIN);
        if (e != cudaSuccess) return e;
        once.mask.fetch_or(bit, std::memory_order_release);
    }
    return cudaSuccess;
}

// every entry point that takes a handle: the handle's memory must be on the CURRENT device
inline bool on_handle_device(const pent_handle* h)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return false; }
    return dev == h->device;
}

#define PENT_CUDA(call)                                           \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) return ::pent::cuda_fail(e__);    \
    } while (0)

#define PENT_LAUNCH_CHECK()                                       \
    do {                                                          \
        cudaError_t e__ = cudaGetLastError();                     \
        if (e__ != cudaSuccess) return ::pent::cuda_fail(e__);    \
    } while (0)

template <typename T> struct Vec;
template <> struct Vec<double> { using T2 = double2; using T4 = double4; };
template <> struct Vec<float>  { using T2 = float2;  using T4 = float4;  };

#ifdef __CUDACC__
// read-only-path loads of the coefficient tuples (warp-uniform addresses: one broadcast each)
__device__ __forceinline__ double4 ldg4(const double4* p)
{
    const double2* q = reinterpret_cast<const double2*>(p);
    double2 lo = __ldg(q), hi = __ldg(q + 1);
    return make_double4(lo.x, lo.y, hi.x, hi.y);
}
__device__ __forceinline__ float4 ldg4(const float4* p) { return __ldg(p); }
__device__ __forceinline__ double2 ldg2(const double2* p) { return __ldg(p); }
__device__ __forceinline__ float2 ldg2(const float2* p) { return __ldg(p); }
#endif

// shared-A factorisation with every kernel, copy and temporary on the private stream `s` (pent_factor.cu)
template <typename T>
int factor_on_stream(int N, const void* const src[5], pent_dtype dtype, pent_handle** out, int* bad_row,
                     cudaStream_t s);

// kernels / launchers implemented across the .cu files
int launch_solve_tps(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s);
// Q = CTAs per cluster along k, S = systems per tile; 0 = choose (pent_solve_chunked.cu)
int launch_solve_chunked(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s,
                         int Q, int S);
bool chunk_stitching_stable(const pent_handle* h);
bool chunked_supported(const pent_handle* h, int64_t M, const void* f /* may be null */, int Q, int S);
bool step_chunked_supported(const pent_handle* h, int64_t M, const void* c /* may be null */);
int launch_step_chunked(const pent_handle* h, const pent_step_params* p, const pent_forcing* g, int64_t M, void* c,
                        int nsteps, cudaStream_t s);
bool periodic_fused_supported(const pent_handle* h, int64_t M, const void* f /* may be null */);
int launch_solve_chunked_periodic(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s);
int solve_periodic(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s, int kernel);
int step_periodic(const pent_handle* h, int64_t M, void* c, void* scratch, int nsteps, cudaStream_t s);
bool step_chunked_periodic_supported(const pent_handle* h, int64_t M, const void* c /* may be null */);
int launch_step_chunked_periodic(const pent_handle* h, int64_t M, void* c, int nsteps, cudaStream_t s);
bool chunked_rows_supported(const pent_handle* h, int64_t M);
int launch_solve_chunked_rows(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s,
                              int Q = 0, int S = 0, int loader = 0);
// x = 2 A^{-1} f - f on an interleaved / a system-major batch (default plans, pentadiagonal tables); PENT_UNSUPPORTED: no plan
int launch_solve_chunked_epi(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s);
int launch_solve_chunked_rows_epi(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s);
int chunked_choice(const pent_handle* h, int64_t M, int* Q, int* S);   // 1 and the default plan, or 0
int chunked_rows_choice(const pent_handle* h, int64_t M, int* Q, int* S, int* mode);   // the same for a system-major batch

}  // namespace pent
