// pent_solve_chunked.cu -- the headline solve kernel: 2 passes over HBM (read f once, write x
// once), the intermediate vector g never leaves the SM.
//
// WHY NOT ONE THREAD PER SYSTEM (the paper's design): one system's g is N values
// (8 KiB at N=1024 fp64); a warp of 32 systems needs 256 KiB on chip, more than an SM has, so
// g must round-trip through memory (4 passes).  Because A is SHARED by all systems, the sweeps
// are linear recurrences with system-independent coefficients, so k can be split into chunks
// of C rows solved independently from a zero state and stitched exactly:
//
//   chunk p (rows s..s+C-1), thread (system i, chunk p) holds its C values in registers
//   1. local forward sweep from g_{s-2}=g_{s-1}=0      -> g~ ,  E~_p = last two g~
//   2. local back substitution of g~ from x_{e+1}=x_{e+2}=0 -> x^ , S^_p = first two x^
//   3. chunk states, serial over the P chunks of a system (2x2 matrices from the handle):
//        F_p = E~_p + TPhi_p F_{p-1}                      true (g_{e-1}, g_e) of chunk p
//        B_p = S^_p + TX_p F_{p-1} + TPsi_p B_{p+1}       true (x_s, x_{s+1}) of chunk p
//   4. x_{s+j} = x^_j + chi0_j F_{p-1,0} + chi1_j F_{p-1,1} + psi0_j B_{p+1,0} + psi1_j B_{p+1,1}
//
//   Phi = response of the forward recurrence to a unit incoming state, X = local back
//   substitution of Phi, Psi = response of the backward recurrence to a unit incoming state.
//   All are functions of the shared factors only and are built once in pent_factor.  Exact in
//   exact arithmetic; in fp64 it differs from the serial sweep by rounding only.
//
// DATA MOVEMENT (one persistent CTA per SM, tile = S systems x all N rows):
//   f tile --TMA (cp.async.bulk.tensor.2d, 4 boxes, mbarrier complete_tx)--> smem landing
//   buffer --LDS--> registers; the landing buffer is free again after the first block barrier,
//   so the TMA load of the NEXT tile runs under the chunk-state scan, the correction and the
//   stores of this tile.  x goes registers --st.global.cs--> HBM as 128-byte row segments.
//   The shared coefficient tables (9 values per row) are staged ONCE per CTA into shared memory
//   with one cp.async.bulk; every sweep step reads them as 16-byte warp-broadcast LDS.
#include <cuda.h>
#include <cstdio>
#include "pent_internal.h"

namespace pent {

template <typename T> struct ChunkCfg;
template <> struct ChunkCfg<double> { static constexpr int C = 32, S = 16; };
template <> struct ChunkCfg<float>  { static constexpr int C = 64, S = 32; };
#ifndef PENT_L2_PROMOTION
#define PENT_L2_PROMOTION CU_TENSOR_MAP_L2_PROMOTION_L2_256B   // 197 us vs 201 us with 128 B
#endif
#ifndef PENT_TILE_GROUP
#define PENT_TILE_GROUP 1      // consecutive tiles handled back to back by one CTA
#endif
constexpr int CHUNK_MAX_THREADS = 512;
constexpr int BOX_ROWS_MAX = 256;           // TMA box dimension limit
constexpr int MAX_BOXES = 4;

// After the P chunk blocks of a table comes the chunk-transfer table W used by the Kogge-Stone
// scan over chunks (lane q = chunk), stored compactly (only the entries a level can use):
//   TX   : 4 rows x P          TX_q (row-major 2x2, element e at [e*P + q])
//   then for each level l = 0..4, d = 2^l, n = max(0, P-d):
//   WF_l : 4 rows x n          TPhi_q TPhi_{q-1} ... TPhi_{q-d+1}  for q >= d,     at [e*n + q-d]
//   WB_l : 4 rows x n          TPsi_q TPsi_{q+1} ... TPsi_{q+d-1}  for q+d <= P-1, at [e*n + q]
constexpr int W_LEVELS = 5;
__host__ __device__ inline int w_level_off(int P, int l)
{
    int off = 4 * P;
    for (int k = 0; k < l; ++k) { int n = P - (1 << k); off += 8 * (n > 0 ? n : 0); }
    return off;
}
__host__ __device__ inline int w_len(int P) { return w_level_off(P, W_LEVELS); }

// per-chunk coefficient block, in units of T:  [fwd 3C | bwd 2C | corr 4C | pad to 16 B]
template <typename T> __host__ __device__ constexpr int chunk_block_len()
{
    return 9 * ChunkCfg<T>::C + (int)(16 / sizeof(T));
}
template <typename T> __host__ __device__ constexpr size_t table_len(int P)
{
    return (size_t)P * chunk_block_len<T>() + (size_t)w_len(P);
}

// ------------------------------------------------------------------------------------------
// table construction (once per handle): one thread per chunk, fp64 arithmetic, rounded to T
// ------------------------------------------------------------------------------------------
template <typename T>
__global__ void build_chunk_tables_kernel(int N, int P, const double* __restrict__ fac,
                                          T* __restrict__ tab, double* __restrict__ tmat)
{
    constexpr int C = ChunkCfg<T>::C;
    constexpr int BL = chunk_block_len<T>();
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    const double *eps = fac, *beta = fac + N, *alpha = fac + 2 * N, *gamma = fac + 3 * N,
                 *delta = fac + 4 * N;
    T* blk = tab + (size_t)p * BL;
    const int s = p * C;
    double phi0[C], phi1[C];
    // forward: coefficients and Phi
    double h0m2 = 1.0, h0m1 = 0.0, h1m2 = 0.0, h1m1 = 1.0;
    for (int j = 0; j < C; ++j) {
        int k = s + j;
        double ia = 0.0, en = 0.0, bn = 0.0;
        if (k < N) { ia = 1.0 / alpha[k]; en = eps[k] / alpha[k]; bn = beta[k] / alpha[k]; }
        blk[3 * j + 0] = (T)ia; blk[3 * j + 1] = (T)en; blk[3 * j + 2] = (T)bn;
        double h0 = -en * h0m2 - bn * h0m1;
        double h1 = -en * h1m2 - bn * h1m1;
        phi0[j] = h0; phi1[j] = h1;
        h0m2 = h0m1; h0m1 = h0; h1m2 = h1m1; h1m1 = h1;
    }
    double* cm = tmat + (size_t)p * 12;         // TPhi | TX | TPsi, fp64, for the product kernel
    cm[0] = phi0[C - 2]; cm[1] = phi1[C - 2]; cm[2] = phi0[C - 1]; cm[3] = phi1[C - 1];
    // backward: coefficients, X = local back substitution of Phi, Psi
    double x0p1 = 0.0, x0p2 = 0.0, x1p1 = 0.0, x1p2 = 0.0;     // chi_{j+1}, chi_{j+2}
    double q0p1 = 1.0, q0p2 = 0.0, q1p1 = 0.0, q1p2 = 1.0;     // psi_{j+1}, psi_{j+2}
    for (int j = C - 1; j >= 0; --j) {
        int k = s + j;
        double ga = 0.0, de = 0.0;
        if (k < N) { ga = gamma[k]; de = delta[k]; }
        blk[3 * C + 2 * j + 0] = (T)ga; blk[3 * C + 2 * j + 1] = (T)de;
        double x0 = phi0[j] - ga * x0p1 - de * x0p2;
        double x1 = phi1[j] - ga * x1p1 - de * x1p2;
        double q0 = -ga * q0p1 - de * q0p2;
        double q1 = -ga * q1p1 - de * q1p2;
        T* o = blk + 5 * C + 4 * j;
        o[0] = (T)x0; o[1] = (T)x1; o[2] = (T)q0; o[3] = (T)q1;
        if (j <= 1) {
            cm[4 + 2 * j] = x0; cm[5 + 2 * j] = x1;      // TX rows 0,1
            cm[8 + 2 * j] = q0; cm[9 + 2 * j] = q1;      // TPsi rows 0,1
        }
        x0p2 = x0p1; x0p1 = x0; x1p2 = x1p1; x1p1 = x1;
        q0p2 = q0p1; q0p1 = q0; q1p2 = q1p1; q1p1 = q1;
    }
    for (int j = 9 * C; j < BL; ++j) blk[j] = (T)0;
}

// Products of the chunk transfer matrices by doubling (one block, thread q = chunk, P <= 32):
//   WF_{q,2d} = WF_{q,d} WF_{q-d,d},   WB_{q,2d} = WB_{q,d} WB_{q+d,d}.
// levels[0], levels[1] = number of Kogge-Stone levels the forward / backward scan must apply:
// a level whose every entry is below 1e-25 in magnitude (and all levels above it) cannot change
// a double-precision state and is skipped (for diagonally dominant A the products decay
// geometrically, so typically 2-3 levels remain).
template <typename T>
__global__ void build_chunk_products_kernel(int P, const double* __restrict__ tmat,
                                            T* __restrict__ wtab, int* __restrict__ levels)
{
    __shared__ double wf[W_LEVELS][32][4], wb[W_LEVELS][32][4];
    __shared__ int need_f, need_b;
    const int q = threadIdx.x;
    if (q == 0) { need_f = 0; need_b = 0; }
    for (int l = 0; l < W_LEVELS; ++l)
        for (int e = 0; e < 4; ++e) { wf[l][q][e] = 0.0; wb[l][q][e] = 0.0; }
    if (q < P) {
        for (int e = 0; e < 4; ++e) {
            wf[0][q][e] = (q >= 1) ? tmat[q * 12 + e] : 0.0;           // TPhi_q acts on F_{q-1}
            wb[0][q][e] = (q + 1 <= P - 1) ? tmat[q * 12 + 8 + e] : 0.0;   // TPsi_q acts on B_{q+1}
        }
    }
    __syncthreads();
    for (int l = 1; l < W_LEVELS; ++l) {
        const int d = 1 << (l - 1);       // combine two windows of d chunks
        if (q < P && q >= 2 * d) {
            const double* A = wf[l - 1][q];
            const double* B = wf[l - 1][q - d];
            wf[l][q][0] = A[0] * B[0] + A[1] * B[2]; wf[l][q][1] = A[0] * B[1] + A[1] * B[3];
            wf[l][q][2] = A[2] * B[0] + A[3] * B[2]; wf[l][q][3] = A[2] * B[1] + A[3] * B[3];
        }
        if (q < P && q + 2 * d <= P - 1) {
            const double* A = wb[l - 1][q];
            const double* B = wb[l - 1][q + d];
            wb[l][q][0] = A[0] * B[0] + A[1] * B[2]; wb[l][q][1] = A[0] * B[1] + A[1] * B[3];
            wb[l][q][2] = A[2] * B[0] + A[3] * B[2]; wb[l][q][3] = A[2] * B[1] + A[3] * B[3];
        }
        __syncthreads();
    }
    if (q < P) {
        for (int l = 0; l < W_LEVELS; ++l) {
            double mf = 0.0, mb = 0.0;
            const int d = 1 << l, n = P - d;
            T* base = wtab + w_level_off(P, l);
            for (int e = 0; e < 4; ++e) {
                if (q >= d) base[e * n + (q - d)] = (T)wf[l][q][e];
                if (q + d <= P - 1) base[4 * n + e * n + q] = (T)wb[l][q][e];
                mf = fmax(mf, fabs(wf[l][q][e])); mb = fmax(mb, fabs(wb[l][q][e]));
            }
            if (!(mf < 1e-25)) atomicMax(&need_f, l + 1);      // also catches NaN
            if (!(mb < 1e-25)) atomicMax(&need_b, l + 1);
        }
        for (int e = 0; e < 4; ++e) wtab[(size_t)e * P + q] = (T)tmat[q * 12 + 4 + e];
    }
    __syncthreads();
    if (q == 0) { levels[0] = need_f; levels[1] = need_b; }
}

int build_chunk_tables(pent_handle* h, cudaStream_t s)
{
    const bool f64 = h->dtype == PENT_F64;
    const int C = f64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
    const int P = (h->N + C - 1) / C;
    h->nchunks = P;
    h->lev_f = h->lev_b = 0;
    if (P > 32) return PENT_OK;        // too long for the on-chip kernel: tables are not needed
    size_t bytes = f64 ? table_len<double>(P) * 8 : table_len<float>(P) * 4;
    cudaError_t e = cudaMalloc(&h->cf, bytes);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return PENT_ERR_ALLOC; }
    PENT_CUDA(e);
    double* tmat = nullptr;
    int* lev = nullptr;
    PENT_CUDA(cudaMalloc(&tmat, sizeof(double) * 12 * P));
    PENT_CUDA(cudaMalloc(&lev, 2 * sizeof(int)));
    int tb = 32, nb = (P + tb - 1) / tb;
    if (f64) {
        build_chunk_tables_kernel<double><<<nb, tb, 0, s>>>(h->N, P, h->fac, (double*)h->cf, tmat);
        build_chunk_products_kernel<double><<<1, 32, 0, s>>>(
            P, tmat, (double*)h->cf + (size_t)P * chunk_block_len<double>(), lev);
    } else {
        build_chunk_tables_kernel<float><<<nb, tb, 0, s>>>(h->N, P, h->fac, (float*)h->cf, tmat);
        build_chunk_products_kernel<float><<<1, 32, 0, s>>>(
            P, tmat, (float*)h->cf + (size_t)P * chunk_block_len<float>(), lev);
    }
    count_launch(2);
    cudaError_t le = cudaGetLastError();
    int hl[2] = {0, 0};
    if (le == cudaSuccess) le = cudaMemcpyAsync(hl, lev, sizeof(hl), cudaMemcpyDeviceToHost, s);
    if (le == cudaSuccess) le = cudaStreamSynchronize(s);
    cudaFree(tmat); cudaFree(lev);
    if (le != cudaSuccess) return cuda_fail(le);
    h->lev_f = hl[0]; h->lev_b = hl[1];
    return PENT_OK;
}

// ------------------------------------------------------------------------------------------
// PTX helpers: mbarrier, TMA (sm_90+ async proxy; SASS: UTMALDG / UBLKCP / SYNCS)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t addr = smem_u32(bar), ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* tm, int c0, int c1, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes "
        "[%0], [%1, {%2, %3}], [%4];"
        ::"r"(smem_u32(dst)), "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(smem_u32(dst)), "l"((uint64_t)src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// n consecutive T values from shared memory with 16-byte loads (n*sizeof(T) % 16 == 0)
template <typename T, int n>
__device__ __forceinline__ void lds_vec(T (&dst)[n], const T* src)
{
    constexpr int V = 16 / sizeof(T);
    static_assert(n % V == 0, "vector load granularity");
    const uint4* s4 = reinterpret_cast<const uint4*>(src);
#pragma unroll
    for (int v = 0; v < n / V; ++v) {
        uint4 q = s4[v];
        if constexpr (sizeof(T) == 8) {
            dst[2 * v + 0] = __hiloint2double((int)q.y, (int)q.x);
            dst[2 * v + 1] = __hiloint2double((int)q.w, (int)q.z);
        } else {
            dst[4 * v + 0] = __uint_as_float(q.x); dst[4 * v + 1] = __uint_as_float(q.y);
            dst[4 * v + 2] = __uint_as_float(q.z); dst[4 * v + 3] = __uint_as_float(q.w);
        }
    }
}

#include "pent_chunked_kernel.cuh"

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        return (EncodeTiledFn)p;
    }();
    return fn;
}

template <typename T> static int chunk_P(const pent_handle* h)
{
    return (h->N + ChunkCfg<T>::C - 1) / ChunkCfg<T>::C;
}

bool chunked_supported(const pent_handle* h, int64_t M, const void* f)
{
    if (!h || h->kind != 0 || !h->cf) return false;
    const bool f64 = h->dtype == PENT_F64;
    const int esz = f64 ? 8 : 4;
    const int S = f64 ? ChunkCfg<double>::S : ChunkCfg<float>::S;
    const int P = f64 ? chunk_P<double>(h) : chunk_P<float>(h);
    if (P * S > CHUNK_MAX_THREADS) return false;            // N too large to keep a tile on chip
    {
        const int C = f64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
        const int rows = P * C, br = rows < BOX_ROWS_MAX ? rows : BOX_ROWS_MAX;
        const size_t tl = f64 ? table_len<double>(P) : table_len<float>(P);
        const size_t smem = ((size_t)((rows + br - 1) / br) * br * S + tl + (size_t)4 * (P + 1) * S) * esz +
                            (1 + 2 * MAX_BOXES) * sizeof(uint64_t);
        if (smem > 232448) return false;                    // 227 KB dynamic shared memory per CTA
    }
    if ((M * esz) % 16 != 0) return false;                  // TMA global stride alignment
    if (f && ((uintptr_t)f % 16) != 0) return false;        // TMA global address alignment
    if (M > (int64_t)0x7fffffff) return false;              // TMA coordinates are 32-bit
    return encode_fn() != nullptr;
}

template <typename T>
static int launch_chunked_t(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s)
{
    constexpr int C = ChunkCfg<T>::C, S = ChunkCfg<T>::S;
    const int P = chunk_P<T>(h);
    ChunkParams<T> prm;
    prm.N = h->N; prm.P = P; prm.M = M;
    int Pw = 1, lg = 0;
    while (Pw < P) { Pw *= 2; ++lg; }
    prm.Pw = Pw;
    prm.lev_f = h->lev_f < lg ? h->lev_f : lg;
    prm.lev_b = h->lev_b < lg ? h->lev_b : lg;
    for (int l = 0; l < W_LEVELS; ++l) prm.woff[l] = w_level_off(P, l);
    const int rows = P * C;
    prm.box_rows = rows < BOX_ROWS_MAX ? rows : BOX_ROWS_MAX;
    prm.nbox = (rows + prm.box_rows - 1) / prm.box_rows;
    prm.ntiles = (M + S - 1) / S;
    for (int b = 0; b < MAX_BOXES; ++b) prm.wcount[b] = 0;
    for (int w = 0; w * 32 < P * S; ++w) prm.wcount[((w * 32 / S) * C) / prm.box_rows] += 1;
    prm.table = (const T*)h->cf;
    prm.x = (T*)x;

    CUtensorMap tm;
    cuuint64_t gdim[2] = {(cuuint64_t)M, (cuuint64_t)h->N};
    cuuint64_t gstr[1] = {(cuuint64_t)M * sizeof(T)};
    cuuint32_t box[2] = {(cuuint32_t)S, (cuuint32_t)prm.box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult cr = encode_fn()(&tm, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                              2, const_cast<void*>(f), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_NONE, PENT_L2_PROMOTION,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) { g_last_cuda_error = (int)cudaErrorInvalidValue; return PENT_ERR_CUDA; }

    const size_t smem = ((size_t)prm.nbox * prm.box_rows * S + table_len<T>(P) + (size_t)4 * (P + 1) * S) * sizeof(T) +
                        (1 + 2 * MAX_BOXES) * sizeof(uint64_t);
    auto kern = solve_chunked_kernel<T>;
    static thread_local size_t smem_set = 0;
    if (smem > smem_set) {
        PENT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        smem_set = smem;
    }
    const int threads = (P * S + 31) / 32 * 32;
    int dev = 0, nsm = 0, occ = 0;
    PENT_CUDA(cudaGetDevice(&dev));
    PENT_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    PENT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem));
    if (occ < 1) return PENT_ERR_ARG;
    int64_t grid = (int64_t)nsm * occ;
    const int64_t groups = (prm.ntiles + PENT_TILE_GROUP - 1) / PENT_TILE_GROUP;
    if (grid > groups) grid = groups;
    kern<<<(unsigned)grid, threads, smem, s>>>(tm, prm);
    count_launch();
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}

int launch_solve_chunked(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s)
{
    if (h->dtype == PENT_F64) return launch_chunked_t<double>(h, M, f, x, s);
    return launch_chunked_t<float>(h, M, f, x, s);
}
}  // namespace pent
