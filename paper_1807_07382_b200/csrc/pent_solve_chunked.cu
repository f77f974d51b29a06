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
constexpr int CHUNK_MAX_THREADS = 512;
constexpr int BOX_ROWS_MAX = 256;           // TMA box dimension limit
constexpr int MAX_BOXES = 4;

// per-chunk coefficient block, in units of T:  [fwd 3C | bwd 2C | corr 4C | pad to 16 B]
template <typename T> __host__ __device__ constexpr int chunk_block_len()
{
    return 9 * ChunkCfg<T>::C + (int)(16 / sizeof(T));
}
template <typename T> __host__ __device__ constexpr size_t table_len(int P)
{
    return (size_t)P * chunk_block_len<T>() + (size_t)P * 12;
}

// ------------------------------------------------------------------------------------------
// table construction (once per handle): one thread per chunk, fp64 arithmetic, rounded to T
// ------------------------------------------------------------------------------------------
template <typename T>
__global__ void build_chunk_tables_kernel(int N, int P, const double* __restrict__ fac,
                                          T* __restrict__ tab)
{
    constexpr int C = ChunkCfg<T>::C;
    constexpr int BL = chunk_block_len<T>();
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    const double *eps = fac, *beta = fac + N, *alpha = fac + 2 * N, *gamma = fac + 3 * N,
                 *delta = fac + 4 * N;
    T* blk = tab + (size_t)p * BL;
    T* cm = tab + (size_t)P * BL + (size_t)p * 12;
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
    cm[0] = (T)phi0[C - 2]; cm[1] = (T)phi1[C - 2]; cm[2] = (T)phi0[C - 1]; cm[3] = (T)phi1[C - 1];
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
            cm[4 + 2 * j] = (T)x0; cm[5 + 2 * j] = (T)x1;      // TX rows 0,1
            cm[8 + 2 * j] = (T)q0; cm[9 + 2 * j] = (T)q1;      // TPsi rows 0,1
        }
        x0p2 = x0p1; x0p1 = x0; x1p2 = x1p1; x1p1 = x1;
        q0p2 = q0p1; q0p1 = q0; q1p2 = q1p1; q1p1 = q1;
    }
    for (int j = 9 * C; j < BL; ++j) blk[j] = (T)0;
}

int build_chunk_tables(pent_handle* h, cudaStream_t s)
{
    const bool f64 = h->dtype == PENT_F64;
    const int C = f64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
    const int P = (h->N + C - 1) / C;
    h->nchunks = P;
    size_t bytes = f64 ? table_len<double>(P) * 8 : table_len<float>(P) * 4;
    cudaError_t e = cudaMalloc(&h->cf, bytes);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return PENT_ERR_ALLOC; }
    PENT_CUDA(e);
    int tb = 32, nb = (P + tb - 1) / tb;
    if (f64) build_chunk_tables_kernel<double><<<nb, tb, 0, s>>>(h->N, P, h->fac, (double*)h->cf);
    else build_chunk_tables_kernel<float><<<nb, tb, 0, s>>>(h->N, P, h->fac, (float*)h->cf);
    count_launch();
    PENT_LAUNCH_CHECK();
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

template <typename T>
struct ChunkParams {
    int N;            // rows
    int P;            // chunks per system = blockDim.x / S
    int box_rows;     // rows per TMA box
    int nbox;         // boxes per tile
    int64_t M;
    int64_t ntiles;
    const T* table;   // global coefficient table (layout = shared-memory layout)
    T* x;
};

template <typename T>
__global__ void __launch_bounds__(CHUNK_MAX_THREADS, 1)
solve_chunked_kernel(const __grid_constant__ CUtensorMap tm, const ChunkParams<T> prm)
{
    constexpr int C = ChunkCfg<T>::C, S = ChunkCfg<T>::S, BL = chunk_block_len<T>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int P = prm.P;
    T* landing = reinterpret_cast<T*>(smem_raw);
    T* table = landing + (size_t)prm.nbox * prm.box_rows * S;
    T* stE = table + table_len<T>(P);
    T* stS = stE + (size_t)P * S * 2;
    uint64_t* bars = reinterpret_cast<uint64_t*>(stS + (size_t)P * S * 2);

    const int tid = threadIdx.x, i = tid % S, p = tid / S;
    const uint32_t box_bytes = (uint32_t)(prm.box_rows * S * sizeof(T));
    const uint32_t table_bytes = (uint32_t)(table_len<T>(P) * sizeof(T));
    const int64_t stride = gridDim.x;

    auto issue_tile = [&](int64_t t) {
        for (int b = 0; b < prm.nbox; ++b) {
            mbar_expect_tx(&bars[1 + b], box_bytes);
            tma_load_2d(landing + (size_t)b * prm.box_rows * S, &tm, (int)(t * S), b * prm.box_rows,
                        &bars[1 + b]);
        }
    };

    if (tid == 0) {
        for (int b = 0; b <= MAX_BOXES; ++b) mbar_init(&bars[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    int64_t tile = blockIdx.x;
    if (tid == 0) {
        mbar_expect_tx(&bars[0], table_bytes);
        bulk_load_1d(table, prm.table, table_bytes, &bars[0]);
        if (tile < prm.ntiles) issue_tile(tile);
    }
    mbar_wait(&bars[0], 0);

    const T* blk = table + (size_t)p * BL;
    const T* cmat = table + (size_t)P * BL;
    const int mybox = (p * C) / prm.box_rows;
    uint32_t parity = 0;

    for (; tile < prm.ntiles; tile += stride) {
        // ---- tile data: landing buffer -> registers ----
        mbar_wait(&bars[1 + mybox], parity);
        T v[C];
        {
            const T* src = landing + (size_t)p * C * S + i;
#pragma unroll
            for (int j = 0; j < C; ++j) v[j] = src[j * S];
        }
        // ---- 1. local forward sweep from a zero state (normalised) ----
        {
            T g1 = 0, g2 = 0;
#pragma unroll
            for (int jg = 0; jg < C / 4; ++jg) {
                T w[12];
                lds_vec<T, 12>(w, blk + 12 * jg);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int j = 4 * jg + r;
                    T t = w[3 * r] * v[j];
                    t = fma(-w[3 * r + 1], g2, t);
                    T g = fma(-w[3 * r + 2], g1, t);
                    v[j] = g; g2 = g1; g1 = g;
                }
            }
            stE[(p * S + i) * 2 + 0] = v[C - 2];
            stE[(p * S + i) * 2 + 1] = v[C - 1];
        }
        // ---- 2. local back substitution of g~ from a zero state ----
        {
            T x1 = 0, x2 = 0;
#pragma unroll
            for (int jg = C / 4 - 1; jg >= 0; --jg) {
                T w[8];
                lds_vec<T, 8>(w, blk + 3 * C + 8 * jg);
#pragma unroll
                for (int r = 3; r >= 0; --r) {
                    const int j = 4 * jg + r;
                    T xv = fma(-w[2 * r + 1], x2, fma(-w[2 * r], x1, v[j]));
                    v[j] = xv; x2 = x1; x1 = xv;
                }
            }
            stS[(p * S + i) * 2 + 0] = v[0];
            stS[(p * S + i) * 2 + 1] = v[1];
        }
        __syncthreads();       // states published; landing buffer fully consumed
        if (tid == 0 && tile + stride < prm.ntiles) issue_tile(tile + stride);

        // ---- 3. chunk-state scans, one thread per system ----
        if (tid < S) {
            T f0 = 0, f1 = 0;
            for (int q = 0; q < P; ++q) {
                const T* m = cmat + q * 12;
                T e0 = stE[(q * S + tid) * 2], e1 = stE[(q * S + tid) * 2 + 1];
                T n0 = fma(m[1], f1, fma(m[0], f0, e0));
                T n1 = fma(m[3], f1, fma(m[2], f0, e1));
                f0 = n0; f1 = n1;
                stE[(q * S + tid) * 2] = f0; stE[(q * S + tid) * 2 + 1] = f1;
            }
            T b0 = 0, b1 = 0;
            for (int q = P - 1; q >= 0; --q) {
                const T* m = cmat + q * 12;
                T fi0 = 0, fi1 = 0;
                if (q > 0) { fi0 = stE[((q - 1) * S + tid) * 2]; fi1 = stE[((q - 1) * S + tid) * 2 + 1]; }
                T s0 = stS[(q * S + tid) * 2], s1 = stS[(q * S + tid) * 2 + 1];
                s0 = fma(m[5], fi1, fma(m[4], fi0, s0));
                s1 = fma(m[7], fi1, fma(m[6], fi0, s1));
                T n0 = fma(m[9], b1, fma(m[8], b0, s0));
                T n1 = fma(m[11], b1, fma(m[10], b0, s1));
                b0 = n0; b1 = n1;
                stS[(q * S + tid) * 2] = b0; stS[(q * S + tid) * 2 + 1] = b1;
            }
        }
        __syncthreads();
        T F0 = 0, F1 = 0, B0 = 0, B1 = 0;
        if (p > 0) { F0 = stE[((p - 1) * S + i) * 2]; F1 = stE[((p - 1) * S + i) * 2 + 1]; }
        if (p + 1 < P) { B0 = stS[((p + 1) * S + i) * 2]; B1 = stS[((p + 1) * S + i) * 2 + 1]; }
        __syncthreads();       // states consumed: the next tile may overwrite them

        // ---- 4. correction and store ----
        {
            const int64_t col = tile * S + i;
            const bool colok = col < prm.M;
            T* xo = prm.x + (int64_t)(p * C) * prm.M + col;
#pragma unroll
            for (int jg = 0; jg < C / 4; ++jg) {
                T w[16];
                lds_vec<T, 16>(w, blk + 5 * C + 16 * jg);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int j = 4 * jg + r;
                    T xv = fma(w[4 * r + 3], B1, fma(w[4 * r + 2], B0,
                           fma(w[4 * r + 1], F1, fma(w[4 * r], F0, v[j]))));
                    if (colok && p * C + j < prm.N) __stcs(xo + (int64_t)j * prm.M, xv);
                }
            }
        }
        parity ^= 1;
    }
}

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
    const int rows = P * C;
    prm.box_rows = rows < BOX_ROWS_MAX ? rows : BOX_ROWS_MAX;
    prm.nbox = (rows + prm.box_rows - 1) / prm.box_rows;
    prm.ntiles = (M + S - 1) / S;
    prm.table = (const T*)h->cf;
    prm.x = (T*)x;

    CUtensorMap tm;
    cuuint64_t gdim[2] = {(cuuint64_t)M, (cuuint64_t)h->N};
    cuuint64_t gstr[1] = {(cuuint64_t)M * sizeof(T)};
    cuuint32_t box[2] = {(cuuint32_t)S, (cuuint32_t)prm.box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult cr = encode_fn()(&tm, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                              2, const_cast<void*>(f), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) { g_last_cuda_error = (int)cudaErrorInvalidValue; return PENT_ERR_CUDA; }

    const size_t smem = ((size_t)prm.nbox * prm.box_rows * S + table_len<T>(P) + (size_t)4 * P * S) * sizeof(T) +
                        (1 + MAX_BOXES) * sizeof(uint64_t);
    auto kern = solve_chunked_kernel<T>;
    static thread_local size_t smem_set = 0;
    if (smem > smem_set) {
        PENT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        smem_set = smem;
    }
    const int threads = P * S;
    int dev = 0, nsm = 0, occ = 0;
    PENT_CUDA(cudaGetDevice(&dev));
    PENT_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    PENT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem));
    if (occ < 1) return PENT_ERR_ARG;
    int64_t grid = (int64_t)nsm * occ;
    if (grid > prm.ntiles) grid = prm.ntiles;
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
