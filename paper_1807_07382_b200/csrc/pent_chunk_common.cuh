// pent_chunk_common.cuh -- shared by the chunked solve kernel (pent_solve_chunked.cu) and the
// on-chip fused time-step kernel (pent_step_chunked.cu): table layout, PTX helpers (mbarrier, TMA,
// DSMEM), and the three arithmetic stages of the chunked algorithm (local sweeps, chunk-state
// scan, correction).  See the algorithm notes at the top of pent_solve_chunked.cu.
#pragma once
#include <cuda.h>
#include "pent_internal.h"

namespace pent {

template <typename T> struct ChunkCfg;
template <> struct ChunkCfg<double> { static constexpr int C = 32; };   // rows per thread
template <> struct ChunkCfg<float>  { static constexpr int C = 64; };
#ifndef PENT_L2_PROMOTION
#define PENT_L2_PROMOTION CU_TENSOR_MAP_L2_PROMOTION_L2_256B   // 197 us vs 201 us with 128 B
#endif
constexpr int CHUNK_MAX_THREADS = 512;
constexpr int BOX_ROWS_MAX = 256;           // TMA box dimension limit
constexpr int MAX_BOXES = 4;
constexpr int MAX_PL = 32;                  // chunks per CTA (one warp scans a system's chunks)
constexpr size_t SMEM_LIMIT = 232448;       // 227 KB dynamic shared memory per CTA

// After the P chunk blocks of a (per-rank) table comes the chunk-transfer table W (P = chunks of
// this CTA, q = local chunk; every 2x2 matrix is row-major with element e at [e*len + index]):
//   TX   : 4 x P     TX_q
//   (the next three only in the tables of a cluster, Q > 1)
//   PF   : 4 x P     TPhi_q TPhi_{q-1} ... TPhi_{first chunk of the block}   (acts on the F entering the block)
//   PB   : 4 x P     TPsi_q TPsi_{q+1} ... TPsi_{last chunk of the block}    (acts on the B entering the block)
//   BLK  : 8 MAXQ    block products of every cluster rank r < MAXQ = 16: TPhiBlock(r) at [4r..4r+3] (contiguous
//                    2x2), TPsiBlock(r) at [4 MAXQ + 4r..]
//   then for each Kogge-Stone level l = 0..4, d = 2^l, n = max(0, P-d):
//   WF_l : 4 x n     TPhi_q TPhi_{q-1} ... TPhi_{q-d+1}  for q >= d,     at [e*n + q-d]
//   WB_l : 4 x n     TPsi_q TPsi_{q+1} ... TPsi_{q+d-1}  for q+d <= P-1, at [e*n + q]
// Only the levels a handle needs are staged into shared memory (they come last).
// BAND = 1 (tridiagonal A, a = e = 0: cuThomasBatch's case): the recurrences have ONE term, the
// chunk states and every transfer "matrix" are scalars, so every 4 above becomes 1 (BLK: MAXQ + MAXQ scalars).
constexpr int W_LEVELS = 5;
__host__ __device__ inline int w_level_off(int P, int l, int Q, int BAND = 2)
{
    const int u = BAND == 2 ? 4 : 1;
    int off = Q > 1 ? 3 * u * P + 2 * PENT_MAXQ * u : u * P;      // PF, PB, BLK exist only in cluster tables
    for (int k = 0; k < l; ++k) { int n = P - (1 << k); off += 2 * u * (n > 0 ? n : 0); }
    return off;
}
__host__ __device__ inline int w_len(int P, int Q, int BAND = 2) { return w_level_off(P, W_LEVELS, Q, BAND); }

// per-chunk coefficient block, in units of T:  [fwd 3C | bwd 2C | corr 4C | pad to 16 B]   (BAND 2)
//                                              [fwd 2C | bwd  C | corr 2C | pad to 16 B]   (BAND 1)
template <typename T, int BAND = 2> __host__ __device__ constexpr int chunk_block_len()
{
    return (BAND == 2 ? 9 : 5) * ChunkCfg<T>::C + (int)(16 / sizeof(T));
}
template <typename T, int BAND = 2> __host__ __device__ constexpr size_t table_len(int P, int Q)
{
    // rounded up to 4 words: every rank's table starts 16-byte aligned in global memory (cp.async.bulk source)
    return ((size_t)P * chunk_block_len<T, BAND>() + (size_t)w_len(P, Q, BAND) + 3) & ~(size_t)3;
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

__device__ __forceinline__ void tma_store_2d(const CUtensorMap* tm, int c0, int c1, const void* src)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(smem_u32(src)) : "memory");
}

// per-thread asynchronous copies global -> shared (LDGSTS), 8 or 4 bytes
__device__ __forceinline__ void cp_async_elem(double* dst, const double* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_elem(float* dst, const float* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N_>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N_) : "memory"); }

// 32 bytes per thread in one global access (LDG.256 / STG.256, sm_100): a whole DRAM sector per lane, so a
// lane that walks a contiguous run never splits a sector between two requests.  addr must be 32-byte aligned.
__device__ __forceinline__ void ldg256(double (&o)[4], const double* p)
{
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(o[0]), "=d"(o[1]), "=d"(o[2]), "=d"(o[3]) : "l"(p));
}
__device__ __forceinline__ void ldg256(float (&o)[8], const float* p)
{
    asm volatile("ld.global.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(o[0]), "=f"(o[1]), "=f"(o[2]), "=f"(o[3]), "=f"(o[4]), "=f"(o[5]), "=f"(o[6]), "=f"(o[7]) : "l"(p));
}
__device__ __forceinline__ void stg256(double* p, const double (&v)[4])
{
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(v[3]) : "memory");
}
__device__ __forceinline__ void stg256(float* p, const float (&v)[8])
{
    asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 ::"l"(p), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "f"(v[4]), "f"(v[5]), "f"(v[6]), "f"(v[7]) : "memory");
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

template <typename T> struct Pair;
template <> struct Pair<double> { using type = double2; };
template <> struct Pair<float>  { using type = float2; };
// chunk state: the last two g / first two x of a chunk (BAND 2), or the last g / first x (BAND 1)
template <typename T, int BAND> struct ChunkState { using type = typename Pair<T>::type; };
template <typename T> struct ChunkState<T, 1> { using type = T; };

template <typename T>
__device__ __forceinline__ T shfl_up_t(T v, int d, int w) { return __shfl_up_sync(0xffffffffu, v, d, w); }
template <typename T>
__device__ __forceinline__ T shfl_down_t(T v, int d, int w) { return __shfl_down_sync(0xffffffffu, v, d, w); }

// y += m * u for a row-major 2x2 m stored with element stride `n` (m[e*n])
template <typename T>
__device__ __forceinline__ void mat2_acc(T& y0, T& y1, const T* m, int n, T u0, T u1)
{
    y0 = fma(m[n], u1, fma(m[0], u0, y0));
    y1 = fma(m[3 * n], u1, fma(m[2 * n], u0, y1));
}

// ---- thread-block-cluster helpers (CUDA 12 sm_90+ intrinsics; SASS: UCGABAR_ARV / UCGABAR_WAIT,
// remote stores through the distributed-shared-memory window)
__device__ __forceinline__ void cluster_sync_all()
{
    __cluster_barrier_arrive();      // release
    __cluster_barrier_wait();        // acquire
}
__device__ __forceinline__ uint32_t map_to_rank(const void* local, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(local)), "r"(rank));
    return r;
}
// Remote store of one chunk state into CTA `rank`'s shared memory that signals that CTA's mbarrier
// with complete_tx (16 or 8 bytes): producer -> consumer over DSMEM with no thread-scope fence, so
// the x stores still in flight from the previous tile are not drained (a release-scoped cluster
// barrier in the tile loop measured 271 us against 215 us for cfg3: profiles/r01_ab_tuning.md).
__device__ __forceinline__ void st_async_pair(const void* local, const uint64_t* local_bar, uint32_t rank,
                                              double a, double b)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];"
                 ::"r"(map_to_rank(local, rank)), "d"(a), "d"(b), "r"(map_to_rank(local_bar, rank)) : "memory");
}
__device__ __forceinline__ void st_async_pair(const void* local, const uint64_t* local_bar, uint32_t rank,
                                              float a, float b)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];"
                 ::"r"(map_to_rank(local, rank)), "f"(a), "f"(b), "r"(map_to_rank(local_bar, rank)) : "memory");
}

__device__ __forceinline__ void st_async_one(const void* local, const uint64_t* local_bar, uint32_t rank, double a)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];"
                 ::"r"(map_to_rank(local, rank)), "d"(a), "r"(map_to_rank(local_bar, rank)) : "memory");
}
__device__ __forceinline__ void st_async_one(const void* local, const uint64_t* local_bar, uint32_t rank, float a)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f32 [%0], %1, [%2];"
                 ::"r"(map_to_rank(local, rank)), "f"(a), "r"(map_to_rank(local_bar, rank)) : "memory");
}

// One CTA = S systems x P chunks (thread = one system, one chunk of C rows, held in registers).
// blockDim.x >= P*S (a multiple of 32); threads with p >= P only take part in barriers/scan.
// CLUSTER: the Q CTAs of a cluster own consecutive blocks of P chunks of the SAME S systems; the
// chunk states are stitched across CTAs through distributed shared memory (two exchanges per tile).

// ------------------------------------------------------------------------------------------
// stage 1+2: local forward sweep (normalised coefficients) and local back
// substitution of one chunk held in registers, both from a zero state.
// blk = the chunk's coefficient block in shared memory.  v: f -> x^ ; e = last two g~ ; s = first two x^.
// ------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void chunk_local_sweeps(T (&v)[ChunkCfg<T>::C], const T* blk,
                                                   typename Pair<T>::type& e, typename Pair<T>::type& s)
{
    constexpr int C = ChunkCfg<T>::C;
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
    e.x = v[C - 2]; e.y = v[C - 1];
    T x1 = 0, x2 = 0;
#pragma unroll
    for (int jg = C / 4 - 1; jg >= 0; --jg) {
        T w[8];
        lds_vec<T, 8>(w, blk + 3 * C + 8 * jg);
#pragma unroll
        for (int r = 3; r >= 0; --r) {
            const int j = 4 * jg + r;
            T xv = fma(-w[2 * r], x1, fma(-w[2 * r + 1], x2, v[j]));   // x1 last: 1 fma on the chain
            v[j] = xv; x2 = x1; x1 = xv;
        }
    }
    s.x = v[0]; s.y = v[1];
}

// stage 4, one group of 4 rows: x = x^ + chi0 F0 + chi1 F1 + psi0 B0 + psi1 B1
template <typename T>
__device__ __forceinline__ void chunk_correct4(T (&out)[4], const T* v4, const T* blk, int jg, T F0, T F1, T B0, T B1)
{
    constexpr int C = ChunkCfg<T>::C;
    T w[16];
    lds_vec<T, 16>(w, blk + 5 * C + 16 * jg);
#pragma unroll
    for (int r = 0; r < 4; ++r)
        out[r] = fma(w[4 * r + 3], B1, fma(w[4 * r + 2], B0, fma(w[4 * r + 1], F1, fma(w[4 * r], F0, v4[r]))));
}

// ---- SPT systems per thread (register blocking over systems) ------------------------------------------------
// A coefficient LDS.128 is a warp broadcast: it costs the shared-memory pipe the same whether the thread then
// feeds one system's recurrence with it or several.  With one system per thread the coefficient broadcasts are
// 13 of the ~15 shared-memory wavefronts per warp-row (profiles/r01_ncu_full.md: l1tex 72 %, the busiest unit of
// the solve kernel, and THE bound of the on-chip step kernel); a thread that carries SPT adjacent systems through
// the same chunk divides them by SPT (and gives the scheduler SPT independent FMA chains per warp).
// v[u][j] = row j of the thread's u-th system.  Same arithmetic, same order, per system, as the SPT = 1 functions.
template <typename T, int SPT>
__device__ __forceinline__ void lds_sys(T (&o)[SPT], const T* p)
{
    if constexpr (SPT == 1) o[0] = *p;
    else if constexpr (SPT * sizeof(T) == 8) {
        const float2 q = *reinterpret_cast<const float2*>(p);
        o[0] = q.x; o[1] = q.y;
    } else {
        static_assert((SPT * sizeof(T)) % 16 == 0, "systems per thread");
        lds_vec<T, SPT>(o, p);
    }
}
template <typename T, int SPT>
__device__ __forceinline__ void sts_sys(T* p, const T (&o)[SPT])
{
    if constexpr (SPT == 1) *p = o[0];
    else if constexpr (SPT * sizeof(T) == 8) *reinterpret_cast<float2*>(p) = make_float2(o[0], o[1]);
    else {
        static_assert(SPT * sizeof(T) == 16, "systems per thread");
        if constexpr (sizeof(T) == 8) *reinterpret_cast<double2*>(p) = make_double2(o[0], o[1]);
        else *reinterpret_cast<float4*>(p) = make_float4(o[0], o[1], o[2], o[3]);
    }
}

template <typename T, int SPT>
__device__ __forceinline__ void chunk_local_sweeps_n(T (&v)[SPT][ChunkCfg<T>::C], const T* blk,
                                                     typename Pair<T>::type (&e)[SPT], typename Pair<T>::type (&s)[SPT])
{
    constexpr int C = ChunkCfg<T>::C;
    T g1[SPT], g2[SPT];
#pragma unroll
    for (int u = 0; u < SPT; ++u) { g1[u] = 0; g2[u] = 0; }
#pragma unroll
    for (int jg = 0; jg < C / 4; ++jg) {
        T w[12];
        lds_vec<T, 12>(w, blk + 12 * jg);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int j = 4 * jg + r;
#pragma unroll
            for (int u = 0; u < SPT; ++u) {
                T t = w[3 * r] * v[u][j];
                t = fma(-w[3 * r + 1], g2[u], t);
                T g = fma(-w[3 * r + 2], g1[u], t);
                v[u][j] = g; g2[u] = g1[u]; g1[u] = g;
            }
        }
    }
    T x1[SPT], x2[SPT];
#pragma unroll
    for (int u = 0; u < SPT; ++u) { e[u].x = v[u][C - 2]; e[u].y = v[u][C - 1]; x1[u] = 0; x2[u] = 0; }
#pragma unroll
    for (int jg = C / 4 - 1; jg >= 0; --jg) {
        T w[8];
        lds_vec<T, 8>(w, blk + 3 * C + 8 * jg);
#pragma unroll
        for (int r = 3; r >= 0; --r) {
            const int j = 4 * jg + r;
#pragma unroll
            for (int u = 0; u < SPT; ++u) {
                T xv = fma(-w[2 * r], x1[u], fma(-w[2 * r + 1], x2[u], v[u][j]));
                v[u][j] = xv; x2[u] = x1[u]; x1[u] = xv;
            }
        }
    }
#pragma unroll
    for (int u = 0; u < SPT; ++u) { s[u].x = v[u][0]; s[u].y = v[u][1]; }
}

// stage 4, rows 4 jg .. 4 jg + 3 of every system of the thread: out[u][r]
template <typename T, int SPT>
__device__ __forceinline__ void chunk_correct4_n(T (&out)[SPT][4], const T (&v)[SPT][ChunkCfg<T>::C], const T* blk, int jg,
                                                 const T (&F0)[SPT], const T (&F1)[SPT], const T (&B0)[SPT], const T (&B1)[SPT])
{
    constexpr int C = ChunkCfg<T>::C;
    T w[16];
    lds_vec<T, 16>(w, blk + 5 * C + 16 * jg);
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int u = 0; u < SPT; ++u)
            out[u][r] = fma(w[4 * r + 3], B1[u], fma(w[4 * r + 2], B0[u], fma(w[4 * r + 1], F1[u], fma(w[4 * r], F0[u], v[u][4 * jg + r]))));
}

// ---- BAND = 1: the same three stages for a tridiagonal A (one-term recurrences) -----------------
// blk: [ {1/alpha, beta/alpha} x C | gamma x C | {chi, psi} x C ].  v: f -> x^ ; e = last g~ ; s = first x^.
template <typename T>
__device__ __forceinline__ void tri_local_sweeps(T (&v)[ChunkCfg<T>::C], const T* blk, T& e, T& s)
{
    constexpr int C = ChunkCfg<T>::C;
    T g1 = 0;
#pragma unroll
    for (int jg = 0; jg < C / 4; ++jg) {
        T w[8];
        lds_vec<T, 8>(w, blk + 8 * jg);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const int j = 4 * jg + r;
            T g = fma(-w[2 * r + 1], g1, w[2 * r] * v[j]);
            v[j] = g; g1 = g;
        }
    }
    e = v[C - 1];
    T x1 = 0;
#pragma unroll
    for (int jg = C / 4 - 1; jg >= 0; --jg) {
        T w[4];
        lds_vec<T, 4>(w, blk + 2 * C + 4 * jg);
#pragma unroll
        for (int r = 3; r >= 0; --r) {
            const int j = 4 * jg + r;
            T xv = fma(-w[r], x1, v[j]);
            v[j] = xv; x1 = xv;
        }
    }
    s = v[0];
}

template <typename T>
__device__ __forceinline__ void tri_correct4(T (&out)[4], const T* v4, const T* blk, int jg, T F, T B)
{
    constexpr int C = ChunkCfg<T>::C;
    T w[8];
    lds_vec<T, 8>(w, blk + 3 * C + 8 * jg);
#pragma unroll
    for (int r = 0; r < 4; ++r) out[r] = fma(w[2 * r + 1], B, fma(w[2 * r], F, v4[r]));
}

// Chunk states live in shared memory as [chunk][system] with the system index rotated by the chunk
// index.  The sweep threads (consecutive lanes = consecutive systems of one chunk) and the scan
// threads (consecutive lanes = consecutive chunks of one system) then both touch every bank group
// equally: the plain [chunk][system] layout made the scan read with a 32-way bank conflict
// (9.5 M conflicts per cfg3 launch, profiles/r01_solve_chunked_ncu_full.md).
template <int S>
__device__ __forceinline__ int state_slot(int chunk, int sys)
{
#ifdef PENT_AB_PLAIN_STATE
    return chunk * S + sys;
#else
    return chunk * S + ((sys + chunk) & (S - 1));
#endif
}

// Geometry of the chunk-state scan (stage 3): a group of Pw lanes scans one system, lane = chunk.
struct ScanGeom {
    int P, Pw, lev_f, lev_b;
    const int* woff;      // w_level_off(P, l), l < W_LEVELS
};

constexpr int BAR_F = 1 + 2 * MAX_BOXES, BAR_B = 2 + 2 * MAX_BOXES, NUM_BARS = 3 + 2 * MAX_BOXES;

// Periodic (cyclic) systems, Eqs. 8-12, fused into the scan: the kernel solves y = E^{-1} f^
// for the (N-2) x (N-2) block E (n = N-2 rows) and needs, per system,
//     t = S2^{-1} [ (f_n, f_{n+1}) - h^T y ],     h^T y = six entries: y_0, y_1, y_{n-2}, y_{n-1}
// before it can store x^ = y - Z t.  (y_0, y_1) is the true state B of the first chunk;
// y_{n-2}, y_{n-1} are rows (pa, ja), (pb, jb) of cluster rank ra (the last rank with real rows, whose
// state entering from the right is zero, so its values are final right after its own scan).
template <typename T>
struct PeriodicParams {                   // kernel parameter (constant bank)
    int ra, pa, ja, pb, jb;               // location of rows n-2 and n-1: cluster rank, local chunk, row in chunk
    T h00, h0a, h0b, h10, h11, h1a;       // h (Eq. 9): row N-2 of A at cols 0, N-4, N-3; row N-1 at cols 0, 1, N-3
    T i00, i01, i10, i11;                 // inverse of the 2 x 2 Schur complement (Eq. 12)
    const T* fold;                        // chunk states of the Z solve, 8 values per GLOBAL chunk (periodic_fold_kernel)
    const typename Pair<T>::type* zedge;  // explicit rows of Z of chunk 0 and of the chunks of rows n-2, n-1: [3][C]
    const T* f;                           // the caller's right-hand side (rows n, n+1 are read directly)
};
template <typename T>
struct PeriodicCtx {
    const PeriodicParams<T>* pp;
    T* ypub;                              // smem [S][2]: x^ of rows n-2 / n-1 (written by the sweep threads of rank ra)
    typename Pair<T>::type *yab, *ftail, *stT;   // smem [S]: (y_{n-2}, y_{n-1}); (f_n, f_{n+1}); t
    const T* table;                       // smem chunk blocks (correction rows of chunks pa, pb)
    T* x; int64_t M, col0; int n;         // tail rows go to x[n*M + col], x[(n+1)*M + col]
};

// stage 3 for one (system, chunk q) lane: Kogge-Stone over chunks with warp shuffles.
//   F_q = E~_q + TPhi_q F_{q-1};  B_q = (S^_q + TX_q F_{q-1}) + TPsi_q B_{q+1}
// In:  stE[sl] = E~_q, stS[sl] = S^_q.  Out: stE[sl] = F_{q-1}, stS[sl] = B_{q+1} (what thread (sys, q)
// needs).  CLUSTER: the block aggregates travel between the CTAs of the cluster (rank = this
// CTA's position along k, Q CTAs) through aggF/aggB and the two aggregate mbarriers.
// PER: also computes t of the periodic reduction (PeriodicCtx) into per.stT[sys] and stores the two
// tail rows of x; in a cluster every rank then receives every rank's backward aggregate (not only
// the later ranks') plus (y_{n-2}, y_{n-1}) from rank ra, all under the same mbarrier phase.
// ---- lean scan for the on-chip step kernel (single CTA, non-periodic) ------------------------------------------
// In the step kernel the scan runs once per time step with the same lane -> chunk assignment, and it is a pure
// latency chain (per level: 64-bit shuffles + two dependent FMAs), so everything that does not depend on the data
// is taken off it (profiles/r02_step_spt.md: the branchy version below spent ~90 cycles per level on shared-memory
// address arithmetic and reconvergence points; the scan was 37 % of a step):
//   * the lane's base address and validity bits are computed ONCE per launch (ScanLane, made opaque so that the
//     compiler does not rematerialise them from the block geometry inside every step); the per-level offsets are
//     uniform and come from the constant bank (ScanOffsets);
//   * a lane that takes no part in a level gets a ZERO matrix through a predicated load (inline PTX: the
//     conditional expression compiled to a branch around the load), so a level is straight-line code;
//   * R systems per lane (register blocking as in the sweeps): the matrices are loaded once for the R systems and
//     their R shuffle -> FMA chains overlap.
// Levels beyond lev_f / lev_b (matrices below 1e-25) are still skipped by a uniform branch.  What remains is bound by
// the SHFL pipe (8 SHFL.32 per level and warp, all warps of the SM at once: ~150 cycles per level).
struct ScanOffsets {                  // byte offsets, relative to W, of element e of the level-l matrices of lane q = 0
    uint32_t f[W_LEVELS][4], b[W_LEVELS][4], tx[4];
};
template <typename T>
inline ScanOffsets make_scan_offsets(int P, const int* woff)
{
    ScanOffsets o;
    for (int l = 0; l < W_LEVELS; ++l) {
        const int d = 1 << l, n = P - d > 0 ? P - d : 0;
        for (int e = 0; e < 4; ++e) {
            o.f[l][e] = (uint32_t)((woff[l] + e * n - d) * (int)sizeof(T));
            o.b[l][e] = (uint32_t)((woff[l] + 4 * n + e * n) * (int)sizeof(T));
        }
    }
    for (int e = 0; e < 4; ++e) o.tx[e] = (uint32_t)(e * P * (int)sizeof(T));
    return o;
}
struct ScanLane {
    uint32_t abase;                               // shared-memory byte address of W + q * sizeof(T)
    uint32_t valid;                               // bit l: forward level l applies; bit 8 + l: backward; bit 16: q < P
};
template <typename T>
__device__ __forceinline__ ScanLane make_scan_lane(const ScanGeom& g, const T* wtab, int q)
{
    ScanLane s;
    const int P = g.P;
    s.valid = q < P ? 1u << 16 : 0u;
    s.abase = smem_u32(wtab) + (uint32_t)(q * (int)sizeof(T));
#pragma unroll
    for (int l = 0; l < W_LEVELS; ++l) {
        const int d = 1 << l;
        const bool vf = l < g.lev_f && q >= d && q < P, vb = l < g.lev_b && q + d <= P - 1;
        s.valid |= (vf ? 1u : 0u) << l | (vb ? 1u : 0u) << (8 + l);
    }
    asm volatile("" : "+r"(s.abase), "+r"(s.valid));
    return s;
}
// value at shared address `addr` if `on`, else 0: one predicated LDS, no branch
__device__ __forceinline__ double lds_if(uint32_t addr, uint32_t on, double)
{
    double v;
    asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\tmov.f64 %0, 0d0000000000000000;\n\t@p ld.shared.f64 %0, [%1];\n\t}"
        : "=d"(v) : "r"(addr), "r"(on));
    return v;
}
__device__ __forceinline__ float lds_if(uint32_t addr, uint32_t on, float)
{
    float v;
    asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\tmov.f32 %0, 0f00000000;\n\t@p ld.shared.f32 %0, [%1];\n\t}"
        : "=f"(v) : "r"(addr), "r"(on));
    return v;
}
// In: stE[sl[r]] = E~_q, stS[sl[r]] = S^_q of the lane's R systems.  Out: F_{q-1}, B_{q+1} in the same slots.
// sl[r] < 0: the lane has no r-th system (its states are zero and nothing is stored).
template <typename T, int R>
__device__ __forceinline__ void chunk_state_scan_lean(const ScanLane& ln, const ScanOffsets& so, int P, int Pw, int lev_f,
                                                      int lev_b, int q, typename Pair<T>::type* stE,
                                                      typename Pair<T>::type* stS, const int (&sl)[R])
{
    using T2 = typename Pair<T>::type;
    T y0[R], y1[R], z0[R], z1[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        y0[r] = 0; y1[r] = 0; z0[r] = 0; z1[r] = 0;
        if (sl[r] >= 0) { T2 e = stE[sl[r]]; y0[r] = e.x; y1[r] = e.y; T2 s = stS[sl[r]]; z0[r] = s.x; z1[r] = s.y; }
    }
#pragma unroll
    for (int l = 0; l < W_LEVELS; ++l) {
        if (l < lev_f) {
            const int d = 1 << l;
            const uint32_t on = ln.valid & (1u << l);
            const T m0 = lds_if(ln.abase + so.f[l][0], on, T()), m1 = lds_if(ln.abase + so.f[l][1], on, T()),
                    m2 = lds_if(ln.abase + so.f[l][2], on, T()), m3 = lds_if(ln.abase + so.f[l][3], on, T());
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T u0 = shfl_up_t(y0[r], d, Pw), u1 = shfl_up_t(y1[r], d, Pw);
                y0[r] = fma(m1, u1, fma(m0, u0, y0[r]));
                y1[r] = fma(m3, u1, fma(m2, u0, y1[r]));
            }
        }
    }
    T f0[R], f1[R];
    {
        const uint32_t on = ln.valid & (1u << 16);
        const T m0 = lds_if(ln.abase + so.tx[0], on, T()), m1 = lds_if(ln.abase + so.tx[1], on, T()),
                m2 = lds_if(ln.abase + so.tx[2], on, T()), m3 = lds_if(ln.abase + so.tx[3], on, T());
#pragma unroll
        for (int r = 0; r < R; ++r) {
            f0[r] = shfl_up_t(y0[r], 1, Pw); f1[r] = shfl_up_t(y1[r], 1, Pw);      // F_{q-1}
            if (q == 0) { f0[r] = 0; f1[r] = 0; }
            z0[r] = fma(m1, f1[r], fma(m0, f0[r], z0[r]));                         // TX_q F_{q-1}
            z1[r] = fma(m3, f1[r], fma(m2, f0[r], z1[r]));
        }
    }
#pragma unroll
    for (int l = 0; l < W_LEVELS; ++l) {
        if (l < lev_b) {
            const int d = 1 << l;
            const uint32_t on = ln.valid & (1u << (8 + l));
            const T m0 = lds_if(ln.abase + so.b[l][0], on, T()), m1 = lds_if(ln.abase + so.b[l][1], on, T()),
                    m2 = lds_if(ln.abase + so.b[l][2], on, T()), m3 = lds_if(ln.abase + so.b[l][3], on, T());
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const T u0 = shfl_down_t(z0[r], d, Pw), u1 = shfl_down_t(z1[r], d, Pw);
                z0[r] = fma(m1, u1, fma(m0, u0, z0[r]));
                z1[r] = fma(m3, u1, fma(m2, u0, z1[r]));
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        T b0 = shfl_down_t(z0[r], 1, Pw), b1 = shfl_down_t(z1[r], 1, Pw);          // B_{q+1}
        if (q >= P - 1) { b0 = 0; b1 = 0; }
        if (sl[r] >= 0) {
            T2 fo; fo.x = f0[r]; fo.y = f1[r]; stE[sl[r]] = fo;
            T2 bo; bo.x = b0; bo.y = b1; stS[sl[r]] = bo;
        }
    }
}

// NBR (CLUSTER, not PER): neighbour-only exchange.  When every block transfer product of the handle is below 1e-25
// (pent_handle::xdepth == 1: a state entering a block of >= 32 chunks has decayed to nothing by its end) the state
// entering this CTA's block is the adjacent rank's aggregate alone: one send and one receive per direction, no chain
// over the ranks.  A compile-time variant so that the full-exchange code (and its SASS) stays what it was.
template <typename T, int S, bool CLUSTER, bool PER = false, bool NBR = false>
__device__ __forceinline__ void chunk_state_scan(const ScanGeom& g, const T* wtab, typename Pair<T>::type* stE,
                                                 typename Pair<T>::type* stS, int sys, int q, bool ok,
                                                 int rank, int Q, typename Pair<T>::type* aggF,
                                                 typename Pair<T>::type* aggB, uint64_t* bars,
                                                 uint32_t agg_bytes_f, uint32_t agg_bytes_b, uint32_t parity,
                                                 const PeriodicCtx<T>* per = nullptr)
{
    using T2 = typename Pair<T>::type;
    constexpr int C = ChunkCfg<T>::C, BL = chunk_block_len<T>();
    const int P = g.P, Pw = g.Pw;
    const int sl = ok ? state_slot<S>(q, sys) : 0;
    const int sy = ok ? sys : 0;
    T y0 = 0, y1 = 0, z0 = 0, z1 = 0;
    if (ok) { T2 e = stE[sl]; y0 = e.x; y1 = e.y; T2 s = stS[sl]; z0 = s.x; z1 = s.y; }
#pragma unroll
    for (int l = 0; l < W_LEVELS; ++l) {
        if (l < g.lev_f) {
            const int d = 1 << l, n = P - d;
            T u0 = shfl_up_t(y0, d, Pw), u1 = shfl_up_t(y1, d, Pw);
            if (ok && q >= d) mat2_acc(y0, y1, wtab + g.woff[l] + (q - d), n, u0, u1);
        }
    }
    T fin0 = 0, fin1 = 0;                 // F entering this CTA's block of chunks
    if constexpr (CLUSTER) {
        // y = F of chunk q for a ZERO state entering the block.  The last chunk's value is the
        // block aggregate: send it to every later rank, then chain the earlier ranks' aggregates.
        if constexpr (NBR) {
            // two slots: [0] = the forward aggregate of the rank before, [1] = the backward aggregate of the rank after
            if (ok && q == P - 1 && rank + 1 < Q) st_async_pair(&aggF[sys], &bars[BAR_F], rank + 1, y0, y1);
            if (agg_bytes_f) mbar_wait(&bars[BAR_F], parity);
            if (rank > 0) { T2 a = aggF[sy]; fin0 = a.x; fin1 = a.y; }
        } else {
        if (ok && q == P - 1)
            for (int rr = rank + 1; rr < Q; ++rr) st_async_pair(&aggF[rank * S + sys], &bars[BAR_F], rr, y0, y1);
        if (agg_bytes_f) mbar_wait(&bars[BAR_F], parity);
        }
        for (int rr = 0; rr < (NBR ? 0 : rank); ++rr) {        // F_in(rr+1) = aggF[rr] + TPhiBlock(rr) F_in(rr)
            T2 a = aggF[rr * S + sy];
            T n0 = a.x, n1 = a.y;
            mat2_acc(n0, n1, wtab + 12 * P + 4 * rr, 1, fin0, fin1);
            fin0 = n0; fin1 = n1;
        }
        if (ok && rank > 0) mat2_acc(y0, y1, wtab + 4 * P + q, P, fin0, fin1);   // PF_q F_in
    }
    T f0 = shfl_up_t(y0, 1, Pw), f1 = shfl_up_t(y1, 1, Pw);      // F_{q-1}
    if (q == 0) { f0 = fin0; f1 = fin1; }
    if (ok) mat2_acc(z0, z1, wtab + q, P, f0, f1);               // TX_q F_{q-1}
#pragma unroll
    for (int l = 0; l < W_LEVELS; ++l) {
        if (l < g.lev_b) {
            const int d = 1 << l, n = P - d;
            T u0 = shfl_down_t(z0, d, Pw), u1 = shfl_down_t(z1, d, Pw);
            if (ok && q + d <= P - 1) mat2_acc(z0, z1, wtab + g.woff[l] + 4 * n + q, n, u0, u1);
        }
    }
    T ya = 0, yb = 0;                     // y_{n-2}, y_{n-1}
    if constexpr (PER) {
        // rank ra: nothing enters its block from the right, so z is the true B of its chunks already
        T bq0 = shfl_down_t(z0, 1, Pw), bq1 = shfl_down_t(z1, 1, Pw);
        if (q >= P - 1) { bq0 = 0; bq1 = 0; }
        if (ok && rank == per->pp->ra) {
            if (q == per->pp->pa) {
                const T* cr = per->table + (size_t)per->pp->pa * BL + 5 * C + 4 * per->pp->ja;
                ya = fma(cr[3], bq1, fma(cr[2], bq0, fma(cr[1], f1, fma(cr[0], f0, per->ypub[2 * sys]))));
            }
            if (q == per->pp->pb) {
                const T* cr = per->table + (size_t)per->pp->pb * BL + 5 * C + 4 * per->pp->jb;
                yb = fma(cr[3], bq1, fma(cr[2], bq0, fma(cr[1], f1, fma(cr[0], f0, per->ypub[2 * sys + 1]))));
            }
        }
        ya = __shfl_sync(0xffffffffu, ya, per->pp->pa, Pw);
        yb = __shfl_sync(0xffffffffu, yb, per->pp->pb, Pw);
    }
    T bin0 = 0, bin1 = 0;                 // B of the first chunk of the NEXT block
    T B00 = 0, B01 = 0;                   // PER: (y_0, y_1) = true B of the system's first chunk
    if constexpr (CLUSTER) {
        if (ok && q == 0) {
            if constexpr (PER) {
                for (int rr = 0; rr < Q; ++rr) st_async_pair(&aggB[rank * S + sys], &bars[BAR_B], rr, z0, z1);
                if (rank == per->pp->ra)
                    for (int rr = 0; rr < Q; ++rr) st_async_pair(&per->yab[sys], &bars[BAR_B], rr, ya, yb);
            } else if constexpr (NBR) {
                if (rank > 0) st_async_pair(&aggB[S + sys], &bars[BAR_B], rank - 1, z0, z1);
            } else {
                for (int rr = 0; rr < rank; ++rr) st_async_pair(&aggB[rank * S + sys], &bars[BAR_B], rr, z0, z1);
            }
        }
        if (agg_bytes_b) mbar_wait(&bars[BAR_B], parity);
        if constexpr (NBR) {
            if (rank < Q - 1) { T2 a = aggB[S + sy]; bin0 = a.x; bin1 = a.y; }
        }
        for (int rr = Q - 1; rr > (NBR ? Q - 1 : rank); --rr) {   // B_in(rr-1) = aggB[rr] + TPsiBlock(rr) B_in(rr)
            T2 a = aggB[rr * S + sy];
            T n0 = a.x, n1 = a.y;
            mat2_acc(n0, n1, wtab + 12 * P + 4 * PENT_MAXQ + 4 * rr, 1, bin0, bin1);
            bin0 = n0; bin1 = n1;
        }
        if (ok && rank < Q - 1) mat2_acc(z0, z1, wtab + 8 * P + q, P, bin0, bin1);   // PB_q B_in
        if constexpr (PER) {
            for (int rr = Q - 1; rr >= 0; --rr) {  // continue the chain down to the first block: B of chunk 0
                T2 a = aggB[rr * S + sy];
                T n0 = a.x, n1 = a.y;
                mat2_acc(n0, n1, wtab + 12 * P + 4 * PENT_MAXQ + 4 * rr, 1, B00, B01);
                B00 = n0; B01 = n1;
            }
            T2 yy = per->yab[sy];
            ya = yy.x; yb = yy.y;
        }
    } else if constexpr (PER) {
        B00 = __shfl_sync(0xffffffffu, z0, 0, Pw);
        B01 = __shfl_sync(0xffffffffu, z1, 0, Pw);
    }
    T b0 = shfl_down_t(z0, 1, Pw), b1 = shfl_down_t(z1, 1, Pw);  // B_{q+1}
    if (q >= P - 1) { b0 = bin0; b1 = bin1; }
    if (ok) {
        T2 fo; fo.x = f0; fo.y = f1; stE[sl] = fo;
        T2 bo; bo.x = b0; bo.y = b1; stS[sl] = bo;
    }
    if constexpr (PER) {
        if (ok && q == 0) {
            const T2 ft = per->ftail[sys];
            const T r0 = ft.x - fma(per->pp->h0b, yb, fma(per->pp->h0a, ya, per->pp->h00 * B00));
            const T r1 = ft.y - fma(per->pp->h1a, yb, fma(per->pp->h11, B01, per->pp->h10 * B00));
            T2 t;
            t.x = fma(per->pp->i01, r1, per->pp->i00 * r0);
            t.y = fma(per->pp->i11, r1, per->pp->i10 * r0);
            per->stT[sys] = t;
            if (rank == 0 && per->col0 + sys < per->M) {
                per->x[(int64_t)per->n * per->M + per->col0 + sys] = t.x;
                per->x[(int64_t)(per->n + 1) * per->M + per->col0 + sys] = t.y;
            }
        }
    }
}

// stage 3 for BAND = 1: scalar states, scalar transfer coefficients (layout: see w_level_off with BAND = 1).
//   F_q = E~_q + TPhi_q F_{q-1};  B_q = (S^_q + TX_q F_{q-1}) + TPsi_q B_{q+1}
template <typename T, int S, bool CLUSTER, bool NBR = false>
__device__ __forceinline__ void tri_state_scan(const ScanGeom& g, const T* wtab, T* stE, T* stS, int sys, int q, bool ok,
                                               int rank, int Q, T* aggF, T* aggB, uint64_t* bars,
                                               uint32_t agg_bytes_f, uint32_t agg_bytes_b, uint32_t parity)
{
    const int P = g.P, Pw = g.Pw;
    const int sl = ok ? state_slot<S>(q, sys) : 0;
    const int sy = ok ? sys : 0;
    T y = 0, z = 0;
    if (ok) { y = stE[sl]; z = stS[sl]; }
#pragma unroll
    for (int l = 0; l < W_LEVELS; ++l) {
        if (l < g.lev_f) {
            const int d = 1 << l;
            T u = shfl_up_t(y, d, Pw);
            if (ok && q >= d) y = fma(wtab[g.woff[l] + (q - d)], u, y);
        }
    }
    T fin = 0;
    if constexpr (CLUSTER) {
        if constexpr (NBR) {
            if (ok && q == P - 1 && rank + 1 < Q) st_async_one(&aggF[sys], &bars[BAR_F], rank + 1, y);
            if (agg_bytes_f) mbar_wait(&bars[BAR_F], parity);
            if (rank > 0) fin = aggF[sy];
        } else {
        if (ok && q == P - 1)
            for (int rr = rank + 1; rr < Q; ++rr) st_async_one(&aggF[rank * S + sys], &bars[BAR_F], rr, y);
        if (agg_bytes_f) mbar_wait(&bars[BAR_F], parity);
        for (int rr = 0; rr < rank; ++rr) fin = fma(wtab[3 * P + rr], fin, aggF[rr * S + sy]);
        }
        if (ok && rank > 0) y = fma(wtab[P + q], fin, y);                     // PF_q F_in
    }
    T f = shfl_up_t(y, 1, Pw);
    if (q == 0) f = fin;
    if (ok) z = fma(wtab[q], f, z);                                           // TX_q F_{q-1}
#pragma unroll
    for (int l = 0; l < W_LEVELS; ++l) {
        if (l < g.lev_b) {
            const int d = 1 << l, n = P - d;
            T u = shfl_down_t(z, d, Pw);
            if (ok && q + d <= P - 1) z = fma(wtab[g.woff[l] + n + q], u, z);
        }
    }
    T bin = 0;
    if constexpr (CLUSTER) {
        if constexpr (NBR) {
            if (ok && q == 0 && rank > 0) st_async_one(&aggB[S + sys], &bars[BAR_B], rank - 1, z);
            if (agg_bytes_b) mbar_wait(&bars[BAR_B], parity);
            if (rank < Q - 1) bin = aggB[S + sy];
        } else {
        if (ok && q == 0)
            for (int rr = 0; rr < rank; ++rr) st_async_one(&aggB[rank * S + sys], &bars[BAR_B], rr, z);
        if (agg_bytes_b) mbar_wait(&bars[BAR_B], parity);
        for (int rr = Q - 1; rr > rank; --rr) bin = fma(wtab[3 * P + PENT_MAXQ + rr], bin, aggB[rr * S + sy]);
        }
        if (ok && rank < Q - 1) z = fma(wtab[2 * P + q], bin, z);             // PB_q B_in
    }
    T b = shfl_down_t(z, 1, Pw);
    if (q >= P - 1) b = bin;
    if (ok) { stE[sl] = f; stS[sl] = b; }
}

// ------------------------------------------------------------------------------------------
// host side (defined in pent_solve_chunked.cu)
// ------------------------------------------------------------------------------------------
// A launch plan: cluster size Q (CTAs along k), S systems per tile, Pl chunks per CTA.
struct ChunkPlan {
    bool ok = false;
    int j = 0, Q = 1, S = 0, Pl = 0, Pw = 1, threads = 0, levels = 0, box_rows = 0, nbox = 0;
    bool ldg = false;          // LDG loader instead of TMA (pitch not a multiple of 16 bytes, or system-major batch)
    bool rows = false;         // system-major batch: implies ldg
    int pace_ns = 0;           // ChunkParams::pace_ns
    int band = 2;              // 1: the tridiagonal instantiation and its tables (handle with a == e == 0)
    bool nbr = false;          // neighbour-only cluster exchange (two [S] aggregate slots instead of [Q][S]); LM = 0, not periodic
    int mode = 0;              // ChunkParams::ldg: 0 TMA (interleaved), 1 LDG (interleaved), 4 cp.async ring (interleaved), 2 LDG.256 (system-major),
                               // 3 swizzled TMA loads + STG.256 stores, 4 swizzled TMA loads AND stores (system-major)
    size_t table_bytes = 0, smem = 0;
};
// any_S: accept tile widths the SOLVE kernel is not instantiated for (the step kernel has its own)
// ldg: plan for the LDG loader (no TMA alignment requirements, no landing buffer)
ChunkPlan make_plan(const pent_handle* h, int64_t M, const void* f, int Q, int S, bool any_S = false,
                    bool ldg = false, int band = 2);
void plan_drop_nbr(ChunkPlan& pl, size_t esz);
ChunkPlan chunk_auto_plan(const pent_handle* h, int64_t M, const void* f, bool ring_ok = true);   // what PENT_KERNEL_AUTO runs
// rank-2 tensor map {M, N} of an interleaved batch with box {S, box_rows}; false on failure
bool encode_batch_map(CUtensorMap* tm, const void* base, int64_t M, int N, int S, int box_rows, bool f64);
bool encode_batch_map_cached(CUtensorMap* tm, const void* base, int64_t M, int N, int S, int box_rows, bool f64);
// launch of a system-major plan (pent_solve_chunked_rows.cu: the LM = 2, 3, 4 instantiations of the kernel)
int launch_plan_rows(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s);
// the same plans launched with the 2 x - f epilogue (pent_solve_chunked_epi.cu: BAND = 2, all-ranks exchange, LM 0, 2, 5, 6)
int launch_plan_epi(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s);
// rank-2 tensor map {N, M} of a system-major batch with box {128 bytes, S} and SWIZZLE_128B
bool encode_rows_map_cached(CUtensorMap* tm, const void* base, int64_t M, int N, int S, bool f64);

}  // namespace pent
