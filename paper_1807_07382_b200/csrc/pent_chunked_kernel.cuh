// pent_chunked_kernel.cuh -- device code of the chunked on-chip solve (included by
// pent_solve_chunked.cu inside namespace pent; see the algorithm notes at the top of that file).
#pragma once

// Measured A/B switches (cfg3 fp64 on B200, profiles/r01_ab_tuning.md).  Defaults = fastest:
//   store policy of the x stream: plain write-back st.global (201 us) beat .cs (212), .cg (210), .wt (211)
//   chunk-state layout: [P][S] (197 us with 256-B L2 promotion) beat the bank-conflict-free padded
//   [S][P+1] (221 us) although the scan then reads with a 32-way conflict: see DESIGN.md section 6.2.
#if defined(PENT_AB_ST_CS)
#define PENT_STORE(p, v) __stcs((p), (v))
#elif defined(PENT_AB_ST_CG)
#define PENT_STORE(p, v) __stcg((p), (v))
#elif defined(PENT_AB_ST_WT)
#define PENT_STORE(p, v) __stwt((p), (v))
#else
#define PENT_STORE(p, v) (*(p) = (v))
#endif

template <typename T>
struct ChunkParams {
    int N;            // rows
    int P;            // chunks per CTA (local chunks; the system has Q*P chunks)
    int Q;            // CTAs per cluster (k is split across them); 1 = no cluster
    int Pw;           // P rounded up to a power of two (lanes per system in the chunk-state scan)
    int lev_f, lev_b; // Kogge-Stone levels to apply (<= log2 Pw)
    int woff[W_LEVELS]; // w_level_off(P, l)
    int box_rows;     // rows per TMA box
    int nbox;         // boxes per tile
    int wcount[MAX_BOXES]; // warps that read each box (arrival count of its "empty" barrier)
    uint32_t table_bytes;  // bytes of the per-CTA table staged into shared memory
    int64_t table_stride;  // elements between the tables of consecutive cluster ranks
    int64_t M;
    int64_t ntiles;
    const T* table;   // global coefficient tables (layout = shared-memory layout), one per rank
    T* x;
};

template <typename T> struct Pair;
template <> struct Pair<double> { using type = double2; };
template <> struct Pair<float>  { using type = float2; };

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

// One CTA = S systems x P chunks (thread = one system, one chunk of C rows, held in registers).
// blockDim.x >= P*S (a multiple of 32); threads with p >= P only take part in barriers/scan.
// CLUSTER: the Q CTAs of a cluster own consecutive blocks of P chunks of the SAME S systems; the
// chunk states are stitched across CTAs through distributed shared memory (two exchanges per tile).
constexpr int BAR_F = 1 + 2 * MAX_BOXES, BAR_B = 2 + 2 * MAX_BOXES, NUM_BARS = 3 + 2 * MAX_BOXES;

template <typename T, int S, bool CLUSTER>
__global__ void __launch_bounds__(CHUNK_MAX_THREADS, 1)
solve_chunked_kernel(const __grid_constant__ CUtensorMap tm, const ChunkParams<T> prm)
{
    constexpr int C = ChunkCfg<T>::C, BL = chunk_block_len<T>();
    using T2 = typename Pair<T>::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int P = prm.P;
    T* landing = reinterpret_cast<T*>(smem_raw);
    T* table = landing + (size_t)prm.nbox * prm.box_rows * S;
    // chunk states [P][S]: E~ then F_{p-1};  S^ then B_{p+1}
    T2* stE = reinterpret_cast<T2*>(reinterpret_cast<unsigned char*>(table) + prm.table_bytes);
    T2* stS = stE + (size_t)S * P;
    // cluster: block aggregates of every rank, [Q][S] each (written by the owning rank through DSMEM)
    T2* aggF = stS + (size_t)S * P;
    T2* aggB = aggF + (CLUSTER ? (size_t)prm.Q * S : 0);
    uint64_t* bars = reinterpret_cast<uint64_t*>(aggB + (CLUSTER ? (size_t)prm.Q * S : 0));

    const int tid = threadIdx.x, i = tid % S, p = tid / S;
    const bool active = p < P;
    const int lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const uint32_t box_bytes = (uint32_t)(prm.box_rows * S * sizeof(T));
    const int rank = CLUSTER ? (int)__clusterRelativeBlockRank() : 0;
    const int row_base = rank * P * C;                       // first row of this CTA's block
    const int64_t stride = CLUSTER ? (int64_t)__clusterGridDimInClusters().x : (int64_t)gridDim.x;
    const int64_t first = CLUSTER ? (int64_t)__clusterIdx().x : (int64_t)blockIdx.x;

    if (tid == 0) {
        for (int b = 0; b <= MAX_BOXES; ++b) mbar_init(&bars[b], 1);
        for (int b = 0; b < MAX_BOXES; ++b)
            mbar_init(&bars[1 + MAX_BOXES + b], prm.wcount[b] > 0 ? prm.wcount[b] : 1);
        mbar_init(&bars[BAR_F], 1);
        mbar_init(&bars[BAR_B], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    int64_t tile = first;
    if (tid == 0) {
        mbar_expect_tx(&bars[0], prm.table_bytes);
        bulk_load_1d(table, prm.table + (size_t)rank * prm.table_stride, prm.table_bytes, &bars[0]);
        if (tile < prm.ntiles)
            for (int b = 0; b < prm.nbox; ++b) {
                mbar_expect_tx(&bars[1 + b], box_bytes);
                tma_load_2d(landing + (size_t)b * prm.box_rows * S, &tm, (int)(tile * S),
                            row_base + b * prm.box_rows, &bars[1 + b]);
            }
    }
    // every CTA of the cluster is resident, with its mbarriers initialised, before any DSMEM store
    if constexpr (CLUSTER) cluster_sync_all();
    const uint32_t agg_bytes_f = (uint32_t)(rank * S * sizeof(T2));                 // from the earlier ranks
    const uint32_t agg_bytes_b = (uint32_t)((prm.Q - 1 - rank) * S * sizeof(T2));   // from the later ranks
    mbar_wait(&bars[0], 0);

    const T* blk = table + (size_t)(active ? p : 0) * BL;
    const T* wtab = table + (size_t)P * BL;          // W: TX | PF | PB | BLK | levels
    const int mybox = active ? (p * C) / prm.box_rows : 0;
    const int slot = (active ? p : 0) * S + i;
    const int row0 = row_base + p * C;
    const bool rows_full = active && (row0 + C <= prm.N);
    uint32_t parity = 0;

    // chunk-state scan geometry: a group of Pw lanes scans one system; G groups per warp
    const int Pw = prm.Pw, G = 32 / Pw;
    const int q = lane % Pw, grp = lane / Pw;
    const int rounds = (S + nwarps * G - 1) / (nwarps * G);     // host guarantees 1 when CLUSTER

    for (; tile < prm.ntiles; tile += stride) {
        const int64_t next_tile = tile + stride;
        T v[C];
        if (active) {
            // ---- tile data: landing buffer -> registers ----
            mbar_wait(&bars[1 + mybox], parity);
            const T* src = landing + (size_t)p * C * S + i;
#pragma unroll
            for (int j = 0; j < C; ++j) v[j] = src[j * S];
        }
        // The box is free once every warp that reads it has its values in registers: each such
        // warp arrives on the box's "empty" barrier and thread 0 re-arms it with the NEXT tile's
        // TMA load, which then runs under all of this tile's arithmetic and stores.
        __syncwarp();
        if (lane == 0 && warp * 32 < P * S) mbar_arrive(&bars[1 + MAX_BOXES + mybox]);
        if constexpr (CLUSTER) {
            if (tid == 0) {        // arm this tile's aggregate barriers (complete_tx may already have arrived)
                if (agg_bytes_f) mbar_expect_tx(&bars[BAR_F], agg_bytes_f);
                if (agg_bytes_b) mbar_expect_tx(&bars[BAR_B], agg_bytes_b);
            }
        }
        if (tid == 0 && next_tile < prm.ntiles) {
            for (int b = 0; b < prm.nbox; ++b) {
                mbar_wait(&bars[1 + MAX_BOXES + b], parity);
                mbar_expect_tx(&bars[1 + b], box_bytes);
                tma_load_2d(landing + (size_t)b * prm.box_rows * S, &tm, (int)(next_tile * S),
                            row_base + b * prm.box_rows, &bars[1 + b]);
            }
        }
        if (active) {
            // ---- 1. local forward sweep from a zero state (normalised) ----
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
            T2 e; e.x = v[C - 2]; e.y = v[C - 1];
            stE[slot] = e;
            // ---- 2. local back substitution of g~ from a zero state ----
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
            T2 s; s.x = v[0]; s.y = v[1];
            stS[slot] = s;
        }
        __syncthreads();       // states published

        // ---- 3. chunk-state scans: Kogge-Stone over chunks with warp shuffles ----
        //   F_q = E~_q + TPhi_q F_{q-1};  B_q = (S^_q + TX_q F_{q-1}) + TPsi_q B_{q+1}
        // Slot (q, sys) receives what thread (sys, q) needs: F_{q-1} and B_{q+1}.
        if (CLUSTER || P > 1) {
            for (int r = 0; r < rounds; ++r) {
                const int sys = (r * nwarps + warp) * G + grp;
                const bool ok = (sys < S) && (q < P);
                const int sl = ok ? q * S + sys : 0;
                T y0 = 0, y1 = 0, z0 = 0, z1 = 0;
                if (ok) { T2 e = stE[sl]; y0 = e.x; y1 = e.y; T2 s = stS[sl]; z0 = s.x; z1 = s.y; }
#pragma unroll
                for (int l = 0; l < W_LEVELS; ++l) {
                    if (l < prm.lev_f) {
                        const int d = 1 << l, n = P - d;
                        T u0 = shfl_up_t(y0, d, Pw), u1 = shfl_up_t(y1, d, Pw);
                        if (ok && q >= d) mat2_acc(y0, y1, wtab + prm.woff[l] + (q - d), n, u0, u1);
                    }
                }
                T fin0 = 0, fin1 = 0;                 // F entering this CTA's block of chunks
                if constexpr (CLUSTER) {
                    // y = F of chunk q for a ZERO state entering the block.  The last chunk's value is
                    // the block aggregate: publish it to every later rank, then chain the earlier ones.
                    if (ok && q == P - 1)
                        for (int rr = rank + 1; rr < prm.Q; ++rr)
                            st_async_pair(&aggF[rank * S + sys], &bars[BAR_F], rr, y0, y1);
                    if (agg_bytes_f) mbar_wait(&bars[BAR_F], parity);
                    for (int rr = 0; rr < rank; ++rr) {        // F_in(rr+1) = aggF[rr] + TPhiBlock(rr) F_in(rr)
                        T2 a = aggF[rr * S + (ok ? sys : 0)];
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
                    if (l < prm.lev_b) {
                        const int d = 1 << l, n = P - d;
                        T u0 = shfl_down_t(z0, d, Pw), u1 = shfl_down_t(z1, d, Pw);
                        if (ok && q + d <= P - 1) mat2_acc(z0, z1, wtab + prm.woff[l] + 4 * n + q, n, u0, u1);
                    }
                }
                T bin0 = 0, bin1 = 0;                 // B of the first chunk of the NEXT block
                if constexpr (CLUSTER) {
                    if (ok && q == 0)
                        for (int rr = 0; rr < rank; ++rr)
                            st_async_pair(&aggB[rank * S + sys], &bars[BAR_B], rr, z0, z1);
                    if (agg_bytes_b) mbar_wait(&bars[BAR_B], parity);
                    for (int rr = prm.Q - 1; rr > rank; --rr) {   // B_in(rr-1) = aggB[rr] + TPsiBlock(rr) B_in(rr)
                        T2 a = aggB[rr * S + (ok ? sys : 0)];
                        T n0 = a.x, n1 = a.y;
                        mat2_acc(n0, n1, wtab + 12 * P + 32 + 4 * rr, 1, bin0, bin1);
                        bin0 = n0; bin1 = n1;
                    }
                    if (ok && rank < prm.Q - 1) mat2_acc(z0, z1, wtab + 8 * P + q, P, bin0, bin1);   // PB_q B_in
                }
                T b0 = shfl_down_t(z0, 1, Pw), b1 = shfl_down_t(z1, 1, Pw);  // B_{q+1}
                if (q >= P - 1) { b0 = bin0; b1 = bin1; }
                if (ok) {
                    T2 fo; fo.x = f0; fo.y = f1; stE[sl] = fo;
                    T2 bo; bo.x = b0; bo.y = b1; stS[sl] = bo;
                }
            }
        }
        __syncthreads();

        // ---- 4. correction and store ----
        if (active) {
            T F0 = 0, F1 = 0, B0 = 0, B1 = 0;
            if (CLUSTER || P > 1) { T2 fo = stE[slot]; F0 = fo.x; F1 = fo.y; T2 bo = stS[slot]; B0 = bo.x; B1 = bo.y; }
            const int64_t col = tile * S + i;
            T* xo = prm.x + (int64_t)row0 * prm.M + col;
            if (rows_full && (tile + 1) * S <= prm.M) {
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T w[16];
                    lds_vec<T, 16>(w, blk + 5 * C + 16 * jg);
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        T xv = fma(w[4 * r + 3], B1, fma(w[4 * r + 2], B0,
                               fma(w[4 * r + 1], F1, fma(w[4 * r], F0, v[4 * jg + r]))));
                        PENT_STORE(xo, xv);
                        xo += prm.M;
                    }
                }
            } else if (col < prm.M) {
                const int nrows = prm.N - row0;      // may be <= 0
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T w[16];
                    lds_vec<T, 16>(w, blk + 5 * C + 16 * jg);
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        T xv = fma(w[4 * r + 3], B1, fma(w[4 * r + 2], B0,
                               fma(w[4 * r + 1], F1, fma(w[4 * r], F0, v[4 * jg + r]))));
                        if (4 * jg + r < nrows) PENT_STORE(xo, xv);
                        xo += prm.M;
                    }
                }
            }
        }
        parity ^= 1;
    }
    if constexpr (CLUSTER) cluster_sync_all();   // no CTA leaves while a peer may still address its shared memory
}
