// pent_chunked_kernel.cuh -- device code of the chunked on-chip solve (included by
// pent_solve_chunked.cu inside namespace pent; see the algorithm notes at the top of that file).
#pragma once

// Measured A/B switches (cfg3 fp64 on B200, profiles/r01_ab_tuning.md).  Default = fastest:
//   store policy of the x stream: plain write-back st.global (201 us) beat .cs (212), .cg (210), .wt (211)
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
    int land_rows;    // rows of the landing buffer (nbox * box_rows for TMA; P * C for the cp.async loader; 0: none)
    int wcount[MAX_BOXES]; // warps that read each box (arrival count of its "empty" barrier)
    uint32_t table_bytes;  // bytes of the per-CTA table staged into shared memory
    int64_t table_stride;  // elements between the tables of consecutive cluster ranks
    int64_t M;
    int64_t ntiles;
    const T* table;   // global coefficient tables (layout = shared-memory layout), one per rank
    const T* f;       // right-hand side (used by the LDG loader)
    unsigned pace_ns; // sleep this long before the store stage (0: none)
    int ldg;          // 1: the pitch M*sizeof(T) is not a multiple of 16 bytes, so TMA cannot address the batch:
                      // every thread loads its rows with coalesced LDG instead (no landing buffer, nbox = 0)
                      // 4: the same batch through per-thread cp.async copies (LDGSTS) into a landing buffer, one tile ahead:
                      // every thread copies the C rows IT will read, so it waits only for its own copies (no barrier)
                      // and re-issues them for the next tile as soon as its values are in registers
                      // 2: SYSTEM-MAJOR batch ("one system per row", the paper's serial layout):
                      // element k of system i at f[i*N + k]; a thread's chunk is one contiguous run of C
                      // elements, loaded and stored with 32-byte vector accesses
                      // 3: system-major batch through TMA: the tensor map is {N, M} with 128-byte x S boxes and
                      // SWIZZLE_128B, so the global side moves whole 128-byte pieces of every system (prefetched one
                      // tile ahead like the interleaved loader) and a thread reads its run out of the swizzled
                      // landing buffer with conflict-free LDS.128; stores as in mode 2
                      // 5: system-major batch through 1-D bulk copies (cp.async.bulk, UBLKCP): ONE copy per system and tile
                      // moves that system's whole run of this CTA's rows into a landing buffer whose per-system pitch is
                      // padded by 16 bytes (conflict-free LDS.128); prefetched one tile ahead.  The tensor-tile TMA of
                      // mode 3 is bound by its row rate (~8 ns per 128-byte row and SM, profiles/r02_rows_loader.md);
                      // a 1-D bulk copy has no rows.  Stores as in mode 2.
                      // 6: mode 5 with the stores through 1-D bulk copies too (x -> padded staging buffer -> one
                      // copy per system): x leaves as whole lines instead of 32-byte sectors
    T* x;
};

// PER = true: the periodic (cyclic) solve fused into the kernel, see PeriodicCtx in pent_chunk_common.cuh.
// BAND = 1: tridiagonal A (a == e == 0, cuThomasBatch's case): one-term recurrences, a 5-word
// coefficient row instead of 9, scalar chunk states; same data movement.
// LM = layout / loader mode, compile-time so that every instantiation carries only its own data path (a run-time
// switch over all of them cost 80-120 bytes of register spills in every instance): 0 = interleaved batch (TMA, or
// the LDG loader when prm.ldg == 1); 2, 3, 4 = system-major batch, the modes described at ChunkParams::ldg.
// NBR: neighbour-only cluster exchange (see chunk_state_scan); chosen by the plan (ChunkPlan::nbr) for Q >= 8 when the handle allows it.
// EPI: the kernel stores 2 x - f instead of x (f = its own right-hand side, re-read from global memory / L2 just before the
// store; x == f allowed).  With A = I - (dt/2) D this is (2I - A) A^{-1} f, the explicit half of the NEXT half step of a
// Peaceman-Rachford ADI sweep (pent_adi.cu): the stencil kernels between the solves disappear.
template <typename T, int S, bool CLUSTER, bool PER, int BAND, int LM, bool NBR = false, bool EPI = false>
__global__ void __launch_bounds__(CHUNK_MAX_THREADS, 1)
solve_chunked_kernel(const __grid_constant__ CUtensorMap tm, const ChunkParams<T> prm,
                     const __grid_constant__ PeriodicParams<T> pp, const __grid_constant__ CUtensorMap tmx)
{
    static_assert(BAND == 2 || !PER, "the fused periodic tail is built on the pentadiagonal tables");
    static_assert(LM == 0 || !PER, "periodic handles take interleaved batches only");
    constexpr int C = ChunkCfg<T>::C, BL = chunk_block_len<T, BAND>();
    using T2 = typename Pair<T>::type;
    using ST = typename ChunkState<T, BAND>::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int P = prm.P;
    // (mode 3: the 128-byte swizzle pattern repeats every 1024 bytes of the shared-memory ADDRESS)
    T* landing = reinterpret_cast<T*>(LM == 3 ? smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u) : smem_raw);
    // modes 5, 6: one padded run per system (pitch in bytes); mode 6: a staging buffer of the same size and layout
    const uint32_t run_pitch = (uint32_t)(prm.box_rows * sizeof(T)) + 16u;
    const size_t tile_elems = LM >= 5 ? (size_t)S * run_pitch / sizeof(T) : (size_t)prm.land_rows * S;
    T* staging = landing + tile_elems;
    T* table = staging + (LM == 6 ? tile_elems : 0);
    // chunk states [P][S]: E~ then F_{p-1};  S^ then B_{p+1}
    ST* stE = reinterpret_cast<ST*>(reinterpret_cast<unsigned char*>(table) + prm.table_bytes);
    ST* stS = stE + (size_t)S * P;
    // cluster: block aggregates of every rank, [Q][S] each (written by the owning rank through DSMEM)
    // Slot rr holds rank rr's FORWARD aggregate when rr < rank and its BACKWARD aggregate when rr > rank
    // (a CTA needs nothing else), so both directions share one array; the periodic kernel needs every
    // rank's backward aggregate and keeps two.
    ST* aggF = stS + (size_t)S * P;
    ST* aggB = aggF + ((CLUSTER && PER) ? (size_t)prm.Q * S : 0);
    // periodic: the Z-solve chunk states of this CTA's chunks (8 values each), the explicit rows of Z of the three edge
    // chunks, then x^ of rows n-2/n-1, (y_{n-2}, y_{n-1}), (f_n, f_{n+1}), t  ([S] each)
    T2* zfold = reinterpret_cast<T2*>(aggB + (CLUSTER ? (NBR ? (size_t)2 * S : (size_t)prm.Q * S) : 0));
    T2* zedge = zfold + (PER ? (size_t)4 * P : 0);
    T2* ypub = zedge + (PER ? (size_t)3 * C : 0);
    T2* yab = ypub + (PER ? S : 0);
    T2* ftail2 = yab + (PER ? S : 0);             // [2][S]
    T2* stT = ftail2 + (PER ? 2 * S : 0);
    uint64_t* bars = reinterpret_cast<uint64_t*>(stT + (PER ? S : 0));

    const int tid = threadIdx.x, i = tid % S, p = tid / S;
    const bool active = p < P;
    const int lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
    const uint32_t box_bytes = (uint32_t)(prm.box_rows * S * sizeof(T));
    const int rank = CLUSTER ? (int)__clusterRelativeBlockRank() : 0;
    const int row_base = rank * P * C;                       // first row of this CTA's block
    const int64_t stride = CLUSTER ? (int64_t)__clusterGridDimInClusters().x : (int64_t)gridDim.x;
    const int64_t first = CLUSTER ? (int64_t)__clusterIdx().x : (int64_t)blockIdx.x;

    // TMA load(s) of barrier group b (box_rows rows x S systems) of tile t, signalling bars[1 + b]
    auto issue_box = [&](int b, int64_t t) {
        if constexpr (LM >= 5) {
            // one 1-D bulk copy per system of the tile: its run of this CTA's rows (b == 0: a single barrier group)
            int vr = prm.N - row_base;
            vr = vr < 0 ? 0 : (vr > prm.box_rows ? prm.box_rows : vr);
            const uint32_t bytes = (uint32_t)(vr * sizeof(T));
            int64_t nsys = prm.M - t * S;
            nsys = nsys > S ? S : nsys;
            mbar_expect_tx(&bars[1 + b], bytes * (uint32_t)nsys);
            if (bytes)
                for (int is = 0; is < (int)nsys; ++is)
                    bulk_load_1d(reinterpret_cast<unsigned char*>(landing) + (size_t)is * run_pitch,
                                 prm.f + (t * S + is) * (int64_t)prm.N + row_base, bytes, &bars[1 + b]);
        } else if constexpr (LM == 3) {
            mbar_expect_tx(&bars[1 + b], box_bytes);
            // system-major batch: tensor {N, M}, boxes of 128 bytes (W rows) x S systems, laid out [sub-box][S][128 B]
            constexpr int W = 128 / (int)sizeof(T);
            for (int sb = 0; sb < prm.box_rows / W; ++sb)
                tma_load_2d(landing + ((size_t)b * prm.box_rows + (size_t)sb * W) * S, &tm,
                            row_base + b * prm.box_rows + sb * W, (int)(t * S), &bars[1 + b]);
        } else {
            mbar_expect_tx(&bars[1 + b], box_bytes);
            tma_load_2d(landing + (size_t)b * prm.box_rows * S, &tm, (int)(t * S), row_base + b * prm.box_rows, &bars[1 + b]);
        }
    };
    if (tid == 0) {
        for (int b = 0; b <= MAX_BOXES; ++b) mbar_init(&bars[b], 1);
        for (int b = 0; b < MAX_BOXES; ++b)
            mbar_init(&bars[1 + MAX_BOXES + b], prm.wcount[b] > 0 ? prm.wcount[b] : 1);
        mbar_init(&bars[BAR_F], 1);
        mbar_init(&bars[BAR_B], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if constexpr (LM >= 5) {
        // rows >= N of the last rank and systems >= M of the last tile are never copied: give those slots finite
        // contents once (their coefficients are zero, their results are never stored; 0 * NaN would still poison a run)
        for (size_t w = tid; w < (LM == 6 ? 2 : 1) * tile_elems; w += blockDim.x) landing[w] = (T)0;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
#if PENT_PDL
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
    int64_t tile = first;
    if (tid == 0) {
        const uint32_t fold_bytes = PER ? (uint32_t)(4 * P * sizeof(T2)) : 0u, edge_bytes = PER ? (uint32_t)(3 * C * sizeof(T2)) : 0u;
        mbar_expect_tx(&bars[0], prm.table_bytes + fold_bytes + edge_bytes);
        bulk_load_1d(table, prm.table + (size_t)rank * prm.table_stride, prm.table_bytes, &bars[0]);
        if constexpr (PER) {
            bulk_load_1d(zfold, pp.fold + (size_t)rank * 8 * P, fold_bytes, &bars[0]);
            bulk_load_1d(zedge, pp.zedge, edge_bytes, &bars[0]);
        }
    }
#if PENT_PDL
    // the previous kernel on the stream may have written f or may still read x: wait for it before the
    // first access to the batch (the tables staged above are constant)
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
    if (tid == 0) {
        if (tile < prm.ntiles)
            for (int b = 0; b < prm.nbox; ++b) issue_box(b, tile);
    }
    // every CTA of the cluster is resident, with its mbarriers initialised, before any DSMEM store
    if constexpr (CLUSTER) cluster_sync_all();
    static_assert(!NBR || (CLUSTER && !PER), "neighbour-only exchange: cluster kernels, non-periodic");
    static_assert(!EPI || (!PER && BAND == 2 && LM != 3), "2x - f epilogue: pentadiagonal, non-periodic");
    const uint32_t agg_bytes_f = NBR ? (uint32_t)((rank > 0 ? 1 : 0) * S * sizeof(ST))   // from the rank before
                                     : (uint32_t)(rank * S * sizeof(ST));                 // from the earlier ranks
    // from the later ranks; periodic: from EVERY rank (itself included) plus (y_{n-2}, y_{n-1}) from rank ra
    const uint32_t agg_bytes_b = NBR ? (uint32_t)((rank < prm.Q - 1 ? 1 : 0) * S * sizeof(ST))
                               : PER ? (uint32_t)((prm.Q + 1) * S * sizeof(ST))
                                     : (uint32_t)((prm.Q - 1 - rank) * S * sizeof(ST));
    mbar_wait(&bars[0], 0);

    const T* blk = table + (size_t)(active ? p : 0) * BL;
    const T* wtab = table + (size_t)P * BL;          // W: TX | PF | PB | BLK | levels
    const int mybox = active ? (p * C) / prm.box_rows : 0;
    const int slot = state_slot<S>(active ? p : 0, i);
    const int row0 = row_base + p * C;
    const bool rows_full = active && (row0 + C <= prm.N);
    uint32_t parity = 0;

    // chunk-state scan geometry: a group of Pw lanes scans one system; G groups per warp
    const int Pw = prm.Pw, G = 32 / Pw;
    const int q = lane % Pw, grp = lane / Pw;
    const ScanGeom geom{P, Pw, prm.lev_f, prm.lev_b, prm.woff};
    const int rounds = (S + nwarps * G - 1) / (nwarps * G);     // host guarantees 1 when CLUSTER

    // cp.async loader (prm.ldg == 4): this thread's C rows of tile t -> its own slots of the landing buffer
    auto ring_issue = [&](int64_t t) {
        if (active) {
            const int64_t col = t * S + i;
            const int nrows = (t < prm.ntiles && col < prm.M) ? prm.N - row0 : 0;
            const T* src = prm.f + (int64_t)row0 * prm.M + col;
            T* dst = landing + (size_t)p * C * S + i;
#pragma unroll
            for (int j = 0; j < C; ++j)
                if (j < nrows) cp_async_elem(dst + j * S, src + (int64_t)j * prm.M);
        }
        cp_async_commit();
    };
    if constexpr (LM == 0 && !PER) {
        if (prm.ldg == 4) ring_issue(tile);
    }
    int tcount = 0;
    if constexpr (PER) {
        if (tid < S) {
            if (tile < prm.ntiles && tile * S + tid < prm.M) {
                T* dst = reinterpret_cast<T*>(ftail2 + tid);
                cp_async_elem(dst, pp.f + (int64_t)prm.N * prm.M + tile * S + tid);
                cp_async_elem(dst + 1, pp.f + (int64_t)(prm.N + 1) * prm.M + tile * S + tid);
            }
            cp_async_commit();
        }
    }
    for (; tile < prm.ntiles; tile += stride) {
        const int64_t next_tile = tile + stride;
        T v[C];
        // periodic: (f_n, f_{n+1}) of system tid travel global -> shared by cp.async, one tile ahead
        // (double-buffered), so no thread waits for them and they hold no registers
        T2* ftail = ftail2 + (tcount & 1) * S;
        if constexpr (PER) {
            if (tid < S) {
                if (next_tile < prm.ntiles && next_tile * S + tid < prm.M) {
                    T* dst = reinterpret_cast<T*>(ftail2 + ((tcount + 1) & 1) * S + tid);
                    cp_async_elem(dst, pp.f + (int64_t)prm.N * prm.M + next_tile * S + tid);
                    cp_async_elem(dst + 1, pp.f + (int64_t)(prm.N + 1) * prm.M + next_tile * S + tid);
                }
                cp_async_commit();
            }
        }
        if (active) {
            if constexpr (LM >= 5) {
                // ---- system-major batch, padded per-system runs: this thread's chunk is C consecutive elements ----
                mbar_wait(&bars[1 + mybox], parity);
                constexpr int V = 16 / (int)sizeof(T);
                const T* src = reinterpret_cast<const T*>(reinterpret_cast<const unsigned char*>(landing) + (size_t)i * run_pitch) + p * C;
#pragma unroll
                for (int c = 0; c < C / V; ++c) {
                    T w[V];
                    lds_vec<T, V>(w, src + c * V);
#pragma unroll
                    for (int u = 0; u < V; ++u) v[c * V + u] = w[u];
                }
            } else if constexpr (LM == 3) {
                // ---- system-major batch through the swizzled landing buffer: rows [16-byte chunk c of the 128-byte
                // piece `sb` of system i] sit at chunk c ^ (i & 7) of smem row (sb * S + i) ----
                mbar_wait(&bars[1 + mybox], parity);
                constexpr int W = 128 / (int)sizeof(T), V = 16 / (int)sizeof(T);
                const unsigned char* base = reinterpret_cast<const unsigned char*>(landing) +
                                            ((size_t)(p * C / W) * S + i) * 128;
#pragma unroll
                for (int sb = 0; sb < C / W; ++sb) {
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        T w[V];
                        lds_vec<T, V>(w, reinterpret_cast<const T*>(base + (size_t)sb * S * 128 + ((c ^ (i & 7)) << 4)));
#pragma unroll
                        for (int u = 0; u < V; ++u) v[sb * W + c * V + u] = w[u];
                    }
                }
            } else if constexpr (LM == 2) {
                // ---- system-major batch: this thread's chunk is contiguous in memory ----
                const int64_t col = tile * S + i;
                const T* src = prm.f + col * (int64_t)prm.N + row0;
                const int nrows = col < prm.M ? prm.N - row0 : 0;
                if (nrows >= C && ((reinterpret_cast<uintptr_t>(src) & 31) == 0)) {
                    constexpr int W = 32 / sizeof(T);                 // elements per 256-bit access
#pragma unroll
                    for (int m = 0; m < C / W; ++m) {
                        T w[W];
                        ldg256(w, src + m * W);
#pragma unroll
                        for (int u = 0; u < W; ++u) v[m * W + u] = w[u];
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < C; ++j) v[j] = (j < nrows) ? __ldcs(src + j) : (T)0;
                }
            } else if (!PER && prm.ldg == 4) {
                // ---- tile data: this thread's own cp.async copies -> registers; rows / systems beyond the batch were
                // not copied and read as zero (their slots hold stale values) ----
                cp_async_wait<0>();
                const int64_t col = tile * S + i;
                const int nrows = col < prm.M ? prm.N - row0 : 0;
                const T* src = landing + (size_t)p * C * S + i;
#pragma unroll
                for (int j = 0; j < C; ++j) v[j] = (j < nrows) ? src[j * S] : (T)0;
            } else if (prm.ldg) {
                // ---- tile data: global -> registers (C independent loads in flight per thread) ----
                const int64_t col = tile * S + i;
                const T* src = prm.f + (int64_t)row0 * prm.M + col;
                const int nrows = col < prm.M ? prm.N - row0 : 0;
#pragma unroll
                for (int j = 0; j < C; ++j) v[j] = (j < nrows) ? __ldcs(src + (int64_t)j * prm.M) : (T)0;
            } else {
                // ---- tile data: landing buffer -> registers ----
                mbar_wait(&bars[1 + mybox], parity);
                const T* src = landing + (size_t)p * C * S + i;
#pragma unroll
                for (int j = 0; j < C; ++j) v[j] = src[j * S];
            }
        }
        // The box is free once every warp that reads it has its values in registers: each such
        // warp arrives on the box's "empty" barrier and thread 0 re-arms it with the NEXT tile's
        // TMA load, which then runs under all of this tile's arithmetic and stores.
        if constexpr (LM == 0 && !PER) {
            if (prm.ldg == 4) ring_issue(next_tile);      // the slots are free: their values are in registers
        }
        __syncwarp();
        if (lane == 0 && warp * 32 < P * S && (LM >= 3 || (LM == 0 && !prm.ldg))) mbar_arrive(&bars[1 + MAX_BOXES + mybox]);
        if constexpr (CLUSTER) {
            if (tid == 0) {        // arm this tile's aggregate barriers (complete_tx may already have arrived)
                if (agg_bytes_f) mbar_expect_tx(&bars[BAR_F], agg_bytes_f);
                if (agg_bytes_b) mbar_expect_tx(&bars[BAR_B], agg_bytes_b);
            }
        }
        if (tid == 0 && next_tile < prm.ntiles) {
            for (int b = 0; b < prm.nbox; ++b) {
                mbar_wait(&bars[1 + MAX_BOXES + b], parity);
                issue_box(b, next_tile);
            }
        }
        if (active) {
            // ---- 1+2. local forward sweep and local back substitution from zero states ----
            ST e, s;
            if constexpr (BAND == 2) chunk_local_sweeps<T>(v, blk, e, s);
            else tri_local_sweeps<T>(v, blk, e, s);
            stE[slot] = e;
            stS[slot] = s;
            if constexpr (PER) {
                // x^ of rows n-2 and n-1 (compile-time register indices: predicated scan of the chunk)
                if (rank == pp.ra && (p == pp.pa || p == pp.pb)) {
                    T va = 0, vb = 0;
#pragma unroll
                    for (int j = 0; j < C; ++j) {
                        if (j == pp.ja) va = v[j];
                        if (j == pp.jb) vb = v[j];
                    }
                    if (p == pp.pa) reinterpret_cast<T*>(ypub)[2 * i] = va;
                    if (p == pp.pb) reinterpret_cast<T*>(ypub)[2 * i + 1] = vb;
                }
            }
        }
        if constexpr (PER) {
            if (tid < S) cp_async_wait<1>();      // this tile's pair has landed (the next tile's may be in flight)
        }
        __syncthreads();       // states published

        // ---- 3. chunk-state scans (slot (q, sys) receives F_{q-1} and B_{q+1}) ----
        if (CLUSTER || PER || P > 1) {
            PeriodicCtx<T> per;
            if constexpr (PER) {
                per.pp = &pp; per.ypub = reinterpret_cast<T*>(ypub); per.yab = yab; per.ftail = ftail; per.stT = stT;
                per.table = table; per.x = prm.x; per.M = prm.M; per.n = prm.N; per.col0 = tile * S;
            }
            for (int r = 0; r < rounds; ++r) {
                const int sys = (r * nwarps + warp) * G + grp;
                if constexpr (BAND == 2)
                    chunk_state_scan<T, S, CLUSTER, PER, NBR>(geom, wtab, stE, stS, sys, q, (sys < S) && (q < P), rank,
                                                         prm.Q, aggF, aggB, bars, agg_bytes_f, agg_bytes_b, parity, &per);
                else
                    tri_state_scan<T, S, CLUSTER, NBR>(geom, wtab, stE, stS, sys, q, (sys < S) && (q < P), rank, prm.Q,
                                                  aggF, aggB, bars, agg_bytes_f, agg_bytes_b, parity);
            }
        }
        if constexpr (LM == 6) {      // the staging buffer may be overwritten once the previous tile's copies have read it
            if (tid < S) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        }
        __syncthreads();

        // Pacing of the store burst (profiles/r02_pacing.md): the x stores of this tile and the TMA loads of the next
        // one (in flight since the top of the loop) compete when they overlap in time; holding the stores back for a
        // fixed time raised the tridiagonal kernel from 0.79 to 0.89 of the HBM peak.  (A run-time value from the
        // constant bank: the fp64 cluster instantiation has no register to spare.)
        if (prm.pace_ns) __nanosleep(prm.pace_ns);
        // ---- 4. correction and store ----
        if (active) {
            T F0 = 0, F1 = 0, B0 = 0, B1 = 0;
            if (CLUSTER || PER || P > 1) {
                if constexpr (BAND == 2) { T2 fo = stE[slot]; F0 = fo.x; F1 = fo.y; T2 bo = stS[slot]; B0 = bo.x; B1 = bo.y; }
                else { F0 = stE[slot]; B0 = stS[slot]; }
            }
            // rows 4 jg .. 4 jg + 3 of this thread's chunk: x = x^ + responses to the incoming chunk states
            auto correct4 = [&](T (&out)[4], int jg) {
                if constexpr (BAND == 2) chunk_correct4<T>(out, &v[4 * jg], blk, jg, F0, F1, B0, B1);
                else tri_correct4<T>(out, &v[4 * jg], blk, jg, F0, B0);
                if constexpr (EPI) {
                    const int64_t ecol = tile * S + i;
                    const int k0 = row0 + 4 * jg;
                    if (ecol < prm.M) {
                        if constexpr (LM >= 5) {          // system-major, 16-byte aligned runs: vector loads of the 4 rows
                            if (k0 + 4 <= prm.N) {
                                T fv[4];
                                const uint4* src = reinterpret_cast<const uint4*>(prm.f + ecol * (int64_t)prm.N + k0);
                                if constexpr (sizeof(T) == 8) {
                                    const uint4 q0 = src[0], q1 = src[1];
                                    fv[0] = __hiloint2double((int)q0.y, (int)q0.x); fv[1] = __hiloint2double((int)q0.w, (int)q0.z);
                                    fv[2] = __hiloint2double((int)q1.y, (int)q1.x); fv[3] = __hiloint2double((int)q1.w, (int)q1.z);
                                } else {
                                    const uint4 q0 = src[0];
                                    fv[0] = __uint_as_float(q0.x); fv[1] = __uint_as_float(q0.y);
                                    fv[2] = __uint_as_float(q0.z); fv[3] = __uint_as_float(q0.w);
                                }
#pragma unroll
                                for (int r = 0; r < 4; ++r) out[r] = fma((T)2, out[r], -fv[r]);
                            } else {
#pragma unroll
                                for (int r = 0; r < 4; ++r)
                                    if (k0 + r < prm.N) out[r] = fma((T)2, out[r], -prm.f[ecol * (int64_t)prm.N + k0 + r]);
                            }
                        } else {
#pragma unroll
                            for (int r = 0; r < 4; ++r)
                                if (k0 + r < prm.N)
                                    out[r] = fma((T)2, out[r], -(LM == 0 ? prm.f[(int64_t)(k0 + r) * prm.M + ecol]
                                                                          : prm.f[ecol * (int64_t)prm.N + k0 + r]));
                        }
                    }
                }
            };
            const int64_t col = tile * S + i;
            T* xo = prm.x + (int64_t)row0 * prm.M + col;
            if constexpr (LM == 6) {
                // system-major batch, stores through bulk copies: x -> padded staging buffer (the previous tile's copies
                // have read it: the issuing threads waited before the barrier that precedes this stage)
                constexpr int V = 16 / (int)sizeof(T);
                T* dst = reinterpret_cast<T*>(reinterpret_cast<unsigned char*>(staging) + (size_t)i * run_pitch) + p * C;
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T xv[4];
                    correct4(xv, jg);
#pragma unroll
                    for (int u = 0; u < 4 / V; ++u) {
                        uint4 q;
                        if constexpr (sizeof(T) == 8) {
                            q.x = (uint32_t)__double2loint(xv[2 * u]); q.y = (uint32_t)__double2hiint(xv[2 * u]);
                            q.z = (uint32_t)__double2loint(xv[2 * u + 1]); q.w = (uint32_t)__double2hiint(xv[2 * u + 1]);
                        } else {
                            q.x = __float_as_uint(xv[0]); q.y = __float_as_uint(xv[1]);
                            q.z = __float_as_uint(xv[2]); q.w = __float_as_uint(xv[3]);
                        }
                        *reinterpret_cast<uint4*>(dst + 4 * jg + u * V) = q;
                    }
                }
            }
            if constexpr (LM == 2 || LM == 3 || LM == 5) {
                // system-major batch: contiguous run of this thread's chunk, 32-byte stores where possible
                T* xr = prm.x + col * (int64_t)prm.N + row0;
                const int nrows = col < prm.M ? prm.N - row0 : 0;
                const bool vec = nrows >= C && ((reinterpret_cast<uintptr_t>(xr) & 31) == 0);
                constexpr int W = 32 / sizeof(T);
                T acc[W];
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T xv[4];
                    correct4(xv, jg);
                    if (vec) {
#pragma unroll
                        for (int r = 0; r < 4; ++r) acc[(4 * jg + r) % W] = xv[r];
                        if ((4 * jg + 4) % W == 0) stg256(xr + (4 * jg + 4 - W), acc);
                    } else {
#pragma unroll
                        for (int r = 0; r < 4; ++r)
                            if (4 * jg + r < nrows) xr[4 * jg + r] = xv[r];
                    }
                }
            }
            // periodic: x^ = y - Z t.  Z is folded into the chunk states (F - F^Z t, B - B^Z t); the chunks that hold the
            // non-zero rows of k (chunk 0, the chunks of rows n-2 and n-1) subtract their explicit rows of Z from x^ here,
            // inside the store loops (edge4 below)
            if constexpr (PER) {
                const T2 t = stT[i];
                const T2* fz = zfold + 4 * (size_t)p;
                const T2 a = fz[0], b = fz[1], c = fz[2], d = fz[3];
                F0 = fma(-a.y, t.y, fma(-a.x, t.x, F0)); F1 = fma(-b.y, t.y, fma(-b.x, t.x, F1));
                B0 = fma(-c.y, t.y, fma(-c.x, t.x, B0)); B1 = fma(-d.y, t.y, fma(-d.x, t.x, B1));
            }
            // The chunks that hold the non-zero rows of k take a store loop of their own (the round-1 loop: explicit rows
            // of Z, t in registers); every other chunk runs the loop of the non-periodic kernel.  Two loops rather than
            // a test inside one: the fp64 cluster instantiation is at its 128-register limit, and the test cost 164
            // bytes of spills and 20 % of the kernel's time.
            bool edge_done = false;
            if constexpr (PER) {
                const bool e0 = rank == 0 && p == 0, ea = rank == pp.ra && p == pp.pa, eb = rank == pp.ra && p == pp.pb;
                if (e0 || ea || eb) {
                    edge_done = true;
                    const T2 t = stT[i];
                    const T2* zr = zedge + (e0 ? 0 : ea ? C : 2 * C);
                    const int nrows = (col < prm.M) ? prm.N - row0 : 0;
#pragma unroll
                    for (int jg = 0; jg < C / 4; ++jg) {
                        T xv[4];
                        correct4(xv, jg);
#pragma unroll
                        for (int r = 0; r < 4; ++r) {
                            const T2 z = zr[4 * jg + r];
                            xv[r] = fma(-z.y, t.y, fma(-z.x, t.x, xv[r]));
                            if (4 * jg + r < nrows) PENT_STORE(xo, xv[r]);
                            xo += prm.M;
                        }
                    }
                }
            }
            if constexpr (LM >= 2) {
                // stored above
            } else if (edge_done) {
                // stored above
            } else if (rows_full && (tile + 1) * S <= prm.M) {
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T xv[4];
                    correct4(xv, jg);
#pragma unroll
                    for (int r = 0; r < 4; ++r) { PENT_STORE(xo, xv[r]); xo += prm.M; }
                }
            } else if (col < prm.M) {
                const int nrows = prm.N - row0;      // may be <= 0
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T xv[4];
                    correct4(xv, jg);
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        if (4 * jg + r < nrows) PENT_STORE(xo, xv[r]);
                        xo += prm.M;
                    }
                }
            }
        }
        if constexpr (LM == 6) {
            // every thread's x is in the staging buffer: generic-proxy writes -> async proxy, block barrier, then thread
            // `is` < S issues the ONE bulk copy of system `is` (rows >= N and systems >= M are not stored)
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads();
            if (tid < S && tile * S + tid < prm.M) {
                int vr = prm.N - row_base;
                vr = vr < 0 ? 0 : (vr > prm.box_rows ? prm.box_rows : vr);
                if (vr > 0) {
                    const unsigned char* src = reinterpret_cast<const unsigned char*>(staging) + (size_t)tid * run_pitch;
                    T* dst = prm.x + (tile * S + tid) * (int64_t)prm.N + row_base;
                    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                                 ::"l"((uint64_t)dst), "r"(smem_u32(src)), "r"((uint32_t)(vr * sizeof(T))) : "memory");
                }
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        }
        parity ^= 1;
        ++tcount;
    }
    if constexpr (LM == 6) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    if constexpr (CLUSTER) cluster_sync_all();   // no CTA leaves while a peer may still address its shared memory
}
