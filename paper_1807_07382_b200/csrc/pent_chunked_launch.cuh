// pent_chunked_launch.cuh -- host launcher of solve_chunked_kernel, shared by pent_solve_chunked.cu
// (PER = false) and pent_solve_chunked_periodic.cu (PER = true) so that the two sets of template
// instantiations compile in parallel.
#pragma once
#include <cstdio>
#include <cstdlib>
#include "pent_chunk_common.cuh"

#ifndef PENT_PDL
#define PENT_PDL 1      // programmatic dependent launch (A/B: -DPENT_PDL=0), see the kernel prologue
#endif

namespace pent {
#include "pent_chunked_kernel.cuh"

// extra dynamic shared memory of the periodic kernel: the Z-solve chunk states of this CTA's chunks (4 pairs each), the
// explicit rows of Z of the three edge chunks, five [S] pair arrays and the second aggregate array of a cluster
template <typename T>
inline size_t periodic_extra_smem(const ChunkPlan& pl)
{
    return ((size_t)4 * pl.Pl + 3 * (size_t)ChunkCfg<T>::C + 5 * (size_t)pl.S + (pl.Q > 1 ? (size_t)pl.Q * pl.S : 0)) * 2 * sizeof(T);
}

template <typename T, int S, bool CLUSTER, bool PER, int BAND = 2, int LM = 0, bool NBR = false, bool EPI = false>
static int launch_inst(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x,
                       cudaStream_t s, const PeriodicParams<T>* per)
{
    constexpr int C = ChunkCfg<T>::C;
    ChunkParams<T> prm;
    prm.N = h->N; prm.P = pl.Pl; prm.Q = pl.Q; prm.Pw = pl.Pw; prm.M = M;
    int lg = 0;
    while ((1 << lg) < pl.Pw) ++lg;
    const int hlf = BAND == 2 ? h->lev_f[pl.j] : h->lev_f1[pl.j], hlb = BAND == 2 ? h->lev_b[pl.j] : h->lev_b1[pl.j];
    prm.lev_f = hlf < lg ? hlf : lg;
    prm.lev_b = hlb < lg ? hlb : lg;
    for (int l = 0; l < W_LEVELS; ++l) prm.woff[l] = w_level_off(pl.Pl, l, pl.Q, BAND);
    prm.box_rows = pl.box_rows; prm.nbox = pl.nbox;
    prm.land_rows = pl.mode == 4 ? pl.Pl * C : pl.nbox * pl.box_rows;
    prm.ntiles = (M + S - 1) / S;
    for (int b = 0; b < MAX_BOXES; ++b) prm.wcount[b] = 0;
    for (int w = 0; w * 32 < pl.Pl * S; ++w) prm.wcount[((w * 32 / S) * C) / prm.box_rows] += 1;
    prm.table = (const T*)(BAND == 2 ? h->cf[pl.j] : h->cf1[pl.j]);
    prm.table_stride = (int64_t)table_len<T, BAND>(pl.Pl, pl.Q);
    prm.table_bytes = (uint32_t)pl.table_bytes;
    prm.x = (T*)x;
    prm.f = (const T*)f;
    prm.ldg = pl.mode;
    prm.pace_ns = (unsigned)pl.pace_ns;
    if (const char* e = std::getenv("PENT_AB_PACE")) prm.pace_ns = (unsigned)std::atoi(e);      // measurement override (ns)

    CUtensorMap tm = {};
    const bool enc_ok = pl.mode == 0 ? encode_batch_map_cached(&tm, f, M, h->N, S, prm.box_rows, sizeof(T) == 8)
                      : pl.mode == 3 ? encode_rows_map_cached(&tm, f, M, h->N, S, sizeof(T) == 8) : true;
    CUtensorMap tmx = {};            // (second map: unused since the stores of the system-major modes are bulk copies)
    const bool encx_ok = true;
    if (!enc_ok || !encx_ok) {
        g_last_cuda_error = (int)cudaErrorInvalidValue;
        return PENT_ERR_CUDA;
    }

    PeriodicParams<T> pp = {};
    if (PER) pp = *per;
    const size_t smem_total = pl.smem + (PER ? periodic_extra_smem<T>(pl) : 0);
    if ((LM == 0) != (pl.mode <= 1 || pl.mode == 4) || (LM != 0 && LM != pl.mode) || (PER && pl.mode == 4)) return PENT_ERR_ARG;
    auto kern = solve_chunked_kernel<T, S, CLUSTER, PER, BAND, LM, NBR, EPI>;
    static SmemOnce mark;
    PENT_CUDA(ensure_dynamic_smem(mark, kern, smem_total));
    // the occupancy answer depends only on (device, threads, shared memory, cluster size): keep the last
    // one per thread and kernel instance, so a small solve is not bound by host-side queries
    struct OccCache { int dev = -1, threads = 0, Q = 0, nsm = 0, resident = 0; size_t smem = 0; };
    static thread_local OccCache oc;
    int dev = 0;
    PENT_CUDA(cudaGetDevice(&dev));
    const bool hit = oc.dev == dev && oc.threads == pl.threads && oc.smem == smem_total && oc.Q == pl.Q;
    if (!hit) PENT_CUDA(cudaDeviceGetAttribute(&oc.nsm, cudaDevAttrMultiProcessorCount, dev));
    if constexpr (!CLUSTER) {
        if (!hit) {
            int occ = 0;
            PENT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, pl.threads, smem_total));
            oc.resident = oc.nsm * occ;                          // CTAs resident at once
            oc.dev = dev; oc.threads = pl.threads; oc.smem = smem_total; oc.Q = pl.Q;
        }
        if (oc.resident < 1) return PENT_ERR_ARG;
        int64_t grid = oc.resident;
        if (grid > prm.ntiles) grid = prm.ntiles;
#if PENT_PDL
        // programmatic dependent launch: this grid's prologue (mbarrier init, staging of the constant
        // coefficient table) may overlap the tail of the previous kernel on the stream; the kernel
        // waits (griddepcontrol.wait) before it touches f or x
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)pl.threads);
        cfg.dynamicSmemBytes = smem_total; cfg.stream = s; cfg.attrs = at; cfg.numAttrs = 1;
        PENT_CUDA(cudaLaunchKernelEx(&cfg, kern, tm, prm, pp, tmx));
#else
        kern<<<(unsigned)grid, pl.threads, smem_total, s>>>(tm, prm, pp, tmx);
#endif
    } else {
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute at[2];
        at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[1].val.programmaticStreamSerializationAllowed = 1;
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)pl.Q; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.blockDim = dim3((unsigned)pl.threads); cfg.dynamicSmemBytes = smem_total; cfg.stream = s;
        cfg.attrs = at; cfg.numAttrs = 1 + PENT_PDL;
        if (pl.Q > 8) {           // 16 CTAs per cluster: a non-portable size, allowed once per kernel instance and device
            static SmemOnce npmark;
            int d2 = 0;
            PENT_CUDA(cudaGetDevice(&d2));
            const uint32_t bit = 1u << (d2 & 31);
            if (!(npmark.mask.load(std::memory_order_acquire) & bit)) {
                PENT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
                npmark.mask.fetch_or(bit, std::memory_order_release);
            }
        }
        if (!hit) {
            cfg.gridDim = dim3((unsigned)(pl.Q * oc.nsm));       // upper bound for the occupancy query
            int ncl = 0;
            PENT_CUDA(cudaOccupancyMaxActiveClusters(&ncl, kern, &cfg));
            oc.resident = ncl;                                   // clusters resident at once
            oc.dev = dev; oc.threads = pl.threads; oc.smem = smem_total; oc.Q = pl.Q;
        }
        // no cluster of this size is schedulable here (a partitioned GPU, a 16-CTA cluster on a device whose GPCs are
        // smaller): not an error of the caller; PENT_KERNEL_AUTO then runs the thread-per-system kernel
        if (oc.resident < 1) return PENT_UNSUPPORTED;
        int64_t clusters = oc.resident;
        if (clusters > prm.ntiles) clusters = prm.ntiles;
        cfg.gridDim = dim3((unsigned)(clusters * pl.Q));
        PENT_CUDA(cudaLaunchKernelEx(&cfg, kern, tm, prm, pp, tmx));
    }
    count_launch();
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}

}  // namespace pent
