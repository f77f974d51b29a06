// pent_solve_chunked_periodic.cu -- the periodic (cyclic) solve FUSED into the chunked kernel
// (Eqs. 8-12; PER = true instantiations of solve_chunked_kernel, see PeriodicCtx in
// pent_chunk_common.cuh): y = E^{-1} f^, the 2 x 2 tail solve and x^ = y - Z t in ONE kernel,
// 2 passes over the batch.  The unfused 3-kernel path of pent_periodic.cu stays as the fallback
// (rows n-2 / n-1 in different cluster ranks, or no on-chip plan for E).  Z itself is not on chip: it is folded into
// the chunk states (periodic_fold_kernel in pent_periodic.cu).
#include "pent_chunked_launch.cuh"

namespace pent {

struct PeriodicPlan {
    bool ok = false;
    ChunkPlan pl;
    int ra = 0, pa = 0, ja = 0, pb = 0, jb = 0;
};

static PeriodicPlan periodic_plan(const pent_handle* h, int64_t M, const void* f)
{
    PeriodicPlan pp;
    if (!h || !h->periodic || !h->inner) return pp;
    const pent_handle* in = h->inner;
    pp.pl = chunk_auto_plan(in, M, f, /*ring_ok=*/false);   // (not ok when the stitching of E is flagged unstable)
    plan_drop_nbr(pp.pl, h->dtype == PENT_F64 ? 8 : 4);       // the periodic kernel exchanges with every rank
    if (!pp.pl.ok || !h->pfold || !h->pzedge) return pp;
    const bool f64 = h->dtype == PENT_F64;
    const int C = f64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
    const int n = in->N;
    const int ga = (n - 2) / C, gb = (n - 1) / C;          // global chunks of rows n-2, n-1
    pp.ra = ga / pp.pl.Pl;
    if (gb / pp.pl.Pl != pp.ra) return pp;                 // both rows must sit in one cluster rank
    pp.pa = ga % pp.pl.Pl; pp.ja = (n - 2) % C;
    pp.pb = gb % pp.pl.Pl; pp.jb = (n - 1) % C;
    const size_t extra = f64 ? periodic_extra_smem<double>(pp.pl) : periodic_extra_smem<float>(pp.pl);
    if (pp.pl.smem + extra > SMEM_LIMIT) return pp;
    pp.ok = true;
    return pp;
}

bool periodic_fused_supported(const pent_handle* h, int64_t M, const void* f)
{
    return periodic_plan(h, M, f).ok;
}

template <typename T>
static int launch_periodic_t(const pent_handle* h, const PeriodicPlan& pl, int64_t M, const void* f, void* x,
                             cudaStream_t s)
{
    PeriodicParams<T> pp;
    pp.ra = pl.ra; pp.pa = pl.pa; pp.ja = pl.ja; pp.pb = pl.pb; pp.jb = pl.jb;
    pp.h00 = (T)h->pc[0]; pp.h0a = (T)h->pc[1]; pp.h0b = (T)h->pc[2];
    pp.h10 = (T)h->pc[3]; pp.h11 = (T)h->pc[4]; pp.h1a = (T)h->pc[5];
    pp.i00 = (T)h->pc[6]; pp.i01 = (T)h->pc[7]; pp.i10 = (T)h->pc[8]; pp.i11 = (T)h->pc[9];
    pp.fold = (const T*)h->pfold;
    pp.zedge = (const typename Pair<T>::type*)h->pzedge;
    pp.f = (const T*)f;
    const pent_handle* in = h->inner;
    const bool cl = pl.pl.Q > 1;
    constexpr int Sn = sizeof(T) == 8 ? 16 : 32, Sw = 2 * Sn;
    if (pl.pl.S == Sn)
        return cl ? launch_inst<T, Sn, true, true>(in, pl.pl, M, f, x, s, &pp)
                  : launch_inst<T, Sn, false, true>(in, pl.pl, M, f, x, s, &pp);
    if (pl.pl.S == Sw)
        return cl ? launch_inst<T, Sw, true, true>(in, pl.pl, M, f, x, s, &pp)
                  : launch_inst<T, Sw, false, true>(in, pl.pl, M, f, x, s, &pp);
    return PENT_ERR_ARG;
}

int launch_solve_chunked_periodic(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s)
{
    const PeriodicPlan pl = periodic_plan(h, M, f);
    if (!pl.ok) return PENT_ERR_ARG;
    if (h->dtype == PENT_F64) return launch_periodic_t<double>(h, pl, M, f, x, s);
    return launch_periodic_t<float>(h, pl, M, f, x, s);
}
}  // namespace pent
