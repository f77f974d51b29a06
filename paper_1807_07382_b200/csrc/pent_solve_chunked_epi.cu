// pent_solve_chunked_epi.cu -- the instantiations of the chunked solve kernel with the "2 x - f" epilogue (EPI, see
// pent_chunked_kernel.cuh): x = 2 A^{-1} f - f = (2I - A) A^{-1} f, what a Peaceman-Rachford ADI sweep needs between its two
// implicit half steps (pent_adi.cu).  Interleaved batches (LM = 0, every loader of that instantiation) and system-major ones
// (LM = 2, 5, 6); pentadiagonal tables, all-ranks cluster exchange.  A translation unit of its own so that these compile in
// parallel with the others.
#include "pent_chunked_launch.cuh"

namespace pent {

template <typename T, int S>
static int launch_epi_mode(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s)
{
    const bool cl = pl.Q > 1;
#define PENT_EPI_INST(LM_) (cl ? launch_inst<T, S, true, false, 2, LM_, false, true>(h, pl, M, f, x, s, nullptr) \
                               : launch_inst<T, S, false, false, 2, LM_, false, true>(h, pl, M, f, x, s, nullptr))
    if (!pl.rows) return PENT_EPI_INST(0);
    switch (pl.mode) {
        case 2: return PENT_EPI_INST(2);
        case 5: return PENT_EPI_INST(5);
        case 6: return PENT_EPI_INST(6);
        default: return PENT_ERR_ARG;
    }
#undef PENT_EPI_INST
}

int launch_plan_epi(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s)
{
    if (pl.band != 2 || pl.nbr) return PENT_ERR_ARG;
    if (h->dtype == PENT_F64) {
        if (pl.S == 16) return launch_epi_mode<double, 16>(h, pl, M, f, x, s);
        if (pl.S == 32) return launch_epi_mode<double, 32>(h, pl, M, f, x, s);
    } else {
        if (pl.S == 32) return launch_epi_mode<float, 32>(h, pl, M, f, x, s);
        if (pl.S == 64) return launch_epi_mode<float, 64>(h, pl, M, f, x, s);
    }
    return PENT_ERR_ARG;
}
}  // namespace pent
