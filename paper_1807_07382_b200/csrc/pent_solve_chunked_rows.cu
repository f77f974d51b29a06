// pent_solve_chunked_rows.cu -- the system-major ("one system per row") instantiations of the chunked
// solve kernel: LM = 2 (per-thread LDG.256 / STG.256), 3 (swizzled tensor-tile TMA loads, STG.256 stores; kept as
// the A/B baseline of the row-rate finding), 5 (1-D bulk loads, STG.256 stores), 6 (1-D bulk loads and stores).  A separate translation unit so that the instantiations compile in parallel with the
// interleaved ones of pent_solve_chunked.cu.  The plans are made there (rows_plan); see DESIGN.md section 6.7.
#include "pent_chunked_launch.cuh"

namespace pent {

template <typename T, int S, int BAND>
static int launch_rows_mode(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s)
{
    const bool cl = pl.Q > 1;
#define PENT_ROWS_INST(LM_) (cl ? launch_inst<T, S, true, false, BAND, LM_>(h, pl, M, f, x, s, nullptr) \
                                : launch_inst<T, S, false, false, BAND, LM_>(h, pl, M, f, x, s, nullptr))
    switch (pl.mode) {
        case 2: return PENT_ROWS_INST(2);
        case 3: return PENT_ROWS_INST(3);
        case 5: return PENT_ROWS_INST(5);
        case 6: return PENT_ROWS_INST(6);
        default: return PENT_ERR_ARG;
    }
#undef PENT_ROWS_INST
}

int launch_plan_rows(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s)
{
    if (h->dtype == PENT_F64) {
        if (pl.S == 16) return pl.band == 1 ? launch_rows_mode<double, 16, 1>(h, pl, M, f, x, s) : launch_rows_mode<double, 16, 2>(h, pl, M, f, x, s);
        if (pl.S == 32) return pl.band == 1 ? launch_rows_mode<double, 32, 1>(h, pl, M, f, x, s) : launch_rows_mode<double, 32, 2>(h, pl, M, f, x, s);
    } else {
        if (pl.S == 32) return pl.band == 1 ? launch_rows_mode<float, 32, 1>(h, pl, M, f, x, s) : launch_rows_mode<float, 32, 2>(h, pl, M, f, x, s);
        if (pl.S == 64) return pl.band == 1 ? launch_rows_mode<float, 64, 1>(h, pl, M, f, x, s) : launch_rows_mode<float, 64, 2>(h, pl, M, f, x, s);
    }
    return PENT_ERR_ARG;
}
}  // namespace pent
