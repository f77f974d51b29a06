// pent_solve_chunked.cu -- placeholder until the chunked on-chip kernel lands.
#include "pent_internal.h"
namespace pent {
int build_chunk_tables(pent_handle*, cudaStream_t) { return PENT_OK; }
bool chunked_supported(const pent_handle*, int64_t) { return false; }
int launch_solve_chunked(const pent_handle*, int64_t, const void*, void*, cudaStream_t) { return PENT_ERR_ARG; }
}
