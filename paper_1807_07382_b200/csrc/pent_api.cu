// pent_api.cu -- shared-A solve entry points: kernel dispatch and the host-buffer variant.
#include <algorithm>
#include "pent_internal.h"

extern "C" int pent_solve_batch_v(const pent_handle* h, int64_t M, const void* f, void* x,
                                  void* stream, int kernel)
{
    if (!h || h->kind != 0 || M < 0) return PENT_ERR_ARG;
    if (M == 0) return PENT_OK;
    if (!f || !x || !pent::on_handle_device(h)) return PENT_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (kernel < 0 || (kernel >> 24) != 0) return PENT_ERR_ARG;
    if (h->periodic) return pent::solve_periodic(h, M, f, x, s, kernel);
    const int Q = (kernel >> 8) & 0xff, S = (kernel >> 16) & 0xff;
    switch (kernel & 0xff) {
        case PENT_KERNEL_AUTO: {
            if (Q || S) return PENT_ERR_ARG;
            // the plan is resolved once, inside the launcher; PENT_UNSUPPORTED = no on-chip plan for this shape
            const int rc = pent::launch_solve_chunked(h, M, f, x, s, 0, 0);
            return rc == pent::PENT_UNSUPPORTED ? pent::launch_solve_tps(h, M, f, x, s) : rc;
        }
        case PENT_KERNEL_THREAD_PER_SYSTEM:
            if (Q || S) return PENT_ERR_ARG;
            return pent::launch_solve_tps(h, M, f, x, s);
        case PENT_KERNEL_CHUNKED: {
            const int rc = pent::launch_solve_chunked(h, M, f, x, s, Q, S);
            return rc == pent::PENT_UNSUPPORTED ? PENT_ERR_ARG : rc;
        }
        default:
            return PENT_ERR_ARG;
    }
}

// System-major batches ("one system per row", the layout of the paper's serial code; also
// the access an ADI sweep along the contiguous axis of a 2-D field needs).
extern "C" int pent_solve_batch_rows_v(const pent_handle* h, int64_t M, const void* f, void* x, void* stream,
                                       int kernel)
{
    if (!h || h->kind != 0 || h->periodic || M < 0) return PENT_ERR_ARG;
    if (M == 0) return PENT_OK;
    if (!f || !x || !pent::on_handle_device(h)) return PENT_ERR_ARG;
    const int loader = (kernel & PENT_ROWS_LDG) ? 1 : (kernel & PENT_ROWS_STG) ? 2 : (kernel & PENT_ROWS_TMA2D) ? 3 : 0;
    kernel &= ~(PENT_ROWS_LDG | PENT_ROWS_STG | PENT_ROWS_TMA2D);
    if (kernel < 0 || (kernel >> 24) != 0) return PENT_ERR_ARG;
    if ((kernel & 0xff) != PENT_KERNEL_AUTO && (kernel & 0xff) != PENT_KERNEL_CHUNKED) return PENT_ERR_ARG;
    const int Q = (kernel >> 8) & 0xff, S = (kernel >> 16) & 0xff;
    if ((Q != 0) != (S != 0)) return PENT_ERR_ARG;
    const int rc = pent::launch_solve_chunked_rows(h, M, f, x, (cudaStream_t)stream, Q, S, loader);
    return rc == pent::PENT_UNSUPPORTED ? PENT_ERR_ARG : rc;           // N too long to keep a tile on chip
}

extern "C" int pent_solve_batch_rows(const pent_handle* h, int64_t M, const void* f, void* x, void* stream)
{
    return pent_solve_batch_rows_v(h, M, f, x, stream, PENT_KERNEL_AUTO);
}

extern "C" int pent_solve_kernel_choice(const pent_handle* h, int64_t M)
{
    if (!h || h->kind != 0) return -1;
    if (h->periodic) return pent_solve_kernel_choice(h->inner, M);
    int Q = 0, S = 0;
    if (!pent::chunked_choice(h, M, &Q, &S)) return PENT_KERNEL_THREAD_PER_SYSTEM;
    return PENT_KERNEL_CHUNKED_CFG(Q, S);
}

extern "C" int pent_solve_rows_kernel_choice(const pent_handle* h, int64_t M)
{
    if (!h || h->kind != 0 || h->periodic) return -1;
    int Q = 0, S = 0, mode = 0;
    if (!pent::chunked_rows_choice(h, M, &Q, &S, &mode)) return -1;
    return PENT_KERNEL_CHUNKED_CFG(Q, S) | (mode << 24);
}

extern "C" int pent_solve_batch(const pent_handle* h, int64_t M, const void* f, void* x,
                                void* stream)
{
    return pent_solve_batch_v(h, M, f, x, stream, PENT_KERNEL_AUTO);
}

// Host buffers: the batch is cut into slabs of consecutive systems.  A slab of an interleaved
// (N x M) array is a strided 2-D region (N rows of Ms elements, pitch M), moved with
// cudaMemcpy2DAsync into a dense (N x Ms) device array, solved there and moved back.  NB slabs
// rotate over NB streams so the upload of slab j+1, the solve of slab j and the download of slab
// j-1 overlap (PCIe is full duplex).  The staging buffers and streams are a per-thread cache (a call
// used to spend ~1 ms of its 14 ms in cudaMalloc / cudaFree); they hold no state between calls.
namespace {
constexpr int NB = 4;
struct HostPipe {
    int dev = -1;
    size_t cap = 0;                      // bytes per buffer
    void* buf[NB] = {};
    cudaStream_t st[NB] = {};
    void release()
    {
        for (int j = 0; j < NB; ++j) {
            if (buf[j]) cudaFree(buf[j]);
            if (st[j]) cudaStreamDestroy(st[j]);
            buf[j] = nullptr; st[j] = nullptr;
        }
        cap = 0; dev = -1;
        cudaGetLastError();              // at thread exit the context may already be gone
    }
    ~HostPipe() { release(); }
    int ensure(size_t bytes)
    {
        int d = 0;
        cudaError_t e = cudaGetDevice(&d);
        if (e != cudaSuccess) return pent::cuda_fail(e);
        if (d == dev && bytes <= cap) return PENT_OK;
        release();
        for (int j = 0; j < NB; ++j) {
            e = cudaMalloc(&buf[j], bytes);
            if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); release(); return PENT_ERR_ALLOC; }
            if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&st[j], cudaStreamNonBlocking);
            if (e != cudaSuccess) { release(); return pent::cuda_fail(e); }
        }
        dev = d; cap = bytes;
        return PENT_OK;
    }
};
thread_local HostPipe g_pipe;
}  // namespace

extern "C" void pent_release_thread_cache(void) { g_pipe.release(); }

extern "C" int pent_solve_batch_host(const pent_handle* h, int64_t M, const void* f_host,
                                     void* x_host)
{
    if (!h || h->kind != 0 || M < 0) return PENT_ERR_ARG;
    if (M == 0) return PENT_OK;
    if (!f_host || !x_host || !pent::on_handle_device(h)) return PENT_ERR_ARG;
    const size_t esz = h->dtype == PENT_F64 ? 8 : 4;
    const int N = h->N;
    // cudaMemcpy2DAsync takes the host pitch M*esz, which must stay below cudaDevAttrMaxPitch (2^31 - 1 bytes)
    if ((uint64_t)M * esz > 0x7fffffffull) return PENT_ERR_ARG;
    // ~16 MiB slabs, a multiple of 256 systems (keeps the slab pitch 16-byte aligned for TMA)
    int64_t Ms = std::max<int64_t>(256, ((16ll << 20) / ((int64_t)N * (int64_t)esz)) / 256 * 256);
    Ms = std::min(Ms, M);
    int rc = g_pipe.ensure((size_t)N * (size_t)Ms * esz);
    if (rc != PENT_OK) return rc;
    int64_t slab = 0;
    for (int64_t i0 = 0; i0 < M && rc == PENT_OK; i0 += Ms, ++slab) {
        const int j = (int)(slab % NB);
        const int64_t m = std::min(Ms, M - i0);
        const char* src = (const char*)f_host + (size_t)i0 * esz;
        char* dst = (char*)x_host + (size_t)i0 * esz;
        cudaError_t e = cudaMemcpy2DAsync(g_pipe.buf[j], (size_t)m * esz, src, (size_t)M * esz,
                                          (size_t)m * esz, (size_t)N, cudaMemcpyHostToDevice, g_pipe.st[j]);
        if (e != cudaSuccess) { rc = pent::cuda_fail(e); break; }
        rc = pent_solve_batch(h, m, g_pipe.buf[j], g_pipe.buf[j], g_pipe.st[j]);
        if (rc != PENT_OK) break;
        e = cudaMemcpy2DAsync(dst, (size_t)M * esz, g_pipe.buf[j], (size_t)m * esz, (size_t)m * esz,
                              (size_t)N, cudaMemcpyDeviceToHost, g_pipe.st[j]);
        if (e != cudaSuccess) { rc = pent::cuda_fail(e); break; }
    }
    for (int j = 0; j < NB; ++j) {
        cudaError_t e = cudaStreamSynchronize(g_pipe.st[j]);
        if (e != cudaSuccess && rc == PENT_OK) rc = pent::cuda_fail(e);
    }
    return rc;
}
