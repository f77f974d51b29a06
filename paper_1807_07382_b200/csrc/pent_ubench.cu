// pent_ubench.cu -- the three SM-side rates the design notes quote (DESIGN.md sections 6.2, 6.4), measured, not assumed:
//   * FP64 FMA: latency of a dependent chain and throughput per SM (the "alu" roofline of the on-chip step kernel);
//   * shared-memory loads: cycles per warp-wide LDS.64 / LDS.128 when every lane reads the SAME address (the
//     coefficient broadcasts of the sweeps) and when every lane reads its own (tile data);
//   * 64-bit warp shuffles (two SHFL.32): cycles per shuffle with every warp of the SM shuffling (the chunk-state scan).
// Standalone: `python -m paper_1807_07382_b200.build --ubench` builds paper_1807_07382_b200/pent_ubench; run it on the GPU
// box.  One CTA on one SM, clock64() around the loop.  Not part of libpent.so.
#include <cstdio>
#include <cuda_runtime.h>

template <int CH>
__global__ void dfma_chain(double* out, double a, double b, int iters, long long* cyc)
{
    double x[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) x[c] = threadIdx.x + c;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < CH; ++c) x[c] = fma(x[c], a, b);
    }
    long long t1 = clock64();
    double s = 0;
#pragma unroll
    for (int c = 0; c < CH; ++c) s += x[c];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

// W bytes per lane; stride 0: all lanes read one address (broadcast), else lane * stride elements apart
template <int W>
__global__ void lds_rate(double* out, int iters, long long* cyc, int stride)
{
    extern __shared__ double sm[];
    for (int i = threadIdx.x; i < 4096; i += blockDim.x) sm[i] = i;
    __syncthreads();
    double acc = 0;
    const int base = (threadIdx.x >> 5) * 64;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int idx = (base + (i & 15) * 16 + k * 2 + (threadIdx.x & 31) * stride) & 4095;
            if (W == 16) { double2 v = *reinterpret_cast<const double2*>(&sm[idx & ~1]); acc += v.x + v.y; }
            else acc += sm[idx];
        }
    }
    long long t1 = clock64();
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

__global__ void shfl_rate(double* out, int iters, long long* cyc)
{
    double x = threadIdx.x, y = 1.0;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) { y += __shfl_up_sync(0xffffffffu, x, 1 + (k & 3)); x = y * 0.5; }
    }
    long long t1 = clock64();
    out[blockIdx.x * blockDim.x + threadIdx.x] = x + y;
    if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}

int main()
{
    double* out; long long* cyc;
    cudaMalloc(&out, 1 << 24); cudaMalloc(&cyc, 8);
    long long h;
    const int iters = 4096;
#define RUN(CH, THR) { dfma_chain<CH><<<1, THR>>>(out, 1.0000001, 1e-9, iters, cyc); cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost); \
    printf("DFMA  chains/thread=%d threads=%4d : %6.2f cycles per chain step, %6.2f FMA/clk/SM\n", CH, THR, (double)h / iters, (double)CH * THR * iters / h); }
    RUN(1, 32) RUN(4, 32) RUN(1, 128) RUN(4, 128) RUN(2, 256) RUN(4, 256) RUN(1, 512) RUN(2, 512) RUN(4, 512) RUN(2, 1024)
#define RUNL(W, THR, STR) { lds_rate<W><<<1, THR, 32768>>>(out, iters, cyc, STR); cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost); \
    printf("LDS.%-3d %s threads=%4d : %5.2f cycles per warp instruction and SM (%6.1f B/clk into registers)\n", W * 8, STR ? "distinct " : "broadcast", THR, \
           (double)h / (iters * 8.0 * (THR / 32)), (double)W * THR * 8.0 * iters / h); }
    RUNL(16, 256, 0) RUNL(16, 512, 0) RUNL(8, 256, 0) RUNL(8, 512, 0) RUNL(16, 512, 2) RUNL(8, 512, 1)
    for (int thr : {32, 256, 512}) {
        shfl_rate<<<1, thr>>>(out, iters, cyc); cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
        printf("SHFL  64-bit (2 x SHFL.32), dependent, threads=%4d : %6.2f cycles per shuffle and warp, %5.2f cycles per SHFL.32 and SM\n",
               thr, (double)h / (iters * 8.0), (double)h / (iters * 8.0 * 2 * (thr / 32)));
    }
    cudaError_t e = cudaDeviceSynchronize();
    printf("%s\n", cudaGetErrorString(e));
    return e == cudaSuccess ? 0 : 1;
}
