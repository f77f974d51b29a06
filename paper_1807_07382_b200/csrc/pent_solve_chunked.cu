// pent_solve_chunked.cu -- the headline solve kernel: 2 passes over HBM (read f once, write x
// once), the intermediate vector g never leaves the SM.
//
// WHY NOT ONE THREAD PER SYSTEM (the paper's design): one system's g is N values
// (8 KiB at N=1024 fp64); a warp of 32 systems needs 256 KiB on chip, more than an SM has, so
// g must round-trip through memory (4 passes).  Because A is SHARED by all systems, the sweeps
// are linear recurrences with system-independent coefficients, so k can be split into chunks
// of C rows solved independently from a zero state and stitched exactly:
//
//   chunk p (rows s..s+C-1), thread (system i, chunk p) holds its C values in registers
//   1. local forward sweep from g_{s-2}=g_{s-1}=0      -> g~ ,  E~_p = last two g~
//   2. local back substitution of g~ from x_{e+1}=x_{e+2}=0 -> x^ , S^_p = first two x^
//   3. chunk states, serial over the P chunks of a system (2x2 matrices from the handle):
//        F_p = E~_p + TPhi_p F_{p-1}                      true (g_{e-1}, g_e) of chunk p
//        B_p = S^_p + TX_p F_{p-1} + TPsi_p B_{p+1}       true (x_s, x_{s+1}) of chunk p
//   4. x_{s+j} = x^_j + chi0_j F_{p-1,0} + chi1_j F_{p-1,1} + psi0_j B_{p+1,0} + psi1_j B_{p+1,1}
//
//   Phi = response of the forward recurrence to a unit incoming state, X = local back
//   substitution of Phi, Psi = response of the backward recurrence to a unit incoming state.
//   All are functions of the shared factors only and are built once in pent_factor.  Exact in
//   exact arithmetic; in fp64 it differs from the serial sweep by rounding only.
//
// DATA MOVEMENT (persistent CTAs, tile = S systems x the rows of this CTA):
//   f tile --TMA (cp.async.bulk.tensor.2d, <= 4 boxes, mbarrier complete_tx)--> smem landing
//   buffer --LDS--> registers; each box is re-armed with the NEXT tile's load as soon as the warps
//   that read it have their rows in registers, so that load runs under this tile's arithmetic,
//   scan and stores.  x goes registers --st.global--> HBM as full 128/256-byte row segments.
//   The shared coefficient tables (9 values per row) are staged ONCE per CTA into shared memory
//   with one cp.async.bulk; every sweep step reads them as 16-byte warp-broadcast LDS.
// LARGER N / WIDER TILES: a thread-block cluster splits k between its CTAs and stitches the block
//   aggregates through distributed shared memory (chunk_state_scan in pent_chunk_common.cuh).
// This file: the tables (built once per handle and cluster size), the launch plans and dispatch.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include "pent_chunked_launch.cuh"

namespace pent {

// ------------------------------------------------------------------------------------------
// table construction (once per handle and cluster size): fp64 arithmetic, rounded to T
// ------------------------------------------------------------------------------------------
// One thread per GLOBAL chunk p = rank*Pl + local chunk; writes the chunk's coefficient block
// into its rank's table and its three 2x2 end matrices (TPhi | TX | TPsi) into tmat.
template <typename T>
__global__ void build_chunk_tables_kernel(int N, int Pl, int Q, const double* __restrict__ fac,
                                          T* __restrict__ tab, size_t tab_stride,
                                          double* __restrict__ tmat, unsigned long long* __restrict__ growth)
{
    constexpr int C = ChunkCfg<T>::C;
    constexpr int BL = chunk_block_len<T>();
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= Pl * Q) return;
    const double *eps = fac, *beta = fac + N, *alpha = fac + 2 * N, *gamma = fac + 3 * N,
                 *delta = fac + 4 * N;
    T* blk = tab + (size_t)(p / Pl) * tab_stride + (size_t)(p % Pl) * BL;
    const int s = p * C;
    double phi0[C], phi1[C];
    double gphi = 0.0, gchi = 0.0, gpsi = 0.0;     // growth of the three responses inside this chunk (stability guard)
    // forward: coefficients and Phi
    double h0m2 = 1.0, h0m1 = 0.0, h1m2 = 0.0, h1m1 = 1.0;
    for (int j = 0; j < C; ++j) {
        int k = s + j;
        double ia = 0.0, en = 0.0, bn = 0.0;
        if (k < N) { ia = 1.0 / alpha[k]; en = eps[k] / alpha[k]; bn = beta[k] / alpha[k]; }
        blk[3 * j + 0] = (T)ia; blk[3 * j + 1] = (T)en; blk[3 * j + 2] = (T)bn;
        double h0 = -en * h0m2 - bn * h0m1;
        double h1 = -en * h1m2 - bn * h1m1;
        phi0[j] = h0; phi1[j] = h1;
        gphi = fmax(gphi, fmax(fabs(h0), fabs(h1)));
        h0m2 = h0m1; h0m1 = h0; h1m2 = h1m1; h1m1 = h1;
    }
    double* cm = tmat + (size_t)p * 12;         // TPhi | TX | TPsi, fp64, for the product kernel
    cm[0] = phi0[C - 2]; cm[1] = phi1[C - 2]; cm[2] = phi0[C - 1]; cm[3] = phi1[C - 1];
    // backward: coefficients, X = local back substitution of Phi, Psi
    double x0p1 = 0.0, x0p2 = 0.0, x1p1 = 0.0, x1p2 = 0.0;     // chi_{j+1}, chi_{j+2}
    double q0p1 = 1.0, q0p2 = 0.0, q1p1 = 0.0, q1p2 = 1.0;     // psi_{j+1}, psi_{j+2}
    for (int j = C - 1; j >= 0; --j) {
        int k = s + j;
        double ga = 0.0, de = 0.0;
        if (k < N) { ga = gamma[k]; de = delta[k]; }
        blk[3 * C + 2 * j + 0] = (T)ga; blk[3 * C + 2 * j + 1] = (T)de;
        double x0 = phi0[j] - ga * x0p1 - de * x0p2;
        double x1 = phi1[j] - ga * x1p1 - de * x1p2;
        double q0 = -ga * q0p1 - de * q0p2;
        double q1 = -ga * q1p1 - de * q1p2;
        T* o = blk + 5 * C + 4 * j;
        o[0] = (T)x0; o[1] = (T)x1; o[2] = (T)q0; o[3] = (T)q1;
        gchi = fmax(gchi, fmax(fabs(x0), fabs(x1)));
        gpsi = fmax(gpsi, fmax(fabs(q0), fabs(q1)));
        if (j <= 1) {
            cm[4 + 2 * j] = x0; cm[5 + 2 * j] = x1;      // TX rows 0,1
            cm[8 + 2 * j] = q0; cm[9 + 2 * j] = q1;      // TPsi rows 0,1
        }
        x0p2 = x0p1; x0p1 = x0; x1p2 = x1p1; x1p1 = x1;
        q0p2 = q0p1; q0p1 = q0; q1p2 = q1p1; q1p1 = q1;
    }
    for (int j = 9 * C; j < BL; ++j) blk[j] = (T)0;
    if (growth) {      // non-negative doubles order like their bit patterns; NaN (bits above +inf) wins, as it should
        atomicMax(&growth[0], (unsigned long long)__double_as_longlong(gphi));
        atomicMax(&growth[1], (unsigned long long)__double_as_longlong(gchi));
        atomicMax(&growth[2], (unsigned long long)__double_as_longlong(gpsi));
    }
}

__device__ inline void mat2_mul(double* o, const double* A, const double* B)     // o = A B (row-major 2x2)
{
    double r0 = A[0] * B[0] + A[1] * B[2], r1 = A[0] * B[1] + A[1] * B[3];
    double r2 = A[2] * B[0] + A[3] * B[2], r3 = A[2] * B[1] + A[3] * B[3];
    o[0] = r0; o[1] = r1; o[2] = r2; o[3] = r3;
}

// Products of the chunk transfer matrices.  One block per cluster rank (blockIdx.x), thread q =
// local chunk (Pl <= 32).  Windows never cross the block: inside a CTA the scan starts from a zero
// state and the state entering the block is applied afterwards through PF / PB.
//   WF_{q,2d} = WF_{q,d} WF_{q-d,d},   WB_{q,2d} = WB_{q,d} WB_{q+d,d}   (doubling)
// levels[0], levels[1] (atomicMax over ranks) = number of Kogge-Stone levels the forward /
// backward scan must apply: a level whose every entry is below 1e-25 in magnitude (and all levels
// above it) cannot change a double-precision state and is skipped (for diagonally dominant A the
// products decay geometrically, so typically 2-3 levels remain).
template <typename T>
__global__ void build_chunk_products_kernel(int Pl, int Q, const double* __restrict__ tmat,
                                            T* __restrict__ tab, size_t tab_stride,
                                            int* __restrict__ levels)
{
    __shared__ double wf[W_LEVELS][MAX_PL][4], wb[W_LEVELS][MAX_PL][4];
    __shared__ double pf[MAX_PL][4], pb[MAX_PL][4], blkm[8 * PENT_MAXQ];
    __shared__ int need_f, need_b;
    const int q = threadIdx.x, rank = blockIdx.x;
    const double* tm = tmat + (size_t)rank * Pl * 12;
    T* wtab = tab + (size_t)rank * tab_stride + (size_t)Pl * chunk_block_len<T>();
    if (q == 0) { need_f = 0; need_b = 0; }
    for (int l = 0; l < W_LEVELS; ++l)
        for (int e = 0; e < 4; ++e) { wf[l][q][e] = 0.0; wb[l][q][e] = 0.0; }
    if (q < Pl) {
        for (int e = 0; e < 4; ++e) {
            wf[0][q][e] = (q >= 1) ? tm[q * 12 + e] : 0.0;                 // TPhi_q acts on F_{q-1}
            wb[0][q][e] = (q + 1 <= Pl - 1) ? tm[q * 12 + 8 + e] : 0.0;    // TPsi_q acts on B_{q+1}
        }
    }
    if (q == 0) {            // prefix products, serial
        for (int e = 0; e < 4; ++e) pf[0][e] = tm[e];
        for (int j = 1; j < Pl; ++j) mat2_mul(pf[j], tm + j * 12, pf[j - 1]);
    }
    if (q == 1) {
        for (int e = 0; e < 4; ++e) pb[Pl - 1][e] = tm[(Pl - 1) * 12 + 8 + e];
        for (int j = Pl - 2; j >= 0; --j) mat2_mul(pb[j], tm + j * 12 + 8, pb[j + 1]);
    }
    if (q == 2) {   // block products of every rank (each block computes all of them)
        for (int r = 0; r < PENT_MAXQ; ++r) {
            double f[4] = {1.0, 0.0, 0.0, 1.0}, b[4] = {1.0, 0.0, 0.0, 1.0};
            if (r < Q) {
                const double* t = tmat + (size_t)r * Pl * 12;
                for (int j = 0; j < Pl; ++j) mat2_mul(f, t + j * 12, f);            // TPhi_j ... TPhi_0
                for (int j = Pl - 1; j >= 0; --j) mat2_mul(b, t + j * 12 + 8, b);   // TPsi_j ... TPsi_last
            }
            for (int e = 0; e < 4; ++e) { blkm[4 * r + e] = f[e]; blkm[4 * PENT_MAXQ + 4 * r + e] = b[e]; }
            // levels[8]: some block transfer product is not negligible -> the cluster must exchange with every rank
            if (r < Q)
                for (int e = 0; e < 4; ++e)
                    if (!(fabs(f[e]) < 1e-25) || !(fabs(b[e]) < 1e-25)) atomicMax(&levels[8], 1);
        }
    }
    __syncthreads();
    for (int l = 1; l < W_LEVELS; ++l) {
        const int d = 1 << (l - 1);       // combine two windows of d chunks
        if (q < Pl && q >= 2 * d) mat2_mul(wf[l][q], wf[l - 1][q], wf[l - 1][q - d]);
        if (q < Pl && q + 2 * d <= Pl - 1) mat2_mul(wb[l][q], wb[l - 1][q], wb[l - 1][q + d]);
        __syncthreads();
    }
    if (q < Pl) {
        for (int l = 0; l < W_LEVELS; ++l) {
            double mf = 0.0, mb = 0.0;
            const int d = 1 << l, n = Pl - d;
            T* base = wtab + w_level_off(Pl, l, Q);
            for (int e = 0; e < 4; ++e) {
                if (q >= d) base[e * n + (q - d)] = (T)wf[l][q][e];
                if (q + d <= Pl - 1) base[4 * n + e * n + q] = (T)wb[l][q][e];
                mf = fmax(mf, fabs(wf[l][q][e])); mb = fmax(mb, fabs(wb[l][q][e]));
            }
            if (!(mf < 1e-25)) atomicMax(&need_f, l + 1);      // also catches NaN
            if (!(mb < 1e-25)) atomicMax(&need_b, l + 1);
        }
        for (int e = 0; e < 4; ++e) {
            wtab[(size_t)e * Pl + q] = (T)tm[q * 12 + 4 + e];
            if (Q > 1) {
                wtab[(size_t)(4 + e) * Pl + q] = (T)pf[q][e];
                wtab[(size_t)(8 + e) * Pl + q] = (T)pb[q][e];
            }
        }
    }
    if (Q > 1)
        for (int j = q; j < 8 * PENT_MAXQ; j += blockDim.x) wtab[12 * Pl + j] = (T)blkm[j];
    __syncthreads();
    if (q == 0) { atomicMax(&levels[0], need_f); atomicMax(&levels[1], need_b); }
}

// ---- BAND = 1 (tridiagonal A): scalar versions of the two kernels above --------------------------------------
// block: [ {1/alpha, beta/alpha} x C | gamma x C | {chi, psi} x C | pad ];  tmat: TPhi | TX | TPsi (3 per chunk)
template <typename T>
__global__ void build_tri_tables_kernel(int N, int Pl, int Q, const double* __restrict__ fac,
                                        T* __restrict__ tab, size_t tab_stride, double* __restrict__ tmat)
{
    constexpr int C = ChunkCfg<T>::C;
    constexpr int BL = chunk_block_len<T, 1>();
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= Pl * Q) return;
    const double *beta = fac + N, *alpha = fac + 2 * N, *gamma = fac + 3 * N;
    T* blk = tab + (size_t)(p / Pl) * tab_stride + (size_t)(p % Pl) * BL;
    const int s = p * C;
    double phi[C];
    double hm1 = 1.0;                               // response of g to a unit incoming g_{s-1}
    for (int j = 0; j < C; ++j) {
        int k = s + j;
        double ia = 0.0, bn = 0.0;
        if (k < N) { ia = 1.0 / alpha[k]; bn = beta[k] / alpha[k]; }
        blk[2 * j + 0] = (T)ia; blk[2 * j + 1] = (T)bn;
        double h = -bn * hm1;
        phi[j] = h; hm1 = h;
    }
    double* cm = tmat + (size_t)p * 3;
    cm[0] = phi[C - 1];
    double xp1 = 0.0, qp1 = 1.0;                    // chi_{j+1}, psi_{j+1}
    for (int j = C - 1; j >= 0; --j) {
        int k = s + j;
        double ga = (k < N) ? gamma[k] : 0.0;
        blk[2 * C + j] = (T)ga;
        double x = phi[j] - ga * xp1;
        double q = -ga * qp1;
        blk[3 * C + 2 * j + 0] = (T)x; blk[3 * C + 2 * j + 1] = (T)q;
        if (j == 0) { cm[1] = x; cm[2] = q; }
        xp1 = x; qp1 = q;
    }
    for (int j = 5 * C; j < BL; ++j) blk[j] = (T)0;
}

template <typename T>
__global__ void build_tri_products_kernel(int Pl, int Q, const double* __restrict__ tmat,
                                          T* __restrict__ tab, size_t tab_stride, int* __restrict__ levels)
{
    __shared__ double wf[W_LEVELS][MAX_PL], wb[W_LEVELS][MAX_PL], pf[MAX_PL], pb[MAX_PL], blkm[2 * PENT_MAXQ];
    __shared__ int need_f, need_b;
    const int q = threadIdx.x, rank = blockIdx.x;
    const double* tm = tmat + (size_t)rank * Pl * 3;
    T* wtab = tab + (size_t)rank * tab_stride + (size_t)Pl * chunk_block_len<T, 1>();
    if (q == 0) { need_f = 0; need_b = 0; }
    for (int l = 0; l < W_LEVELS; ++l) { wf[l][q] = 0.0; wb[l][q] = 0.0; }
    if (q < Pl) {
        wf[0][q] = (q >= 1) ? tm[q * 3] : 0.0;
        wb[0][q] = (q + 1 <= Pl - 1) ? tm[q * 3 + 2] : 0.0;
    }
    if (q == 0) { pf[0] = tm[0]; for (int j = 1; j < Pl; ++j) pf[j] = tm[j * 3] * pf[j - 1]; }
    if (q == 1) { pb[Pl - 1] = tm[(Pl - 1) * 3 + 2]; for (int j = Pl - 2; j >= 0; --j) pb[j] = tm[j * 3 + 2] * pb[j + 1]; }
    if (q == 2) {
        for (int r = 0; r < PENT_MAXQ; ++r) {
            double f = 1.0, b = 1.0;
            if (r < Q) {
                const double* t = tmat + (size_t)r * Pl * 3;
                for (int j = 0; j < Pl; ++j) { f *= t[j * 3]; b *= t[j * 3 + 2]; }
            }
            blkm[r] = f; blkm[PENT_MAXQ + r] = b;
            if (r < Q && (!(fabs(f) < 1e-25) || !(fabs(b) < 1e-25))) atomicMax(&levels[8], 1);
        }
    }
    __syncthreads();
    for (int l = 1; l < W_LEVELS; ++l) {
        const int d = 1 << (l - 1);
        if (q < Pl && q >= 2 * d) wf[l][q] = wf[l - 1][q] * wf[l - 1][q - d];
        if (q < Pl && q + 2 * d <= Pl - 1) wb[l][q] = wb[l - 1][q] * wb[l - 1][q + d];
        __syncthreads();
    }
    if (q < Pl) {
        for (int l = 0; l < W_LEVELS; ++l) {
            const int d = 1 << l, n = Pl - d;
            T* base = wtab + w_level_off(Pl, l, Q, 1);
            if (q >= d) base[q - d] = (T)wf[l][q];
            if (q + d <= Pl - 1) base[n + q] = (T)wb[l][q];
            if (!(fabs(wf[l][q]) < 1e-25)) atomicMax(&need_f, l + 1);
            if (!(fabs(wb[l][q]) < 1e-25)) atomicMax(&need_b, l + 1);
        }
        wtab[q] = (T)tm[q * 3 + 1];
        if (Q > 1) { wtab[Pl + q] = (T)pf[q]; wtab[2 * Pl + q] = (T)pb[q]; }
    }
    if (Q > 1)
        for (int j = q; j < 2 * PENT_MAXQ; j += blockDim.x) wtab[3 * Pl + j] = (T)blkm[j];
    __syncthreads();
    if (q == 0) { atomicMax(&levels[0], need_f); atomicMax(&levels[1], need_b); }
}

template <typename T, int BAND>
static int build_tables_t(pent_handle* h, int j, cudaStream_t s)
{
    constexpr int C = ChunkCfg<T>::C;
    const int Q = 1 << j;
    const int P = (h->N + C - 1) / C;
    const int Pl = (P + Q - 1) / Q;
    void*& cfj = BAND == 2 ? h->cf[j] : h->cf1[j];
    cfj = nullptr;
    if (BAND == 2) { h->cfP[j] = 0; h->lev_f[j] = h->lev_b[j] = 0; } else { h->lev_f1[j] = h->lev_b1[j] = 0; }
    if (Pl > MAX_PL || (Q > 1 && Q > P)) return PENT_OK;     // not a usable split: no tables
    const size_t tlen = table_len<T, BAND>(Pl, Q);
    cudaError_t e = cudaMalloc(&cfj, tlen * Q * sizeof(T));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return PENT_ERR_ALLOC; }
    PENT_CUDA(e);
    double* tmat = nullptr;
    int* lev = nullptr;
    // temporaries are stream-ordered allocations on the factor's private stream (cudaFree would synchronise
    // the whole device)
    auto release = [&]() { if (tmat) cudaFreeAsync(tmat, s); if (lev) cudaFreeAsync(lev, s); };
    // lev: 2 ints (levels) followed, 8-byte aligned, by 3 x 8 bytes (growth of Phi, X, Psi), then int [8] = full-exchange flag
    cudaError_t le = cudaMallocAsync((void**)&tmat, sizeof(double) * 12 * Pl * Q, s);
    if (le == cudaSuccess) le = cudaMallocAsync((void**)&lev, 48, s);
    if (le == cudaSuccess) le = cudaMemsetAsync(lev, 0, 48, s);
    unsigned long long* growth = (BAND == 2 && j == 0 && lev) ? reinterpret_cast<unsigned long long*>(lev + 2) : nullptr;
    if (le == cudaSuccess) le = cudaMemsetAsync(cfj, 0, tlen * Q * sizeof(T), s);
    if (le != cudaSuccess) {            // temporaries are released on every path; h->cf[j] belongs to the handle
        release();
        if (le == cudaErrorMemoryAllocation) { cudaGetLastError(); return PENT_ERR_ALLOC; }
        return cuda_fail(le);
    }
    const int tb = 32, nb = (Pl * Q + tb - 1) / tb;
    if constexpr (BAND == 2) {
        build_chunk_tables_kernel<T><<<nb, tb, 0, s>>>(h->N, Pl, Q, h->fac, (T*)cfj, tlen, tmat, growth);
        build_chunk_products_kernel<T><<<Q, 32, 0, s>>>(Pl, Q, tmat, (T*)cfj, tlen, lev);
    } else {
        build_tri_tables_kernel<T><<<nb, tb, 0, s>>>(h->N, Pl, Q, h->fac, (T*)cfj, tlen, tmat);
        build_tri_products_kernel<T><<<Q, 32, 0, s>>>(Pl, Q, tmat, (T*)cfj, tlen, lev);
    }
    count_launch(2);
    le = cudaGetLastError();
    int hl[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    if (le == cudaSuccess) le = cudaMemcpyAsync(hl, lev, 48, cudaMemcpyDeviceToHost, s);
    release();
    if (le == cudaSuccess) le = cudaStreamSynchronize(s);
    if (le != cudaSuccess) return cuda_fail(le);
    if (growth) std::memcpy(h->growth, hl + 2, 3 * sizeof(double));
    const int xd = (hl[8] || Q < 2) ? (Q > 1 ? Q - 1 : 1) : 1;
    if (BAND == 2) { h->cfP[j] = Pl; h->lev_f[j] = hl[0]; h->lev_b[j] = hl[1]; h->xdepth[j] = xd; }
    else { h->lev_f1[j] = hl[0]; h->lev_b1[j] = hl[1]; h->xdepth1[j] = xd; }
    return PENT_OK;
}

int build_chunk_tables(pent_handle* h, cudaStream_t s)
{
    for (int j = 0; j < PENT_NQ; ++j) {
        int rc = h->dtype == PENT_F64 ? build_tables_t<double, 2>(h, j, s) : build_tables_t<float, 2>(h, j, s);
        if (rc != PENT_OK) return rc;
        if (h->band == 1) {       // tridiagonal A: also the 5-word tables of the BAND = 1 instantiation
            rc = h->dtype == PENT_F64 ? build_tables_t<double, 1>(h, j, s) : build_tables_t<float, 1>(h, j, s);
            if (rc != PENT_OK) return rc;
        }
    }
    return PENT_OK;
}


// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        return (EncodeTiledFn)p;
    }();
    return fn;
}

static bool s_instantiated(bool f64, int S, bool cluster)
{
    (void)cluster;
    return f64 ? (S == 16 || S == 32) : (S == 32 || S == 64);
}

// a plan made for the neighbour-only exchange, turned into one for the all-ranks exchange ([Q][S] aggregate slots)
void plan_drop_nbr(ChunkPlan& pl, size_t esz)
{
    if (!pl.nbr) return;
    pl.nbr = false;
    pl.smem += (size_t)(pl.band == 2 ? 2 : 1) * (size_t)(pl.Q - 2) * pl.S * esz;
    if (pl.smem > SMEM_LIMIT) pl.ok = false;
}

ChunkPlan make_plan(const pent_handle* h, int64_t M, const void* f, int Q, int S, bool any_S, bool ldg, int band)
{
    ChunkPlan pl;
    if (!h || h->kind != 0) return pl;
    const bool f64 = h->dtype == PENT_F64;
    const size_t esz = f64 ? 8 : 4;
    int j = 0;
    while ((1 << j) < Q) ++j;
    if ((1 << j) != Q || j >= PENT_NQ || !h->cf[j] || h->cfP[j] < 1) return pl;
    if (band != 2 && (band != 1 || !h->cf1[j])) return pl;
    pl.band = band;
    if (!any_S && !s_instantiated(f64, S, Q > 1)) return pl;
    if (S < 4 || (S & (S - 1)) != 0) return pl;
    const int C = f64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
    pl.j = j; pl.Q = Q; pl.S = S; pl.Pl = h->cfP[j];
    while (pl.Pw < pl.Pl) pl.Pw *= 2;
    int lg = 0;
    while ((1 << lg) < pl.Pw) ++lg;
    const int hlf = band == 2 ? h->lev_f[j] : h->lev_f1[j], hlb = band == 2 ? h->lev_b[j] : h->lev_b1[j];
    pl.levels = hlf > hlb ? hlf : hlb;
    if (pl.levels > lg) pl.levels = lg;
    // cluster: one scan round (the scan registers live across the cluster barriers)
    pl.threads = ((Q > 1 ? pl.Pw * S : pl.Pl * S) + 31) / 32 * 32;
    if (pl.threads > CHUNK_MAX_THREADS) return pl;
    const int rows = pl.Pl * C;
    pl.box_rows = rows < BOX_ROWS_MAX ? rows : BOX_ROWS_MAX;
    pl.nbox = (rows + pl.box_rows - 1) / pl.box_rows;
    if (pl.nbox > MAX_BOXES) return pl;
    const size_t bl = band == 2 ? (f64 ? chunk_block_len<double, 2>() : chunk_block_len<float, 2>())
                                : (f64 ? chunk_block_len<double, 1>() : chunk_block_len<float, 1>());
    pl.table_bytes = ((size_t)pl.Pl * bl + (size_t)w_level_off(pl.Pl, pl.levels, Q, band)) * esz;
    pl.table_bytes = (pl.table_bytes + 15) & ~(size_t)15;     // cp.async.bulk moves multiples of 16 bytes (the
                                                              // scalar W entries of BAND = 1 need not end on one)
    pl.ldg = ldg;
    pl.mode = ldg ? 1 : 0;
    if (ldg) pl.nbox = 0;                                    // no landing buffer
    const size_t st = band == 2 ? 2 : 1;                     // words per chunk state
    // Neighbour-only exchange (chunk_state_scan, NBR): clusters of >= 8 CTAs whose handle says that a state does not survive
    // a whole block (pent_handle::xdepth == 1).  Measured against the all-ranks exchange (A/B: PENT_AB_FULL_EXCHANGE=1 in the
    // environment; M as in bench.py's suite): N=8192 (Q=8) 485 -> 409 us, N=12288 (Q=16) 528 -> 354, N=16384 (Q=16) 834 -> 654.
    // With 4 CTAs it is SLOWER (cfg5a 417 -> 437 us, fp32 200 -> 215: the all-ranks wait keeps the four CTAs of a tile in
    // lock-step, which their shared HBM rows reward), with 2 CTAs the neighbour is every rank: both run the full exchange.
    // It needs two [S] aggregate slots instead of [Q][S], which is what lets the TMA plan of N = 16384 fit shared memory.
    static const int full = []() { const char* e = std::getenv("PENT_AB_FULL_EXCHANGE"); return e ? std::atoi(e) : 0; }();
    pl.nbr = Q >= 8 && !full && !h->periodic && (band == 2 ? h->xdepth[j] : h->xdepth1[j]) == 1;
    pl.smem = (size_t)pl.nbox * pl.box_rows * S * esz + pl.table_bytes + (size_t)2 * st * pl.Pl * S * esz +
              (Q > 1 ? st * (pl.nbr ? 2 : Q) * S * esz : 0) + (3 + 2 * MAX_BOXES) * sizeof(uint64_t);   // one [Q][S] state array
    if (pl.smem > SMEM_LIMIT) return pl;
    if (!ldg) {
        if ((M * (int64_t)esz) % 16 != 0) return pl;        // TMA global stride alignment
        if (f && ((uintptr_t)f % 16) != 0) return pl;       // TMA global address alignment
        if (M > (int64_t)0x7fffffff) return pl;             // TMA coordinates are 32-bit
        if (!encode_fn()) return pl;
    }
    pl.ok = true;
    return pl;
}

// The encoded map depends only on (base, M, N, S, box_rows, dtype): a small per-thread cache of the last
// few, so that a launch-bound solve (cfg1: 11 us, cfg2: 27 us) does not pay the driver's encode on every call.
bool encode_batch_map_cached(CUtensorMap* tm, const void* base, int64_t M, int N, int S, int box_rows, bool f64)
{
    struct Key { const void* base; int64_t M; int N, S, box_rows, f64; };
    struct Cache { Key key[8]; CUtensorMap tm[8]; int n = 0, next = 0; };
    static thread_local Cache c;
    for (int j = 0; j < c.n; ++j) {
        const Key& k = c.key[j];
        if (k.base == base && k.M == M && k.N == N && k.S == S && k.box_rows == box_rows && k.f64 == (int)f64) {
            *tm = c.tm[j];
            return true;
        }
    }
    if (!encode_batch_map(tm, base, M, N, S, box_rows, f64)) return false;
    const int j = c.next;
    c.key[j] = Key{base, M, N, S, box_rows, (int)f64};
    c.tm[j] = *tm;
    c.next = (c.next + 1) & 7;
    if (c.n < 8) ++c.n;
    return true;
}

bool encode_batch_map(CUtensorMap* tm, const void* base, int64_t M, int N, int S, int box_rows, bool f64)
{
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    const size_t esz = f64 ? 8 : 4;
    cuuint64_t gdim[2] = {(cuuint64_t)M, (cuuint64_t)N};
    cuuint64_t gstr[1] = {(cuuint64_t)M * esz};
    cuuint32_t box[2] = {(cuuint32_t)S, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    return enc(tm, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
               const_cast<void*>(base), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, PENT_L2_PROMOTION, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Default plan, from the shape sweeps in profiles/r01_ab_tuning.md (narrow tile S_n = 16 fp64 /
// 32 fp32, wide tile S_w = 2 S_n = 256-byte row segments):
//   * the whole system fits a CTA of <= 256 threads (cfg2-like, N <= 512): one CTA, narrow tile
//     (more, smaller tiles balance better over 148 SMs: cfg2 31.0 us vs 33.6 wide, 32.8 Q=2 wide);
//   * otherwise the smallest cluster with the WIDE tile if that is <= 4 CTAs (cfg3: 190.7 us at
//     Q=2,S=32 vs 220 at Q=1,S=16; fp32 105.1 at Q=2,S=64 vs 111.5 at Q=1,S=32);
//   * otherwise the smallest cluster with the narrow tile (cfg5a: 410.6 us at Q=4,S=16 vs 485 at
//     Q=8,S=32: 8-CTA clusters leave SMs idle on the 16/18/20-SM GPCs).
// Stability guard of the chunk stitching: the local sweeps restart from a zero state, so their
// intermediates exceed the serial sweep's by up to G = max |Phi|, |X|, |Psi| (the responses of the two recurrences to
// a unit incoming state inside one chunk, recorded at factor time), and the rounding noise of the result grows with
// it.  For the SPD matrices I + sigma L^2 G ~ 5 sqrt(sigma) (cfg3: 4, cfg4: 430); a matrix whose recurrences are
// unstable inside a chunk gives G ~ rho^C.  Above the bound PENT_KERNEL_AUTO uses the serial thread-per-system kernel.
bool chunk_stitching_stable(const pent_handle* h)
{
    const double g = h->growth[0] > h->growth[1] ? (h->growth[0] > h->growth[2] ? h->growth[0] : h->growth[2])
                                                 : (h->growth[1] > h->growth[2] ? h->growth[1] : h->growth[2]);
    return g <= (h->dtype == PENT_F64 ? 1e6 : 1e3);          // NaN compares false
}

ChunkPlan chunk_auto_plan(const pent_handle* h, int64_t M, const void* f, bool ring_ok)
{
    if (!h || h->kind != 0) return ChunkPlan{};
    if (!chunk_stitching_stable(h)) return ChunkPlan{};
    const int hb = h->band == 1 ? 1 : 2;        // tridiagonal handle: the BAND = 1 instantiation
    const int Sn = h->dtype == PENT_F64 ? 16 : 32, Sw = 2 * Sn, QMAX = 1 << (PENT_NQ - 1);
    // Store pacing of the BAND = 1 kernel (profiles/r02_pacing.md): with its shorter arithmetic the x stores of a tile
    // run into the TMA loads of the next one; on the two cluster shapes below, holding the stores back ~1.5 us takes
    // large batches from 0.79 / 0.72 to 0.89 / 0.83 of the HBM peak (N = 1024 / 4096), while it costs 5-10 % on the
    // other shapes and on batches of a few tiles per cluster.  Measured heuristic, not a model.
    auto paced = [&](ChunkPlan pl) {
        const int64_t tiles_per_cluster = ((M + pl.S - 1) / pl.S) * pl.Q / 148;
        if (pl.ok && pl.band == 1 && pl.mode == 0 && tiles_per_cluster >= 16 &&
            ((pl.Q == 2 && pl.S == Sw) || (pl.Q == 4 && pl.S == Sn)))
            pl.pace_ns = 1500;
        return pl;
    };
    // Where the rules below arrive at a 4-CTA cluster, an 8-CTA cluster with the WIDE tile is faster when it can use the
    // neighbour-only exchange (fp64, pentadiagonal; measured, M as large as fits: N=1536 336 -> 302 us, N=2048 400 -> 370,
    // N=3072 336 -> 332, N=4096 (cfg5a) 416 -> 406; N=2048 with M=4096: 34.2 -> 31.5; fp32: no difference, left alone)
    auto prefer8 = [&](ChunkPlan pl) {
        if (pl.ok && pl.Q == 4 && hb == 2 && h->dtype == PENT_F64) {
            ChunkPlan p8 = make_plan(h, M, f, 8, Sw, false, false, hb);
            if (p8.ok && p8.nbr) return p8;
        }
        return paced(pl);
    };
    ChunkPlan narrow1 = make_plan(h, M, f, 1, Sn, false, false, hb);
    if (narrow1.ok && narrow1.threads <= 256) return narrow1;
    for (int Q = 1; Q <= 4; Q *= 2) {
        ChunkPlan pl = make_plan(h, M, f, Q, Sw, false, false, hb);
        if (pl.ok) return prefer8(pl);
    }
    for (int Q = 1; Q <= QMAX; Q *= 2) {
        ChunkPlan pl = make_plan(h, M, f, Q, Sn, false, false, hb);
        if (pl.ok) return prefer8(pl);
    }
    for (int Q = 1; Q <= QMAX; Q *= 2) {
        ChunkPlan pl = make_plan(h, M, f, Q, Sw, false, false, hb);
        if (pl.ok) return pl;
    }
    // TMA cannot address this batch (pitch or base not 16-byte aligned).  First choice: the same shapes with the
    // cp.async loader (mode 4: per-thread LDGSTS into a landing buffer, one tile ahead).  The fused periodic kernel
    // (which keeps a cp.async group of its own for the tail rows: ring_ok = false) and shapes whose landing buffer does
    // not fit: the LDG loader.  It has no prefetch of the next tile, so prefer CTAs of <= 256 threads: two of them share an SM and
    // one loads while the other computes.
    static const int no_ring = []() { const char* e = std::getenv("PENT_AB_NO_CPASYNC_LOADER"); return e ? std::atoi(e) : 0; }();   // A/B
    if (ring_ok && !no_ring) {
        const size_t esz = h->dtype == PENT_F64 ? 8 : 4;
        const int C = h->dtype == PENT_F64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
        auto ring = [&](int Q, int S) {
            ChunkPlan pl = make_plan(h, M, f, Q, S, false, true, hb);
            if (!pl.ok) return pl;
            pl.smem += (size_t)pl.Pl * C * S * esz;          // the landing buffer the LDG plan does without
            pl.mode = 4;
            pl.ok = pl.smem <= SMEM_LIMIT;
            return pl;
        };
        // (a system that fits a single CTA of <= 256 threads keeps the LDG loader: two such CTAs per SM overlap their
        // loads better than one CTA with a landing buffer, cfg2's shape with M = 16383: 34.1 against 49.1 us)
        ChunkPlan n1 = make_plan(h, M, f, 1, Sn, false, true, hb);
        if (n1.ok && n1.threads <= 256) return n1;
        for (int Q = 1; Q <= 4; Q *= 2) { ChunkPlan pl = ring(Q, Sw); if (pl.ok) return pl; }
        for (int Q = 1; Q <= QMAX; Q *= 2) { ChunkPlan pl = ring(Q, Sn); if (pl.ok) return pl; }
    }
    for (int Q = 1; Q <= QMAX; Q *= 2) {
        ChunkPlan pl = make_plan(h, M, f, Q, Sn, false, true, hb);
        if (pl.ok && pl.threads <= 256) return pl;
    }
    for (int Q = 1; Q <= QMAX; Q *= 2) {
        ChunkPlan pl = make_plan(h, M, f, Q, Sn, false, true, hb);
        if (pl.ok) return pl;
    }
    return ChunkPlan{};
}

static ChunkPlan resolve_plan(const pent_handle* h, int64_t M, const void* f, int Q, int S)
{
    const int hb = (h && h->kind == 0 && h->band == 1) ? 1 : 2;
    if (Q == 0 && S == 0) return chunk_auto_plan(h, M, f);
    if (Q != 0 && S != 0) {
        ChunkPlan pl = make_plan(h, M, f, Q, S, false, false, hb);
        return pl.ok ? pl : make_plan(h, M, f, Q, S, false, true, hb);
    }
    const int cand[3] = {16, 32, 64};
    if (Q != 0) {
        for (int s : cand) { ChunkPlan pl = make_plan(h, M, f, Q, s, false, false, hb); if (pl.ok) return pl; }
    } else {
        for (int q = 1; q <= (1 << (PENT_NQ - 1)); q *= 2) { ChunkPlan pl = make_plan(h, M, f, q, S, false, false, hb); if (pl.ok) return pl; }
    }
    return ChunkPlan{};
}

bool chunked_supported(const pent_handle* h, int64_t M, const void* f, int Q, int S)
{
    return resolve_plan(h, M, f, Q, S).ok;
}

int chunked_choice(const pent_handle* h, int64_t M, int* Q, int* S)
{
    ChunkPlan pl = chunk_auto_plan(h, M, nullptr);
    if (!pl.ok) return 0;
    *Q = pl.Q; *S = pl.S;
    return 1;
}

// System-major batch (element k of system i at f[i*N + k]).  Default loader: TMA over the tensor {N, M} with
// 128-byte x S boxes and SWIZZLE_128B (ChunkParams::ldg = 3), prefetched one tile ahead exactly like the
// interleaved loader, so the shapes follow chunk_auto_plan.  When TMA cannot address the batch (row pitch
// N*sizeof(T) or base not 16-byte aligned), or on request: the per-thread contiguous LDG.256 loader
// (ldg = 2; no prefetch, so CTAs of <= 256 threads are preferred: two per SM overlap).
bool encode_rows_map_cached(CUtensorMap* tm, const void* base, int64_t M, int N, int S, bool f64)
{
    struct Key { const void* base; int64_t M; int N, S, f64; };
    struct Cache { Key key[8]; CUtensorMap tm[8]; int n = 0, next = 0; };
    static thread_local Cache c;
    for (int j = 0; j < c.n; ++j) {
        const Key& k = c.key[j];
        if (k.base == base && k.M == M && k.N == N && k.S == S && k.f64 == (int)f64) { *tm = c.tm[j]; return true; }
    }
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    const size_t esz = f64 ? 8 : 4;
    cuuint64_t gdim[2] = {(cuuint64_t)N, (cuuint64_t)M};
    cuuint64_t gstr[1] = {(cuuint64_t)N * esz};
    cuuint32_t box[2] = {(cuuint32_t)(128 / esz), (cuuint32_t)S};
    cuuint32_t estr[2] = {1, 1};
    if (enc(tm, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base),
            gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, PENT_L2_PROMOTION,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    const int j = c.next;
    c.key[j] = Key{base, M, N, S, (int)f64};
    c.tm[j] = *tm;
    c.next = (c.next + 1) & 7;
    if (c.n < 8) ++c.n;
    return true;
}

// geometry of shape (Q, S) for a system-major batch in loader mode 2, 3, 5 or 6 (ChunkParams::ldg)
static ChunkPlan rows_shape(const pent_handle* h, int64_t M, const void* f, const void* x, int Q, int S, int mode)
{
    const int hb = h->band == 1 ? 1 : 2;
    ChunkPlan pl = make_plan(h, M, nullptr, Q, S, false, true, hb);          // no landing buffer yet
    if (!pl.ok) return pl;
    plan_drop_nbr(pl, h->dtype == PENT_F64 ? 8 : 4);                          // the system-major instantiations exchange with every rank
    pl.rows = true;
    pl.mode = 2;
    if (mode == 2) return pl;
    const size_t esz = h->dtype == PENT_F64 ? 8 : 4;
    const int C = h->dtype == PENT_F64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
    pl.ok = false;
    // TMA and bulk copies address 16-byte aligned runs only
    if (((size_t)h->N * esz) % 16 != 0 || (f && ((uintptr_t)f % 16) != 0) || M > (int64_t)0x7fffffff) return pl;
    size_t tile_bytes;
    if (mode == 3) {                  // swizzled tensor-tile TMA: barrier groups of <= 256 rows, 1 KiB alignment slack
        if (!encode_fn()) return pl;
        pl.nbox = (pl.Pl * C + pl.box_rows - 1) / pl.box_rows;
        tile_bytes = (size_t)pl.nbox * pl.box_rows * S * esz + 1024;
    } else {                          // 1-D bulk copies: one padded run per system, one barrier group
        if (mode == 6 && x && ((uintptr_t)x % 16) != 0) return pl;
        pl.nbox = 1;
        pl.box_rows = pl.Pl * C;
        tile_bytes = (size_t)S * ((size_t)pl.box_rows * esz + 16);
    }
    pl.smem += tile_bytes * (mode == 6 ? 2 : 1);
    if (pl.smem > SMEM_LIMIT) return pl;
    pl.ldg = false;
    pl.mode = mode;
    pl.ok = true;
    return pl;
}

// loader: 0 = best available (bulk copies both ways, else bulk loads + STG.256 stores, else the LDG.256 loader),
// 1 = LDG.256 loader, 2 = bulk loads + STG.256 stores, 3 = swizzled tensor-tile TMA loads + STG.256 stores (A/B)
static ChunkPlan rows_plan(const pent_handle* h, int64_t M, const void* f, const void* x, int Q, int S, int loader)
{
    if (!h || h->kind != 0 || h->periodic) return ChunkPlan{};
    const int Sn = h->dtype == PENT_F64 ? 16 : 32, Sw = 2 * Sn, QMAX = 1 << (PENT_NQ - 1);
    const int want = loader == 1 ? 2 : loader == 2 ? 5 : loader == 3 ? 3 : 6;
    if (!(Q && S) && !chunk_stitching_stable(h)) return ChunkPlan{};
    if (Q && S) {
        for (int mode : {want, 5, 2}) {
            if (mode > want && want != 6) continue;
            ChunkPlan pl = rows_shape(h, M, f, x, Q, S, mode);
            if (pl.ok) return pl;
        }
        return ChunkPlan{};
    }
    if (want != 2) {
        // Smallest cluster first: a bulk copy then moves the longest contiguous run of a system, which is what the
        // measured sweep rewards (profiles/r02_rows_loader.md: cfg3 shape Q=1 0.71, Q=2 0.59, Q=4 0.58 of the HBM peak).
        // Within a cluster size: the wanted mode before its fall-back (bulk loads + STG stores), wide tile first.
        for (int q = 1; q <= QMAX; q *= 2)
            for (int pass = 0; pass < 2; ++pass) {
                if (pass == 1 && want != 6) break;
                const int mode = pass == 0 ? want : 5;
                for (int s_ : {Sw, Sn}) { ChunkPlan pl = rows_shape(h, M, f, x, q, s_, mode); if (pl.ok) return pl; }
            }
    }
    for (int q = 1; q <= QMAX; q *= 2) {
        ChunkPlan pl = rows_shape(h, M, f, x, q, Sn, 2);
        if (pl.ok && pl.threads <= 256) return pl;
    }
    for (int q = 1; q <= QMAX; q *= 2) {
        ChunkPlan pl = rows_shape(h, M, f, x, q, Sn, 2);
        if (pl.ok) return pl;
    }
    return ChunkPlan{};
}

bool chunked_rows_supported(const pent_handle* h, int64_t M) { return rows_plan(h, M, nullptr, nullptr, 0, 0, 0).ok; }

int chunked_rows_choice(const pent_handle* h, int64_t M, int* Q, int* S, int* mode)
{
    const ChunkPlan pl = rows_plan(h, M, nullptr, nullptr, 0, 0, 0);
    if (!pl.ok) return 0;
    *Q = pl.Q; *S = pl.S; *mode = pl.mode;
    return 1;
}

static int launch_plan(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s);

int launch_solve_chunked_rows(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s,
                              int Q, int S, int loader)
{
    const ChunkPlan pl = rows_plan(h, M, f, x, Q, S, loader);
    if (!pl.ok) return PENT_UNSUPPORTED;
    return launch_plan_rows(h, pl, M, f, x, s);
}

// The 2 x - f epilogue (ADI): the default plans with the pentadiagonal tables and the all-ranks exchange (the instantiations
// of pent_solve_chunked_epi.cu); tridiagonal handles are refused (the caller keeps its stencil path)
int launch_solve_chunked_epi(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s)
{
    if (!h || h->kind != 0 || h->periodic || h->band != 2) return PENT_UNSUPPORTED;
    ChunkPlan pl = chunk_auto_plan(h, M, f);
    if (!pl.ok) return PENT_UNSUPPORTED;
    plan_drop_nbr(pl, h->dtype == PENT_F64 ? 8 : 4);
    if (!pl.ok) return PENT_UNSUPPORTED;
    return launch_plan_epi(h, pl, M, f, x, s);
}

int launch_solve_chunked_rows_epi(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s)
{
    if (!h || h->kind != 0 || h->periodic || h->band != 2) return PENT_UNSUPPORTED;
    const ChunkPlan pl = rows_plan(h, M, f, x, 0, 0, 0);
    if (!pl.ok || pl.mode == 3) return PENT_UNSUPPORTED;
    return launch_plan_epi(h, pl, M, f, x, s);
}

int launch_solve_chunked(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s,
                         int Q, int S)
{
    const ChunkPlan pl = resolve_plan(h, M, f, Q, S);
    if (!pl.ok) return PENT_UNSUPPORTED;
    return launch_plan(h, pl, M, f, x, s);
}

static int launch_plan(const pent_handle* h, const ChunkPlan& pl, int64_t M, const void* f, void* x, cudaStream_t s)
{
    const bool cl = pl.Q > 1;
    const bool nbr = pl.nbr;          // decided by make_plan (it sizes the aggregate slots)
#define PENT_INST(T_, S_, B_) (cl ? (nbr ? launch_inst<T_, S_, true, false, B_, 0, true>(h, pl, M, f, x, s, nullptr)  \
                                         : launch_inst<T_, S_, true, false, B_>(h, pl, M, f, x, s, nullptr))          \
                                  : launch_inst<T_, S_, false, false, B_>(h, pl, M, f, x, s, nullptr))
    if (h->dtype == PENT_F64) {
        if (pl.S == 16) return pl.band == 1 ? PENT_INST(double, 16, 1) : PENT_INST(double, 16, 2);
        if (pl.S == 32) return pl.band == 1 ? PENT_INST(double, 32, 1) : PENT_INST(double, 32, 2);
    } else {
        if (pl.S == 32) return pl.band == 1 ? PENT_INST(float, 32, 1) : PENT_INST(float, 32, 2);
        if (pl.S == 64) return pl.band == 1 ? PENT_INST(float, 64, 1) : PENT_INST(float, 64, 2);
    }
#undef PENT_INST
    return PENT_ERR_ARG;
}
}  // namespace pent
