// pent_solve_tps.cu -- "thread per system" kernels: the paper's own GPU design
// (interleaved layout, one thread per system, everything in global memory).
// Consecutive threads own consecutive systems, so every access f[k*M+i] of a warp is one
// contiguous, coalesced segment.  The intermediate vector g round-trips through x (the paper
// overwrites the right-hand side): 4 passes over the batch.  This is the
// reference design and the HBM-spill path for N too large to keep on chip; the headline
// kernel is in pent_solve_chunked.cu.
#include <new>
#include "pent_chunk_common.cuh"

namespace pent {

constexpr int TPS_UNROLL = 8;

// Shared A.  Forward sweep with pre-normalised coefficients, then back
// substitution.  The coefficient loads are warp-uniform (one broadcast
// transaction); the f loads of TPS_UNROLL rows are issued together before the dependent FMA chain.
template <typename T>
__global__ void __launch_bounds__(128)
solve_tps_kernel(int N, int64_t M, const typename Vec<T>::T4* __restrict__ fw,
                 const typename Vec<T>::T2* __restrict__ bw, const T* f, T* x)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    const T* fi = f + i;
    T* xi = x + i;
    T g1 = 0, g2 = 0;
    int k = 0;
    for (; k + TPS_UNROLL <= N; k += TPS_UNROLL) {
        T v[TPS_UNROLL];
#pragma unroll
        for (int u = 0; u < TPS_UNROLL; ++u) v[u] = __ldcs(fi + (int64_t)(k + u) * M);
#pragma unroll
        for (int u = 0; u < TPS_UNROLL; ++u) {
            typename Vec<T>::T4 c = ldg4(fw + k + u);
            T g = fma(-c.z, g1, fma(-c.y, g2, c.x * v[u]));
            xi[(int64_t)(k + u) * M] = g;
            g2 = g1; g1 = g;
        }
    }
    for (; k < N; ++k) {
        typename Vec<T>::T4 c = ldg4(fw + k);
        T g = fma(-c.z, g1, fma(-c.y, g2, c.x * fi[(int64_t)k * M]));
        xi[(int64_t)k * M] = g;
        g2 = g1; g1 = g;
    }
    T x1 = 0, x2 = 0;
    k = N - 1;
    for (; k - TPS_UNROLL + 1 >= 0; k -= TPS_UNROLL) {
        T v[TPS_UNROLL];
#pragma unroll
        for (int u = 0; u < TPS_UNROLL; ++u) v[u] = xi[(int64_t)(k - u) * M];
#pragma unroll
        for (int u = 0; u < TPS_UNROLL; ++u) {
            typename Vec<T>::T2 c = ldg2(bw + k - u);
            T xv = fma(-c.y, x2, fma(-c.x, x1, v[u]));
            __stcs(xi + (int64_t)(k - u) * M, xv);
            x2 = x1; x1 = xv;
        }
    }
    for (; k >= 0; --k) {
        typename Vec<T>::T2 c = ldg2(bw + k);
        T xv = fma(-c.y, x2, fma(-c.x, x1, xi[(int64_t)k * M]));
        xi[(int64_t)k * M] = xv;
        x2 = x1; x1 = xv;
    }
}

int launch_solve_tps(const pent_handle* h, int64_t M, const void* f, void* x, cudaStream_t s)
{
    const int tb = 128;
    unsigned nb = (unsigned)((M + tb - 1) / tb);
    if (h->dtype == PENT_F64)
        solve_tps_kernel<double><<<nb, tb, 0, s>>>(h->N, M, (const double4*)h->fw,
                                                   (const double2*)h->bw, (const double*)f, (double*)x);
    else
        solve_tps_kernel<float><<<nb, tb, 0, s>>>(h->N, M, (const float4*)h->fw,
                                                  (const float2*)h->bw, (const float*)f, (float*)x);
    count_launch();
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}

// ---------------------------------------------------------------------------------------------
// Per-system matrices.  Thread i factors A_i on the fly (the paper's steps 8.1-8.4 with
// out-of-matrix entries masked to zero) while sweeping forward, keeps gamma_k, delta_k (needed
// again by the back substitution) in two batch-sized arrays and g in x.
// One reciprocal per row; every other division becomes a multiply.
//   MODE 0: fused factor+solve (gam/del are scratch)      -- pent_factor_solve_batch
//   MODE 1: factor only, store ia,en,bn,gamma,delta        -- pent_factor_batch
// ---------------------------------------------------------------------------------------------
constexpr int PS_UNROLL = 8;     // rows whose loads are issued together (6 streams x 8 rows in flight per thread)
constexpr int PS_THREADS = 64;   // small blocks: M is the only parallelism, spread it over all SMs

template <typename T, int MODE>
__global__ void __launch_bounds__(PS_THREADS)
factor_tps_kernel(int N, int64_t M, const T* __restrict__ a, const T* __restrict__ b,
                  const T* __restrict__ c, const T* __restrict__ d, const T* __restrict__ e,
                  const T* f, T* x, T* __restrict__ gam, T* __restrict__ del,
                  T* __restrict__ ia_o, T* __restrict__ en_o, T* __restrict__ bn_o,
                  int* __restrict__ info)
{
    constexpr int U = PS_UNROLL;
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    T ga1 = 0, ga2 = 0, de1 = 0, de2 = 0, g1 = 0, g2 = 0;
    int bad = 0;
    for (int k0 = 0; k0 < N; k0 += U) {
        // The serial recurrence below waits on nothing but registers: all loads of the next U rows
        // are in flight before its first step (latency, not bandwidth, bounds one thread per system).
        T av[U], bv[U], cv[U], dv[U], ev[U], fv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int k = k0 + u;
            const int64_t o = (int64_t)k * M + i;
            av[u] = (k >= 2 && k < N) ? __ldcs(a + o) : (T)0;
            bv[u] = (k >= 1 && k < N) ? __ldcs(b + o) : (T)0;
            cv[u] = (k < N) ? __ldcs(c + o) : (T)1;
            dv[u] = (k + 1 < N) ? __ldcs(d + o) : (T)0;
            ev[u] = (k + 2 < N) ? __ldcs(e + o) : (T)0;
            if (MODE == 0) fv[u] = (k < N) ? f[o] : (T)0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int k = k0 + u;
            if (k < N) {
                const int64_t o = (int64_t)k * M + i;
                T be = fma(-av[u], ga2, bv[u]);
                T al = fma(-be, ga1, fma(-av[u], de2, cv[u]));
                if (bad == 0 && (al == (T)0 || !isfinite(al))) bad = k + 1;
                T inv = (T)1 / al;
                T ga = fma(-be, de1, dv[u]) * inv;
                T de = ev[u] * inv;
                gam[o] = ga; del[o] = de;
                if (MODE == 0) {
                    T g = fma(-be, g1, fma(-av[u], g2, fv[u])) * inv;
                    x[o] = g;
                    g2 = g1; g1 = g;
                } else {
                    ia_o[o] = inv; en_o[o] = av[u] * inv; bn_o[o] = be * inv;
                }
                ga2 = ga1; ga1 = ga; de2 = de1; de1 = de;
            }
        }
    }
    if (info) info[i] = bad;
    if (MODE == 0) {
        T x1 = 0, x2 = 0;
        for (int k0 = N - 1; k0 >= 0; k0 -= U) {
            T gv[U], dv[U], xv[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int k = k0 - u;
                const int64_t o = (int64_t)k * M + i;
                gv[u] = (k >= 0) ? gam[o] : (T)0;
                dv[u] = (k >= 0) ? del[o] : (T)0;
                xv[u] = (k >= 0) ? x[o] : (T)0;
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int k = k0 - u;
                if (k >= 0) {
                    T r = fma(-dv[u], x2, fma(-gv[u], x1, xv[u]));
                    __stcs(x + (int64_t)k * M + i, r);
                    x2 = x1; x1 = r;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Fused per-system factor + solve with a cp.async ring (default for pent_factor_solve_batch).
// One thread per system still (the factor recurrence is serial and nonlinear in the matrix
// entries), but M is the only parallelism (cfg5b: 16384 threads on 148 SMs), so every thread must
// keep ~0.5-1 KB of loads in flight on its own: each thread streams ITS column of the six input
// arrays through a private slice of a shared-memory ring with 8-byte cp.async copies, RING_STAGES-1
// stages ahead of the recurrence.  No block barrier: a thread only reads what it copied itself.
// Forward: stage = RING_ROWS rows x {a,b,c,d,e,f}; backward: stage = 2*RING_ROWS rows x {gamma,
// delta, g} (same stage size).  cfg5b: 418 us with register load-ahead -> see profiles/r01_ab_tuning.md.
// ---------------------------------------------------------------------------------------------
#ifndef PENT_RING_ROWS
#define PENT_RING_ROWS 4
#endif
constexpr int RING_ROWS = PENT_RING_ROWS, RING_STAGES = 6, RING_SLOTS = 6 * RING_ROWS;   // values per thread and stage

template <typename T>
__global__ void __launch_bounds__(PS_THREADS)
factor_solve_ring_kernel(int N, int64_t M, const T* __restrict__ a, const T* __restrict__ b,
                         const T* __restrict__ c, const T* __restrict__ d, const T* __restrict__ e,
                         const T* f, T* x, T* __restrict__ scratch, int* __restrict__ info)
{
    constexpr int R = RING_ROWS, NST = RING_STAGES, TB = PS_THREADS;
    extern __shared__ __align__(16) unsigned char ring_raw[];
    T* ring = reinterpret_cast<T*>(ring_raw);           // [NST][RING_SLOTS][TB]
    int64_t i = (int64_t)blockIdx.x * TB + threadIdx.x;
    if (i >= M) i = M - 1;                                // tail threads redo the last system (no divergent exits)
    const bool writer = ((int64_t)blockIdx.x * TB + threadIdx.x) < M;
    T* mine = ring + threadIdx.x;
    // gamma_k, delta_k, g_k of this block's systems: [k][3][TB], private to the block and contiguous, so the
    // six scratch words per unknown (3 written, 3 read back) are sequential DRAM streams, not three more
    // arrays of pitch M
    T* sc = scratch + (size_t)blockIdx.x * N * 3 * TB + threadIdx.x;
    auto slot = [&](int stage, int v) -> T* { return mine + (size_t)(stage * RING_SLOTS + v) * TB; };

    // ---------------- forward: factor rows and sweep in the same loop ----------------
    const int nblk = (N + R - 1) / R;
    auto issue_fwd = [&](int blk) {
        if (blk < nblk) {
            const int st = blk % NST;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int k = blk * R + r;
                if (k < N) {
                    const int64_t o = (int64_t)k * M + i;
                    cp_async_elem(slot(st, 0 * R + r), a + o);
                    cp_async_elem(slot(st, 1 * R + r), b + o);
                    cp_async_elem(slot(st, 2 * R + r), c + o);
                    cp_async_elem(slot(st, 3 * R + r), d + o);
                    cp_async_elem(slot(st, 4 * R + r), e + o);
                    cp_async_elem(slot(st, 5 * R + r), f + o);
                }
            }
        }
        cp_async_commit();
    };
    for (int blk = 0; blk < NST - 1; ++blk) issue_fwd(blk);
    T ga1 = 0, ga2 = 0, de1 = 0, de2 = 0, g1 = 0, g2 = 0;
    int bad = 0;
    for (int blk = 0; blk < nblk; ++blk) {
        issue_fwd(blk + NST - 1);
        cp_async_wait<NST - 1>();
        const int st = blk % NST;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int k = blk * R + r;
            if (k < N) {
                const int64_t o = (int64_t)k * M + i;
                const T ak = (k >= 2) ? *slot(st, 0 * R + r) : (T)0;
                const T bk = (k >= 1) ? *slot(st, 1 * R + r) : (T)0;
                const T ck = *slot(st, 2 * R + r);
                const T dk = (k + 1 < N) ? *slot(st, 3 * R + r) : (T)0;
                const T ek = (k + 2 < N) ? *slot(st, 4 * R + r) : (T)0;
                const T fk = *slot(st, 5 * R + r);
                T be = fma(-ak, ga2, bk);
                T al = fma(-be, ga1, fma(-ak, de2, ck));
                if (bad == 0 && (al == (T)0 || !isfinite(al))) bad = k + 1;
                T inv = (T)1 / al;
                T ga = fma(-be, de1, dk) * inv;
                T de = ek * inv;
                T g = fma(-be, g1, fma(-ak, g2, fk)) * inv;
                { T* w = sc + (size_t)k * 3 * TB; w[0] = ga; w[TB] = de; w[2 * TB] = g; }
                g2 = g1; g1 = g;
                ga2 = ga1; ga1 = ga; de2 = de1; de1 = de;
            }
        }
    }
    if (info && writer) info[i] = bad;
    cp_async_wait<0>();
    __threadfence();              // this thread's gamma, delta, g are in L2 before it copies them back

    // ---------------- backward: x_k = g_k - gamma_k x_{k+1} - delta_k x_{k+2} ----------------
    constexpr int RB = 2 * R;
    const int nblk_b = (N + RB - 1) / RB;
    auto issue_bwd = [&](int blk) {
        if (blk < nblk_b) {
            const int st = blk % NST;
#pragma unroll
            for (int r = 0; r < RB; ++r) {
                const int k = N - 1 - (blk * RB + r);
                if (k >= 0) {
                    const int64_t o = (int64_t)k * M + i;
                    const T* w = sc + (size_t)k * 3 * TB;
                    cp_async_elem(slot(st, 0 * RB + r), w);
                    cp_async_elem(slot(st, 1 * RB + r), w + TB);
                    cp_async_elem(slot(st, 2 * RB + r), w + 2 * TB);
                }
            }
        }
        cp_async_commit();
    };
    for (int blk = 0; blk < NST - 1; ++blk) issue_bwd(blk);
    T x1 = 0, x2 = 0;
    for (int blk = 0; blk < nblk_b; ++blk) {
        issue_bwd(blk + NST - 1);
        cp_async_wait<NST - 1>();
        const int st = blk % NST;
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int k = N - 1 - (blk * RB + r);
            if (k >= 0) {
                T xv = fma(-*slot(st, 1 * RB + r), x2, fma(-*slot(st, 0 * RB + r), x1, *slot(st, 2 * RB + r)));
                if (writer) __stcs(x + (int64_t)k * M + i, xv);
                x2 = x1; x1 = xv;
            }
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// Two threads per system ("burn at both ends"): M is the only parallelism of the per-system problem (cfg5b: 16384
// systems = 3.5 warps per SM with one thread per system), and each thread is one long dependent chain (a division per
// row), so the ring kernel above is bound by the latency of single warps (issue 20 %, no unit above 55 %).  Here the
// system is cut in the middle, m = ceil(N/2):
//     thread T: rows 0 .. m-1 top-down  = LU of the leading block A_TT, forward sweep of f_T;
//     thread B: rows N-1 .. m bottom-up = the same recurrence on the REVERSED trailing block (reversing rows and
//               columns of a pentadiagonal matrix swaps a <-> e, b <-> d), forward sweep of the reversed f_B.
// The halves are coupled only through (x_{m-2}, x_{m-1}) and (x_m, x_{m+1}): A_TT x_T = f_T - C_T (x_m, x_{m+1}) with C_T
// non-zero in its last two rows only, so L_T^{-1} C_T is non-zero in its last two rows only and the last two unknowns of
// each half are  p - P (the other half's two)  with p (2 values) and P (2 x 2) known at the end of its forward loop.  The two
// threads swap (p, P) through shared memory, each solves the 4 x 4 interface system (as two 2 x 2), and then runs its
// ordinary back substitution outward from the two interface values; the rows above the interface use the spilled
// gamma, delta, g unchanged.  Same traffic as the ring kernel (13 words per unknown), twice the warps, chains of half
// the length.  Exactly A_i^{-1} f_i (a twisted factorisation, no pivoting: the leading and the reversed trailing block of
// an SPD / diagonally dominant matrix are SPD / diagonally dominant); it differs from the oracle's LU by rounding only.
// info[i]: the first zero / non-finite pivot met by thread T, else by thread B, as row + 1 (a pivot of the twisted
// factorisation; for the top half it is the pivot of the paper's LU).
// Block = TW_SYS threads T followed by TW_SYS threads B of the same TW_SYS systems.  Measured on cfg5b (profiles/
// r02_bench_all.jsonl; A/B PENT_AB_PER_SYSTEM_ONE_THREAD=1): 381.5 -> 270 us fp64, 240 -> 208 us fp32 (of which the second
// thread alone, at the ring depth of the one-thread kernel: 361 us; the rest is the ring depth below).
// ---------------------------------------------------------------------------------------------
// Ring depth and block width, measured on cfg5b (fp64, us per call; A/B by -DPENT_TW_STAGES / -DPENT_TW_SYS / -DPENT_RING_ROWS
// through PENT_NVCC_FLAGS): (systems per block, rows per stage, stages) = (64,4,3) 270, (128,4,3) 269, (64,4,2) 365,
// (64,4,4) 361, (64,8,3) 340, (64,2,3) 357, (64,2,4) 357, (32,4,3) 368, (32,4,6) 325, (32,2,8) 357.  Two stages of 4 rows
// ahead (8 rows, 3 stages) is a sharp optimum: deeper rings put more of the six input streams and the scratch stream in
// flight than the memory system serves well, shallower ones expose latency.  At 270 us the call moves its 13 words per
// unknown at 6.2 TB/s: it is at the cap of the 13-word design (0.54 of the 7-word roofline).
#ifndef PENT_TW_STAGES
#define PENT_TW_STAGES 3
#endif
#ifndef PENT_TW_SYS
#define PENT_TW_SYS 64
#endif
constexpr int TW_STAGES = PENT_TW_STAGES, TW_SYS = PENT_TW_SYS;

template <typename T>
__global__ void __launch_bounds__(2 * TW_SYS)
factor_solve_twist_kernel(int N, int64_t M, const T* __restrict__ a, const T* __restrict__ b,
                          const T* __restrict__ c, const T* __restrict__ d, const T* __restrict__ e,
                          const T* f, T* x, T* __restrict__ scratch, int* __restrict__ info)
{
    constexpr int R = RING_ROWS, NST = TW_STAGES, TB = 2 * TW_SYS;
    extern __shared__ __align__(16) unsigned char ring_raw[];
    T* ring = reinterpret_cast<T*>(ring_raw);           // [NST][RING_SLOTS][TB]
    T* xch = ring + (size_t)NST * RING_SLOTS * TB;       // [2][7][TW_SYS]: p (2), P (4), bad pivot
    const int lane = threadIdx.x & (TW_SYS - 1), half = threadIdx.x / TW_SYS;
    int64_t i = (int64_t)blockIdx.x * TW_SYS + lane;
    const bool writer = i < M;
    if (i >= M) i = M - 1;                                // tail lanes redo the last system (no divergent exits)
    const int m = (N + 1) / 2, len = half ? N - m : m;   // rows of this thread's half
    // local step s = 0 .. len-1  <->  row k(s); the roles of the diagonals in the (reversed) local system
    auto krow = [&](int s) -> int { return half ? N - 1 - s : s; };
    const T* sub2 = half ? e : a;
    const T* sub1 = half ? d : b;
    const T* sup1 = half ? b : d;
    const T* sup2 = half ? a : e;
    T* mine = ring + threadIdx.x;
    T* sc = scratch + (size_t)blockIdx.x * N * 3 * TW_SYS + lane;       // [k][3][TW_SYS], private to the block
    auto slot = [&](int stage, int v) -> T* { return mine + (size_t)(stage * RING_SLOTS + v) * TB; };

    // ---------------- forward: factor the rows of this half and sweep in the same loop ----------------
    const int nblk = (len + R - 1) / R;
    auto issue_fwd = [&](int blk) {
        if (blk < nblk) {
            const int st = blk % NST;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int s = blk * R + r;
                if (s < len) {
                    const int64_t o = (int64_t)krow(s) * M + i;
                    cp_async_elem(slot(st, 0 * R + r), sub2 + o);
                    cp_async_elem(slot(st, 1 * R + r), sub1 + o);
                    cp_async_elem(slot(st, 2 * R + r), c + o);
                    cp_async_elem(slot(st, 3 * R + r), sup1 + o);
                    cp_async_elem(slot(st, 4 * R + r), sup2 + o);
                    cp_async_elem(slot(st, 5 * R + r), f + o);
                }
            }
        }
        cp_async_commit();
    };
    for (int blk = 0; blk < NST - 1; ++blk) issue_fwd(blk);
    T ga1 = 0, ga2 = 0, de1 = 0, de2 = 0, g1 = 0, g2 = 0;
    T inv1 = 0, inv2 = 0, be1 = 0;             // 1/alpha of the last two rows, beta of the last row
    T c20 = 0, c10 = 0, c11 = 0;               // couplings to the other half: sup2 of row len-2; sup1, sup2 of row len-1
    int bad = 0;
    for (int blk = 0; blk < nblk; ++blk) {
        issue_fwd(blk + NST - 1);
        cp_async_wait<NST - 1>();
        const int st = blk % NST;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int s = blk * R + r;
            if (s < len) {
                const int k = krow(s);
                const T ak = (s >= 2) ? *slot(st, 0 * R + r) : (T)0;
                const T bk = (s >= 1) ? *slot(st, 1 * R + r) : (T)0;
                const T ck = *slot(st, 2 * R + r);
                const T dr = *slot(st, 3 * R + r), er = *slot(st, 4 * R + r);
                const T dk = (s + 1 < len) ? dr : (T)0;          // entries that leave the half are not part of its LU
                const T ek = (s + 2 < len) ? er : (T)0;
                if (s == len - 2) c20 = er;
                if (s == len - 1) { c10 = dr; c11 = er; }
                const T fk = *slot(st, 5 * R + r);
                T be = fma(-ak, ga2, bk);
                T al = fma(-be, ga1, fma(-ak, de2, ck));
                if (bad == 0 && (al == (T)0 || !isfinite(al))) bad = k + 1;
                T inv = (T)1 / al;
                T ga = fma(-be, de1, dk) * inv;
                T de = ek * inv;
                T g = fma(-be, g1, fma(-ak, g2, fk)) * inv;
                { T* w = sc + (size_t)k * 3 * TW_SYS; w[0] = ga; w[TW_SYS] = de; w[2 * TW_SYS] = g; }
                g2 = g1; g1 = g;
                ga2 = ga1; ga1 = ga; de2 = de1; de1 = de;
                inv2 = inv1; inv1 = inv; be1 = be;
            }
        }
    }
    cp_async_wait<0>();
    __threadfence();              // this thread's gamma, delta, g are in L2 before it copies them back

    // ---------------- interface: (y_{len-2}, y_{len-1}) = p - P u,  u = the other half's (y_{len-1}, y_{len-2}) -----------
    // rows len-2, len-1 of L^{-1} C (C = the couplings above, columns u0, u1), then two steps of back substitution
    // (ga2 = gamma of row len-2 after the loop's last shift)
    // (columns outside the matrix -- row N of the top half when N is odd and tiny -- do not occur: N >= 8)
    const T G20 = c20 * inv2;                                   // row len-2: [c20, 0]
    const T G10 = fma(-be1, G20, c10) * inv1, G11 = c11 * inv1; // row len-1: [c10, c11] - beta [G20, 0]
    T pv[2], Pm[4];
    pv[1] = g1;                      Pm[2] = G10;                   Pm[3] = G11;
    pv[0] = fma(-ga2, g1, g2);       Pm[0] = fma(-ga2, G10, G20);   Pm[1] = -ga2 * G11;
    {
        T* o = xch + (size_t)half * 7 * TW_SYS + lane;
        o[0] = pv[0]; o[TW_SYS] = pv[1]; o[2 * TW_SYS] = Pm[0]; o[3 * TW_SYS] = Pm[1]; o[4 * TW_SYS] = Pm[2]; o[5 * TW_SYS] = Pm[3];
        o[6 * TW_SYS] = (T)bad;
    }
    __syncthreads();
    T qv[2], Qm[4];
    {
        const T* o = xch + (size_t)(1 - half) * 7 * TW_SYS + lane;
        qv[0] = o[0]; qv[1] = o[TW_SYS]; Qm[0] = o[2 * TW_SYS]; Qm[1] = o[3 * TW_SYS]; Qm[2] = o[4 * TW_SYS]; Qm[3] = o[5 * TW_SYS];
        const int obad = (int)o[6 * TW_SYS];
        if (info && writer && half == 0) info[i] = bad ? bad : obad;
    }
    // mine = pv - Pm S other,  other = qv - Qm S mine  (S swaps the two entries)  =>  (I - Pm S Qm S) mine = pv - Pm S qv
    // Pm S = columns swapped: (Pm S)[r] = {Pm[2r+1], Pm[2r]}
    T y2, y1;                                  // this half's (y_{len-2}, y_{len-1})
    {
        const T A0 = Pm[1], A1 = Pm[0], A2 = Pm[3], A3 = Pm[2];          // Pm S
        const T B0 = Qm[1], B1 = Qm[0], B2 = Qm[3], B3 = Qm[2];          // Qm S
        const T K0 = (T)1 - fma(A0, B0, A1 * B2), K1 = -fma(A0, B1, A1 * B3);
        const T K2 = -fma(A2, B0, A3 * B2), K3 = (T)1 - fma(A2, B1, A3 * B3);
        const T r0 = pv[0] - fma(A0, qv[0], A1 * qv[1]), r1 = pv[1] - fma(A2, qv[0], A3 * qv[1]);
        const T det = fma(K0, K3, -K1 * K2);
        y2 = fma(K3, r0, -K1 * r1) / det;
        y1 = fma(K0, r1, -K2 * r0) / det;
    }

    // ---------------- backward: outward from the interface, x_s = g_s - gamma_s x_{s+1} - delta_s x_{s+2} ----------------
    if (writer) {
        __stcs(x + (int64_t)krow(len - 1) * M + i, y1);
        __stcs(x + (int64_t)krow(len - 2) * M + i, y2);
    }
    constexpr int RB = 2 * R;
    const int rest = len - 2;                   // local steps len-3 .. 0
    const int nblk_b = (rest + RB - 1) / RB;
    auto issue_bwd = [&](int blk) {
        if (blk < nblk_b) {
            const int st = blk % NST;
#pragma unroll
            for (int r = 0; r < RB; ++r) {
                const int s = rest - 1 - (blk * RB + r);
                if (s >= 0) {
                    const T* w = sc + (size_t)krow(s) * 3 * TW_SYS;
                    cp_async_elem(slot(st, 0 * RB + r), w);
                    cp_async_elem(slot(st, 1 * RB + r), w + TW_SYS);
                    cp_async_elem(slot(st, 2 * RB + r), w + 2 * TW_SYS);
                }
            }
        }
        cp_async_commit();
    };
    for (int blk = 0; blk < NST - 1; ++blk) issue_bwd(blk);
    T x1 = y2, x2 = y1;
    for (int blk = 0; blk < nblk_b; ++blk) {
        issue_bwd(blk + NST - 1);
        cp_async_wait<NST - 1>();
        const int st = blk % NST;
#pragma unroll
        for (int r = 0; r < RB; ++r) {
            const int s = rest - 1 - (blk * RB + r);
            if (s >= 0) {
                T xv = fma(-*slot(st, 1 * RB + r), x2, fma(-*slot(st, 0 * RB + r), x1, *slot(st, 2 * RB + r)));
                if (writer) __stcs(x + (int64_t)krow(s) * M + i, xv);
                x2 = x1; x1 = xv;
            }
        }
    }
    cp_async_wait<0>();
}

// Solve with stored per-system factors (layout ms: ia, en, bn, gamma, delta, each N*M).
template <typename T>
__global__ void __launch_bounds__(PS_THREADS)
solve_multi_kernel(int N, int64_t M, const T* __restrict__ ms, const T* f, T* x)
{
    constexpr int U = PS_UNROLL;
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    const int64_t NM = (int64_t)N * M;
    T g1 = 0, g2 = 0;
    for (int k0 = 0; k0 < N; k0 += U) {
        T iv[U], ev[U], bv[U], fv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int k = k0 + u;
            const int64_t o = (int64_t)k * M + i;
            const bool in = k < N;
            iv[u] = in ? ms[o] : (T)0; ev[u] = in ? ms[NM + o] : (T)0; bv[u] = in ? ms[2 * NM + o] : (T)0;
            fv[u] = in ? f[o] : (T)0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int k = k0 + u;
            if (k < N) {
                T g = fma(-bv[u], g1, fma(-ev[u], g2, iv[u] * fv[u]));
                x[(int64_t)k * M + i] = g;
                g2 = g1; g1 = g;
            }
        }
    }
    T x1 = 0, x2 = 0;
    for (int k0 = N - 1; k0 >= 0; k0 -= U) {
        T gv[U], dv[U], xv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int k = k0 - u;
            const int64_t o = (int64_t)k * M + i;
            gv[u] = (k >= 0) ? ms[3 * NM + o] : (T)0;
            dv[u] = (k >= 0) ? ms[4 * NM + o] : (T)0;
            xv[u] = (k >= 0) ? x[o] : (T)0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int k = k0 - u;
            if (k >= 0) {
                T r = fma(-dv[u], x2, fma(-gv[u], x1, xv[u]));
                x[(int64_t)k * M + i] = r;
                x2 = x1; x1 = r;
            }
        }
    }
}

template <typename T>
static int factor_solve_impl(int N, int64_t M, const void* e, const void* c, const void* d,
                             const void* a, const void* b, const void* f, void* x, int* info,
                             void* workspace, cudaStream_t s)
{
    // gamma_k, delta_k, g_k of every system (needed again by the back substitution): 3*N*M' elements,
    // M' = M rounded up to a multiple of 64; the caller's workspace or a stream-ordered temporary
    T* scratch = (T*)workspace;
    size_t NM = (size_t)N * (size_t)M;
    if (!scratch) {
        cudaError_t er = cudaMallocAsync((void**)&scratch, 3 * (size_t)N * (size_t)((M + 63) / 64 * 64) * sizeof(T), s);
        if (er == cudaErrorMemoryAllocation) { cudaGetLastError(); return PENT_ERR_ALLOC; }
        PENT_CUDA(er);
    }
    const int tb = PS_THREADS;
    unsigned nb = (unsigned)((M + tb - 1) / tb);
#ifdef PENT_AB_NO_RING
    factor_tps_kernel<T, 0><<<nb, tb, 0, s>>>(N, M, (const T*)a, (const T*)b, (const T*)c,
                                              (const T*)d, (const T*)e, (const T*)f, (T*)x,
                                              scratch, scratch + NM, nullptr, nullptr, nullptr, info);
#else
    static const int one_thread = []() { const char* ev = std::getenv("PENT_AB_PER_SYSTEM_ONE_THREAD"); return ev ? std::atoi(ev) : 0; }();
    if (N >= 8 && !one_thread) {        // two threads per system (workspace: 3 N ceil64(M), the contract's size)
        const size_t smem = ((size_t)TW_STAGES * RING_SLOTS * 2 * TW_SYS + 2 * 7 * TW_SYS) * sizeof(T);
        static SmemOnce mark2;
        PENT_CUDA(ensure_dynamic_smem(mark2, factor_solve_twist_kernel<T>, smem));
        nb = (unsigned)((M + TW_SYS - 1) / TW_SYS);
        factor_solve_twist_kernel<T><<<nb, 2 * TW_SYS, smem, s>>>(N, M, (const T*)a, (const T*)b, (const T*)c, (const T*)d,
                                                                   (const T*)e, (const T*)f, (T*)x, scratch, info);
    } else {
        const size_t smem = (size_t)RING_STAGES * RING_SLOTS * PS_THREADS * sizeof(T);
        static SmemOnce mark;
        PENT_CUDA(ensure_dynamic_smem(mark, factor_solve_ring_kernel<T>, smem));
        factor_solve_ring_kernel<T><<<nb, tb, smem, s>>>(N, M, (const T*)a, (const T*)b, (const T*)c, (const T*)d,
                                                         (const T*)e, (const T*)f, (T*)x, scratch, info);
    }
#endif
    count_launch();
    cudaError_t le = cudaGetLastError();
    if (!workspace) cudaFreeAsync(scratch, s);
    if (le != cudaSuccess) return cuda_fail(le);
    return PENT_OK;
}

template <typename T>
static int factor_batch_impl(pent_handle* h, const void* e, const void* c, const void* d,
                             const void* a, const void* b, int* info_dev, cudaStream_t s)
{
    size_t NM = (size_t)h->N * (size_t)h->M;
    T* ms = (T*)h->ms;
    const int tb = PS_THREADS;
    unsigned nb = (unsigned)((h->M + tb - 1) / tb);
    factor_tps_kernel<T, 1><<<nb, tb, 0, s>>>(h->N, h->M, (const T*)a, (const T*)b, (const T*)c,
                                              (const T*)d, (const T*)e, nullptr, nullptr,
                                              ms + 3 * NM, ms + 4 * NM, ms, ms + NM, ms + 2 * NM,
                                              info_dev);
    count_launch();
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}
}  // namespace pent

extern "C" int pent_factor_solve_batch_ws(int N, int64_t M, const void* e, const void* c,
                                          const void* d, const void* a, const void* b,
                                          const void* f, void* x, pent_dtype dtype, int* info,
                                          void* workspace, void* stream)
{
    if (N < 1 || M < 0 || !e || !c || !d || !a || !b || !f || !x) return PENT_ERR_ARG;
    if (M == 0) return PENT_OK;
    cudaStream_t s = (cudaStream_t)stream;
    if (dtype == PENT_F64) return pent::factor_solve_impl<double>(N, M, e, c, d, a, b, f, x, info, workspace, s);
    if (dtype == PENT_F32) return pent::factor_solve_impl<float>(N, M, e, c, d, a, b, f, x, info, workspace, s);
    return PENT_ERR_ARG;
}

extern "C" int pent_factor_solve_batch(int N, int64_t M, const void* e, const void* c,
                                       const void* d, const void* a, const void* b,
                                       const void* f, void* x, pent_dtype dtype, int* info,
                                       void* stream)
{
    return pent_factor_solve_batch_ws(N, M, e, c, d, a, b, f, x, dtype, info, nullptr, stream);
}

extern "C" int pent_factor_batch(int N, int64_t M, const void* e, const void* c, const void* d,
                                 const void* a, const void* b, pent_dtype dtype,
                                 pent_handle** out, int* info, void* stream)
{
    if (!out) return PENT_ERR_ARG;
    *out = nullptr;
    if (N < 1 || M < 1 || !e || !c || !d || !a || !b) return PENT_ERR_ARG;
    if (dtype != PENT_F64 && dtype != PENT_F32) return PENT_ERR_ARG;
    pent_handle* h = new (std::nothrow) pent_handle();
    if (!h) return PENT_ERR_ALLOC;
    *h = pent_handle{};
    h->kind = 1; h->N = N; h->M = M; h->dtype = dtype; h->l2_bc = -1; h->band = 2;
    if (cudaGetDevice(&h->device) != cudaSuccess) { delete h; return pent::cuda_fail(cudaGetLastError()); }
    size_t esz = dtype == PENT_F64 ? 8 : 4;
    cudaError_t er = cudaMalloc(&h->ms, 5 * (size_t)N * (size_t)M * esz);
    if (er != cudaSuccess) {
        cudaGetLastError();
        delete h;
        return er == cudaErrorMemoryAllocation ? PENT_ERR_ALLOC : pent::cuda_fail(er);
    }
    int rc = dtype == PENT_F64
                 ? pent::factor_batch_impl<double>(h, e, c, d, a, b, info, (cudaStream_t)stream)
                 : pent::factor_batch_impl<float>(h, e, c, d, a, b, info, (cudaStream_t)stream);
    if (rc != PENT_OK) { pent_destroy(h); return rc; }
    *out = h;
    return PENT_OK;
}

extern "C" int pent_solve_batch_multi(const pent_handle* h, const void* f, void* x, void* stream)
{
    if (!h || h->kind != 1 || !f || !x || !pent::on_handle_device(h)) return PENT_ERR_ARG;
    const int tb = pent::PS_THREADS;
    unsigned nb = (unsigned)((h->M + tb - 1) / tb);
    cudaStream_t s = (cudaStream_t)stream;
    if (h->dtype == PENT_F64)
        pent::solve_multi_kernel<double><<<nb, tb, 0, s>>>(h->N, h->M, (const double*)h->ms,
                                                           (const double*)f, (double*)x);
    else
        pent::solve_multi_kernel<float><<<nb, tb, 0, s>>>(h->N, h->M, (const float*)h->ms,
                                                          (const float*)f, (float*)x);
    pent::count_launch();
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}

// ---------------------------------------------------------------------------------------------
// pent_factor_solve_batch_noalloc -- the per-system factor + solve for callers that cannot allocate (code under CUDA
// graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same kernels as pent_factor_solve_batch;
// the scratch for gamma_k, delta_k, g_k lives in the file-scope device array below instead of a workspace, so the
// call makes no cudaMalloc / cudaFree / stream-ordered allocation of any kind.
//   * Every GPU that loads libpent.so holds the PENT_NOALLOC_SCRATCH_BYTES of the array until the process exits.
//   * In HOST code the array's name is a host-side stand-in, not a device address: its device address is looked
//     up once per device, with that device current, by cudaGetSymbolAddress (return code checked) and cached.
//   * All calls share the array: two calls that overlap on the GPU (different streams, or graph branches that may
//     run concurrently) race on it.  Nothing has to be cleared between calls: every word a call reads was written
//     earlier by the same thread of the same call (forward loop writes rows k, the back substitution reads them).
// ---------------------------------------------------------------------------------------------
#define PENT_NOALLOC_SCRATCH_BYTES (32u << 20)
static __device__ __align__(256) unsigned char g_noalloc_scratch[PENT_NOALLOC_SCRATCH_BYTES];

namespace pent {
constexpr int NOALLOC_MAX_DEVICES = 64;
static std::atomic<void*> g_noalloc_ptr[NOALLOC_MAX_DEVICES];

// device address of g_noalloc_scratch on the CURRENT device (set-up: once per device)
static int noalloc_scratch(void** out)
{
    int dev = 0;
    PENT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return PENT_ERR_ARG;
    void* p = g_noalloc_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        PENT_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return cuda_fail(cudaErrorInvalidSymbol);
        g_noalloc_ptr[dev].store(p, std::memory_order_release);     // (two racing threads store the same address)
    }
    *out = p;
    return PENT_OK;
}

template <typename T>
static int factor_solve_noalloc_impl(int N, int64_t M, const void* e, const void* c, const void* d, const void* a,
                                     const void* b, const void* f, void* x, int* info, cudaStream_t s)
{
    void* sp = nullptr;
    const int rc = noalloc_scratch(&sp);
    if (rc != PENT_OK) return rc;
    T* scratch = (T*)sp;
    if (N >= 8) {                        // two threads per system: scratch [block][k][3][TW_SYS]
        const size_t smem = ((size_t)TW_STAGES * RING_SLOTS * 2 * TW_SYS + 2 * 7 * TW_SYS) * sizeof(T);
        static SmemOnce mark2;
        PENT_CUDA(ensure_dynamic_smem(mark2, factor_solve_twist_kernel<T>, smem));
        const unsigned nb = (unsigned)((M + TW_SYS - 1) / TW_SYS);
        factor_solve_twist_kernel<T><<<nb, 2 * TW_SYS, smem, s>>>(N, M, (const T*)a, (const T*)b, (const T*)c, (const T*)d,
                                                                   (const T*)e, (const T*)f, (T*)x, scratch, info);
    } else {                             // one thread per system: scratch [block][k][3][PS_THREADS]
        const size_t smem = (size_t)RING_STAGES * RING_SLOTS * PS_THREADS * sizeof(T);
        static SmemOnce mark;
        PENT_CUDA(ensure_dynamic_smem(mark, factor_solve_ring_kernel<T>, smem));
        const unsigned nb = (unsigned)((M + PS_THREADS - 1) / PS_THREADS);
        factor_solve_ring_kernel<T><<<nb, PS_THREADS, smem, s>>>(N, M, (const T*)a, (const T*)b, (const T*)c, (const T*)d,
                                                                 (const T*)e, (const T*)f, (T*)x, scratch, info);
    }
    count_launch();
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}
}  // namespace pent

extern "C" int64_t pent_noalloc_scratch_bytes(void) { return (int64_t)PENT_NOALLOC_SCRATCH_BYTES; }

extern "C" int pent_factor_solve_batch_noalloc(int N, int64_t M, const void* e, const void* c, const void* d,
                                               const void* a, const void* b, const void* f, void* x,
                                               pent_dtype dtype, int* info, void* stream)
{
    if (N < 1 || M < 0 || !e || !c || !d || !a || !b || !f || !x) return PENT_ERR_ARG;
    if (dtype != PENT_F64 && dtype != PENT_F32) return PENT_ERR_ARG;
    if (M == 0) return PENT_OK;
    // 3 * N * M' elements, M' = M rounded up to a multiple of 64 (both kernels' block widths divide 64 or equal it)
    static_assert(64 % pent::PS_THREADS == 0 && (64 % pent::TW_SYS == 0 || pent::TW_SYS == 64), "scratch size formula");
    const uint64_t esz = dtype == PENT_F64 ? 8 : 4;
    const uint64_t Mp = ((uint64_t)M + 63) / 64 * 64;
    if (Mp > (uint64_t)PENT_NOALLOC_SCRATCH_BYTES / (3 * esz * (uint64_t)N)) return PENT_ERR_TOO_LARGE;
    cudaStream_t s = (cudaStream_t)stream;
    if (dtype == PENT_F64) return pent::factor_solve_noalloc_impl<double>(N, M, e, c, d, a, b, f, x, info, s);
    return pent::factor_solve_noalloc_impl<float>(N, M, e, c, d, a, b, f, x, info, s);
}
