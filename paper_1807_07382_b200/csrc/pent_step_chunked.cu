// pent_step_chunked.cu -- fused time stepping with the state ON CHIP across steps
// (BASELINE.json configs[3]; PAPER.md:53 Eq. 2, :87-89 Eq. 6, :117 Eq. 7c, :273).
//
// The systems of a batch never interact, so a CTA can take a tile of S systems through ALL
// `nsteps` steps before it touches HBM again: the tile's state (S x N values, 128 KiB) is loaded
// once by TMA into shared memory, every step builds the explicit right-hand side from it in
// registers (5-point window along k, neighbours of other chunks read from the shared state),
// runs the chunked solve of pent_solve_chunked.cu on the registers (local sweeps, chunk-state
// scan, correction) and writes the new state back to shared memory; after the last step the tile
// goes back to HBM with one TMA store per box.  HBM traffic per launch is 2 passes over the
// state whatever nsteps is (the paper's loop costs 2 kernels and >= 6 passes PER STEP:
// PAPER.md:273); the per-step cost is arithmetic and three block barriers.
//
//  kind 0  Cahn-Hilliard:  form 0  A c+ = c + r L (c^3 - c)
//                          form 1  q = r (c^3 - c) - sigma L c ;  A delta = L q ;  c+ = c + delta
//  kind 1  hyperdiffusion Crank-Nicolson:  A c+ = (2I - A) c   (diagonals read from the handle)
//  (L v)_k = v_{k-1} + dg_k v_k + v_{k+1}, out-of-range terms dropped; dg_k = -2 except
//  dg_0 = dg_{N-1} = -1 when bc = 1 (zero-flux).  Same formulas, in the same order, as
//  step_tps_kernel (pent_step.cu).
#include "pent_chunk_common.cuh"

namespace pent {

template <typename T>
struct StepChunkParams {
    int N, P, Pw, lev_f, lev_b;
    int woff[W_LEVELS];
    int box_rows, nbox;
    uint32_t table_bytes;
    int64_t M, ntiles;
    const T* table;
    const T* dg;          // N x {a,b,c,d,e, cos 2 pi x_k, sin 2 pi x_k, 0} (kind 1; forcing)
    int nsteps, bc;
    T r, sigma;
    // forcing (FORCED = true, reading C-22): per-system parameters and the time axis
    const T* mu1;
    const T* mu2;
    double dt, t0;
};

// Barrier of one thread group of a CTA (named barrier 1+g); the whole CTA when there is one group.
template <int NG>
__device__ __forceinline__ void group_sync(int g, int nthreads)
{
    if constexpr (NG == 1) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + g), "r"(nthreads) : "memory");
}

// NG independent thread groups per CTA, each taking its OWN tile of S systems through the steps
// (own state buffer, own chunk states, own named barrier); they share the coefficient table.  The
// phases of a step alternate between FP64-throughput-bound (right-hand side), latency-bound
// (sweeps, scan) and shared-memory-bound (write-back) work; two groups out of phase fill the pipes
// that one group in lockstep leaves idle.
// FORCED: the travelling-wave forcing of Eq. 3 with per-system (mu1, mu2).  dt Phi(x_k, t_n) = fa cos(2 pi x_k) +
// fb sin(2 pi x_k) with (fa, fb) = dt mu1 (cos, sin)(2 pi mu2 t_n): ONE sincospi per system and step (computed by the
// S threads of chunk 0 one step ahead, under the scan of the current step, double-buffered in shared memory).
// Along k the forcing of one system is a sampled sinusoid, so a thread needs no table loads for its rows: it
// keeps the space factors of its FIRST row in registers for the whole launch and steps the sinusoid with the
// small-angle-stable recurrence  Phi_{j+1} = Phi_j + d_j,  d_{j+1} = d_j - 4 sin^2(pi/N) Phi_{j+1}
// (error growth ~ j u, not j u / sin(2 pi / N) as for the three-term cosine recurrence): 3 flops per unknown.
template <typename T, int S, int KIND, int NG, bool FORCED>
__global__ void __launch_bounds__(CHUNK_MAX_THREADS, 1)
step_chunked_kernel(const __grid_constant__ CUtensorMap tm, const StepChunkParams<T> prm)
{
    constexpr int C = ChunkCfg<T>::C, BL = chunk_block_len<T>();
    using T2 = typename Pair<T>::type;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int P = prm.P, N = prm.N;
    const int TG = blockDim.x / NG, grp_id = threadIdx.x / TG, tid = threadIdx.x % TG;
    const size_t state_elems = (size_t)prm.nbox * prm.box_rows * S;
    T* state = reinterpret_cast<T*>(smem_raw) + grp_id * state_elems;          // [rows][S], this group's tile
    T* table = reinterpret_cast<T*>(smem_raw) + NG * state_elems;
    T2* stE = reinterpret_cast<T2*>(reinterpret_cast<unsigned char*>(table) + prm.table_bytes) +
              (size_t)grp_id * 2 * S * P;
    T2* stS = stE + (size_t)S * P;
    T2* amp_all = reinterpret_cast<T2*>(reinterpret_cast<unsigned char*>(table) + prm.table_bytes) + (size_t)NG * 2 * S * P;
    T2* amp = amp_all + (FORCED ? (size_t)grp_id * 2 * S : 0);                 // [2][S] forcing amplitudes, double-buffered
    uint64_t* bars = reinterpret_cast<uint64_t*>(amp_all + (FORCED ? (size_t)NG * 2 * S : 0));
    uint64_t* bar_state = &bars[1 + grp_id];                                   // [0] table, [1+g] state of group g

    const int i = tid % S, p = tid / S;
    const bool active = p < P;
    const int lane = tid & 31, warp = tid >> 5, nwarps = TG >> 5;
    const uint32_t box_bytes = (uint32_t)(prm.box_rows * S * sizeof(T));

    if (threadIdx.x == 0) {
        for (int b = 0; b <= NG; ++b) mbar_init(&bars[b], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(&bars[0], prm.table_bytes);
        bulk_load_1d(table, prm.table, prm.table_bytes, &bars[0]);
    }
    mbar_wait(&bars[0], 0);

    const T* blk = table + (size_t)(active ? p : 0) * BL;
    const T* wtab = table + (size_t)P * BL;
    const int slot = state_slot<S>(active ? p : 0, i);
    const int row0 = p * C;
    T* cs = state + i;                                   // element (k, i) at cs[k*S]
    const int Pw = prm.Pw, G = 32 / Pw;
    const int q = lane % Pw, grp = lane / Pw;
    const ScanGeom geom{P, Pw, prm.lev_f, prm.lev_b, prm.woff};
    const int rounds = (S + nwarps * G - 1) / (nwarps * G);
    const T r = prm.r, sigma = prm.sigma;
    constexpr bool incr = (KIND == 2);       // KIND: 0 CH direct form, 2 CH increment form, 1 hyperdiffusion
    const T dg_edge = (prm.bc == 1) ? (T)-1 : (T)-2;
    auto ldc = [&](int k) -> T { return ((unsigned)k < (unsigned)N) ? cs[(size_t)k * S] : (T)0; };
    auto Ld = [&](int k) -> T { return (k == 0 || k == N - 1) ? dg_edge : (T)-2; };
    // Warp-uniform choice: a warp that holds one boundary chunk (S=16: two chunks per warp) takes the
    // general path with ALL its lanes instead of executing both paths one after the other; that warp
    // is the straggler every block barrier waits for.
    const bool first = row0 == 0, last = row0 + C == N;
    const T dfirst = first ? dg_edge : (T)-2, dlast = last ? dg_edge : (T)-2;
    const bool interior = __all_sync(0xffffffffu, active && (first || row0 >= 2) && (last || row0 + C + 2 <= N - 1) &&
                                                      C >= 4 && N >= 2 * C);
    uint32_t parity = 0;

    for (int64_t tile = (int64_t)blockIdx.x * NG + grp_id; tile < prm.ntiles; tile += (int64_t)gridDim.x * NG) {
        if (tid == 0) {
            mbar_expect_tx(bar_state, box_bytes * prm.nbox);
            for (int b = 0; b < prm.nbox; ++b)
                tma_load_2d(state + (size_t)b * prm.box_rows * S, &tm, (int)(tile * S), b * prm.box_rows, bar_state);
        }
        mbar_wait(bar_state, parity);
        // forcing amplitudes of system tid (threads of chunk 0) at step n -> amp[n & 1][tid]
        double fm1 = 0.0, fm2 = 0.0;
        // space factors of this thread's first row: (cos, sin)(2 pi x_row0) and their first differences along k,
        // (cos, sin)(theta + dl) - (cos, sin)(theta) = -2 sin^2(dl/2) (cos, sin) -+ sin(dl) (sin, cos), dl = 2 pi / N
        T fcx = 0, fsx = 0, fdcx = 0, fdsx = 0, fkap = 0;
        if constexpr (FORCED) {
            if (active && row0 < N) {
                double sh, ch, sd, cd;
                sincospi(1.0 / (double)N, &sh, &ch);                   // dl / 2
                sincospi(2.0 / (double)N, &sd, &cd);                   // dl
                const double cx = (double)__ldg(prm.dg + 8 * (size_t)row0 + 5), sx = (double)__ldg(prm.dg + 8 * (size_t)row0 + 6);
                const double k2 = 2.0 * sh * sh;
                fcx = (T)cx; fsx = (T)sx;
                fdcx = (T)(-k2 * cx - sd * sx); fdsx = (T)(-k2 * sx + sd * cx);
                fkap = (T)(2.0 * k2);
            }
        }
        auto amp_for_step = [&](int n) {
            double sn, cs;
            sincospi(2.0 * fm2 * (prm.t0 + (double)n * prm.dt), &sn, &cs);
            const double am = prm.dt * fm1;
            T2 ab; ab.x = (T)(am * cs); ab.y = (T)(am * sn);
            amp[(n & 1) * S + tid] = ab;
        };
        if constexpr (FORCED) {
            if (tid < S) {
                const int64_t col = tile * S + tid;
                if (col < prm.M) { fm1 = (double)prm.mu1[col]; fm2 = (double)prm.mu2[col]; }
                amp_for_step(0);
            }
            group_sync<NG>(grp_id, TG);
        }

        for (int step = 0; step < prm.nsteps; ++step) {
            T v[C];
            if (active) {
                // ---- explicit right-hand side of rows row0 .. row0+C-1, in registers ----
                if constexpr (KIND != 1) {
                    // u_k = w_k = c_k^3 - c_k (form 0) or q_k = r w_k - sigma (L c)_k (form 1), 0 outside 0..N-1
                    if (interior) {
                        // Interior chunk, or the first / last chunk of a system whose length is a multiple
                        // of C: the special rows then sit at compile-time positions (j = -1, 0 and C-1, C),
                        // so the loop body carries no range checks; `dfirst`, `dlast` are the diagonal
                        // entries of L at rows row0 and row0+C-1 (-2 unless that row is 0 or N-1).
                        auto U = [&](T cl, T cc, T cr, T dg) -> T {
                            T w = cc * cc * cc - cc;
                            if (!incr) return w;
                            return fma(-sigma, cl + fma(dg, cc, cr), r * w);
                        };
                        const T* cw = cs + (size_t)row0 * S;          // cw[j*S] = c_{row0+j}
                        T cl = first ? (T)0 : *(cw - 2 * S), cc = first ? (T)0 : *(cw - S), cr = cw[0];
                        T u_prev = first ? (T)0 : U(cl, cc, cr, (T)-2);                    // u_{row0-1}
                        cl = cc; cc = cr; cr = cw[S];
                        T u_cur = U(cl, cc, cr, dfirst);                                   // u_{row0}
#pragma unroll
                        for (int j = 0; j < C; ++j) {
                            cl = cc; cc = cr;                                              // cl = c_{row0+j}, cc = c_{row0+j+1}
                            if (j + 2 < C) cr = cw[(j + 2) * S];
                            else cr = last ? (T)0 : cw[(j + 2) * S];                       // rows N, N+1 do not exist
                            T u_next = U(cl, cc, cr, (j + 1 == C - 1) ? dlast : (T)-2);    // u_{row0+j+1}
                            if (j == C - 1 && last) u_next = 0;                            // u_N
                            T Lu = u_prev + fma(j == 0 ? dfirst : (j == C - 1 ? dlast : (T)-2), u_cur, u_next);
                            v[j] = incr ? Lu : fma(r, Lu, cl);
                            u_prev = u_cur; u_cur = u_next;
                        }
                    } else {
                        auto U = [&](int k, T cl, T cc, T cr) -> T {
                            if ((unsigned)k >= (unsigned)N) return (T)0;
                            T w = cc * cc * cc - cc;
                            if (!incr) return w;
                            return fma(-sigma, cl + fma(Ld(k), cc, cr), r * w);
                        };
                        T cl = ldc(row0 - 2), cc = ldc(row0 - 1), cr = ldc(row0);
                        T u_prev = U(row0 - 1, cl, cc, cr);
                        cl = cc; cc = cr; cr = ldc(row0 + 1);
                        T u_cur = U(row0, cl, cc, cr);
#pragma unroll
                        for (int j = 0; j < C; ++j) {
                            const int k = row0 + j;
                            cl = cc; cc = cr; cr = ldc(k + 2);          // window centred on k+1; cl = c_k
                            T u_next = U(k + 1, cl, cc, cr);
                            T Lu = u_prev + fma(Ld(k), u_cur, u_next);
                            v[j] = incr ? Lu : fma(r, Lu, cl);
                            u_prev = u_cur; u_cur = u_next;
                        }
                    }
                } else if (interior) {
                    // (2I - A) c, rows row0 .. row0+C-1 all inside the matrix (see `interior` above); the
                    // entries of the diagonals that fall outside the matrix are zero in prm.dg
                    const T* cw = cs + (size_t)row0 * S;
                    T cm2 = first ? (T)0 : *(cw - 2 * S), cm1 = first ? (T)0 : *(cw - S), c0 = cw[0], cp1 = cw[S];
                    const T* dk = prm.dg + 8 * (size_t)row0;
#pragma unroll
                    for (int j = 0; j < C; ++j) {
                        T cp2;
                        if (j + 2 < C) cp2 = cw[(j + 2) * S];
                        else cp2 = last ? (T)0 : cw[(j + 2) * S];
                        T s = __ldg(dk + 8 * j + 2) * c0;
                        s = fma(__ldg(dk + 8 * j + 1), cm1, s);
                        s = fma(__ldg(dk + 8 * j + 0), cm2, s);
                        s = fma(__ldg(dk + 8 * j + 3), cp1, s);
                        s = fma(__ldg(dk + 8 * j + 4), cp2, s);
                        v[j] = (T)2 * c0 - s;
                        cm2 = cm1; cm1 = c0; c0 = cp1; cp1 = cp2;
                    }
                } else {
                    T cm2 = ldc(row0 - 2), cm1 = ldc(row0 - 1), c0 = ldc(row0), cp1 = ldc(row0 + 1);
#pragma unroll
                    for (int j = 0; j < C; ++j) {
                        const int k = row0 + j;
                        T cp2 = ldc(k + 2);
                        T rhs = 0;
                        if (k < N) {
                            const T* dk = prm.dg + 8 * (size_t)k;
                            T s = __ldg(dk + 2) * c0;
                            s = fma(__ldg(dk + 1), cm1, s);
                            s = fma(__ldg(dk + 0), cm2, s);
                            s = fma(__ldg(dk + 3), cp1, s);
                            s = fma(__ldg(dk + 4), cp2, s);
                            rhs = (T)2 * c0 - s;
                        }
                        v[j] = rhs;
                        cm2 = cm1; cm1 = c0; c0 = cp1; cp1 = cp2;
                    }
                }
                if constexpr (FORCED) {
                    const T2 ab = amp[(step & 1) * S + i];
                    T ph = fma(ab.x, fcx, ab.y * fsx), dph = fma(ab.x, fdcx, ab.y * fdsx);
                    if (row0 + C <= N) {
#pragma unroll
                        for (int j = 0; j < C; ++j) { v[j] += ph; ph += dph; dph = fma(-fkap, ph, dph); }
                    } else {
#pragma unroll
                        for (int j = 0; j < C; ++j) {
                            if (row0 + j < N) v[j] += ph;
                            ph += dph;
                            dph = fma(-fkap, ph, dph);
                        }
                    }
                }
                // ---- chunked solve, stages 1+2 ----
                T2 e, s;
                chunk_local_sweeps<T>(v, blk, e, s);
                stE[slot] = e;
                stS[slot] = s;
            }
            group_sync<NG>(grp_id, TG);
            if constexpr (FORCED) {
                if (tid < S && step + 1 < prm.nsteps) amp_for_step(step + 1);   // read after two more barriers
            }
            if (P > 1) {
                for (int rr = 0; rr < rounds; ++rr) {
                    const int sys = (rr * nwarps + warp) * G + grp;
                    chunk_state_scan<T, S, false>(geom, wtab, stE, stS, sys, q, (sys < S) && (q < P), 0, 1,
                                                  nullptr, nullptr, bars, 0u, 0u, 0u);
                }
            }
            group_sync<NG>(grp_id, TG);
            if (active) {
                T F0 = 0, F1 = 0, B0 = 0, B1 = 0;
                if (P > 1) { T2 fo = stE[slot]; F0 = fo.x; F1 = fo.y; T2 bo = stS[slot]; B0 = bo.x; B1 = bo.y; }
                T* co = cs + (size_t)row0 * S;
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T xv[4];
                    chunk_correct4<T>(xv, &v[4 * jg], blk, jg, F0, F1, B0, B1);
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr) {
                        T* o = co + (size_t)(4 * jg + rr) * S;
                        *o = incr ? *o + xv[rr] : xv[rr];
                    }
                }
            }
            group_sync<NG>(grp_id, TG);       // the next step's windows read rows written by other threads
        }
        // ---- tile back to HBM: generic-proxy writes -> async proxy, then one TMA store per box ----
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        group_sync<NG>(grp_id, TG);
        if (tid == 0) {
            for (int b = 0; b < prm.nbox; ++b)
                tma_store_2d(&tm, (int)(tile * S), b * prm.box_rows, state + (size_t)b * prm.box_rows * S);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory may be overwritten
        }
        group_sync<NG>(grp_id, TG);
        parity ^= 1;
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// Shape of a step launch: NG groups of TG threads, each with a tile of S systems.
struct StepPlan {
    bool ok = false;
    ChunkPlan pl;
    int S = 0, NG = 1, TG = 0;
    size_t smem = 0;
};

static StepPlan step_plan(const pent_handle* h, int64_t M, const void* c, int S, int NG)
{
    StepPlan sp;
    if (!h || h->kind != 0 || h->periodic) return sp;
    const size_t esz = h->dtype == PENT_F64 ? 8 : 4;
    sp.pl = make_plan(h, M, c, 1, S, /*any_S=*/true);
    if (!sp.pl.ok) return sp;
    sp.S = S; sp.NG = NG; sp.TG = sp.pl.threads;
    if (sp.TG * NG > CHUNK_MAX_THREADS) return sp;
    sp.smem = (size_t)NG * ((size_t)sp.pl.nbox * sp.pl.box_rows * S * esz + (size_t)4 * sp.pl.Pl * S * esz) +
              sp.pl.table_bytes + (size_t)(1 + NG) * sizeof(uint64_t) +
              (size_t)NG * 4 * S * esz;                                    // forcing amplitudes (used when FORCED)
    sp.ok = sp.smem <= SMEM_LIMIT;
    return sp;
}

// Default, measured on cfg4 (1000 steps, same box, profiles/r01_ab_tuning.md): fp64 one group of 16
// systems 29.15 us per step against 30.8 for two groups of 8 (narrower tiles double the coefficient
// broadcasts per system and the shared-memory pipe is the busiest unit); fp32 two groups of 16
// systems 20.2 us against 22.2 for one group of 32.
static StepPlan step_auto_plan(const pent_handle* h, int64_t M, const void* c)
{
    if (!h || !chunk_stitching_stable(h)) return StepPlan{};
    if (h->dtype == PENT_F64) return step_plan(h, M, c, 16, 1);
    StepPlan two = step_plan(h, M, c, 16, 2);
    if (two.ok) return two;
    return step_plan(h, M, c, 32, 1);
}

template <typename T, int S, int KIND, int NG, bool FORCED>
static int launch_step_inst(const pent_handle* h, const StepPlan& sp, const pent_step_params* p, const pent_forcing* fg,
                            int64_t M, void* c, int nsteps, cudaStream_t s)
{
    const ChunkPlan& pl = sp.pl;
    StepChunkParams<T> prm;
    prm.N = h->N; prm.P = pl.Pl; prm.Pw = pl.Pw; prm.M = M;
    int lg = 0;
    while ((1 << lg) < pl.Pw) ++lg;
    prm.lev_f = h->lev_f[0] < lg ? h->lev_f[0] : lg;
    prm.lev_b = h->lev_b[0] < lg ? h->lev_b[0] : lg;
    for (int l = 0; l < W_LEVELS; ++l) prm.woff[l] = w_level_off(pl.Pl, l, 1);
    prm.box_rows = pl.box_rows; prm.nbox = pl.nbox;
    prm.ntiles = (M + S - 1) / S;
    prm.table = (const T*)h->cf[0];
    prm.table_bytes = (uint32_t)pl.table_bytes;
    prm.dg = (const T*)h->dg;
    prm.nsteps = nsteps; prm.bc = p->bc;
    prm.r = (T)p->r; prm.sigma = (T)p->sigma;
    prm.mu1 = prm.mu2 = nullptr; prm.dt = prm.t0 = 0.0;
    if (FORCED) { prm.mu1 = (const T*)fg->mu1; prm.mu2 = (const T*)fg->mu2; prm.dt = fg->dt; prm.t0 = fg->t0; }
    CUtensorMap tm;
    if (!encode_batch_map_cached(&tm, c, M, h->N, S, prm.box_rows, sizeof(T) == 8)) {
        g_last_cuda_error = (int)cudaErrorInvalidValue;
        return PENT_ERR_CUDA;
    }
    auto kern = step_chunked_kernel<T, S, KIND, NG, FORCED>;
    static SmemOnce mark;
    PENT_CUDA(ensure_dynamic_smem(mark, kern, sp.smem));
    const int threads = sp.TG * NG;
    int dev = 0, nsm = 0, occ = 0;
    PENT_CUDA(cudaGetDevice(&dev));
    PENT_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    PENT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, sp.smem));
    if (occ < 1) return PENT_ERR_ARG;
    int64_t grid = (int64_t)nsm * occ;
    const int64_t need = (prm.ntiles + NG - 1) / NG;
    if (grid > need) grid = need;
    kern<<<(unsigned)grid, threads, sp.smem, s>>>(tm, prm);
    count_launch();
    PENT_LAUNCH_CHECK();
    return PENT_OK;
}

bool step_chunked_supported(const pent_handle* h, int64_t M, const void* c)
{
    return h && h->kind == 0 && step_auto_plan(h, M, c).ok;
}

template <typename T, int S, int NG>
static int launch_step_kind(const pent_handle* h, const StepPlan& sp, const pent_step_params* p, const pent_forcing* fg,
                            int64_t M, void* c, int nsteps, cudaStream_t s)
{
    if (p->kind == 1) return launch_step_inst<T, S, 1, NG, false>(h, sp, p, nullptr, M, c, nsteps, s);
    if (fg) {
        if (p->form == 1) return launch_step_inst<T, S, 2, NG, true>(h, sp, p, fg, M, c, nsteps, s);
        return launch_step_inst<T, S, 0, NG, true>(h, sp, p, fg, M, c, nsteps, s);
    }
    if (p->form == 1) return launch_step_inst<T, S, 2, NG, false>(h, sp, p, nullptr, M, c, nsteps, s);
    return launch_step_inst<T, S, 0, NG, false>(h, sp, p, nullptr, M, c, nsteps, s);
}

int launch_step_chunked(const pent_handle* h, const pent_step_params* p, const pent_forcing* fg, int64_t M, void* c,
                        int nsteps, cudaStream_t s)
{
    const StepPlan sp = step_auto_plan(h, M, c);
    if (!sp.ok) return PENT_ERR_ARG;
    if (h->dtype == PENT_F64) return launch_step_kind<double, 16, 1>(h, sp, p, fg, M, c, nsteps, s);
    if (sp.NG == 2) return launch_step_kind<float, 16, 2>(h, sp, p, fg, M, c, nsteps, s);
    return launch_step_kind<float, 32, 1>(h, sp, p, fg, M, c, nsteps, s);
}
}  // namespace pent
