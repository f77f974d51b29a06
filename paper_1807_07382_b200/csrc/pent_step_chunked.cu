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
//  kind 1  hyperdiffusion Crank-Nicolson:  A c+ = (2I - A) c, evaluated as c+ = 2 A^{-1} c - c (no stencil at all)
//          KIND 3 = the same on a PERIODIC handle (the paper's own loop): wrap-around halo rows, the
//          chunked solve of the (N-2) x (N-2) block E, then the Navon tail t and x^ = y - Z t with Z folded into the
//          chunk states (periodic_fold_kernel in pent_periodic.cu); N a multiple of the chunk length
//  (L v)_k = v_{k-1} + dg_k v_k + v_{k+1}, out-of-range terms dropped; dg_k = -2 except
//  dg_0 = dg_{N-1} = -1 when bc = 1 (zero-flux).  Same formulas, in the same order, as
//  step_tps_kernel (pent_step.cu).
#include <cstdlib>
#include "pent_chunk_common.cuh"

namespace pent {

template <typename T>
struct StepChunkParams {
    int N, P, Pw, lev_f, lev_b;
    int woff[W_LEVELS];
    int box_rows, nbox;
    uint32_t table_bytes;
    int64_t M, ntiles, tile0;   // this launch takes tiles [tile0, ntiles) of S systems
    const T* table;
    const T* dg;          // N x {a,b,c,d,e, cos 2 pi x_k, sin 2 pi x_k, 0} (kind 1; forcing)
    int nsteps, bc;
    T r, sigma;
    // forcing (FORCED = true, reading C-22): per-system parameters and the time axis
    const T* mu1;
    const T* mu2;
    double dt, t0;
    ScanOffsets so;       // chunk-state scan: uniform byte offsets of the transfer matrices (SPT > 1)
    // periodic handle (KIND 3; Eqs. 8-12): chunk states of the Z solve, explicit Z rows of the first and last
    // chunk, the six entries of h and the inverted 2 x 2 Schur complement
    const T* pfold;
    const typename Vec<T>::T2* pzedge;
    T ph[6], pi[4];
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
// SPT: systems per thread (pent_chunk_common.cuh): thread (column i, chunk p) carries systems SPT i .. SPT i + SPT - 1
// through chunk p, so that every coefficient broadcast feeds SPT recurrences; the CTA has P * S / SPT threads.
template <typename T, int S, int KIND, int NG, bool FORCED, int SPT>
__global__ void __launch_bounds__(CHUNK_MAX_THREADS / SPT, 1)
step_chunked_kernel(const __grid_constant__ CUtensorMap tm, const StepChunkParams<T> prm)
{
    constexpr int C = ChunkCfg<T>::C, BL = chunk_block_len<T>();
    constexpr int SL = S / SPT;                  // thread columns of a tile
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

    const int i = tid % SL, p = tid / SL, sys0 = i * SPT;
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
    int slot[SPT];
#pragma unroll
    for (int u = 0; u < SPT; ++u) slot[u] = state_slot<S>(active ? p : 0, sys0 + u);
    const int row0 = p * C;
    T* cs = state + sys0;                                // element (k, sys0 + u) at cs[k*S + u]
    const int Pw = prm.Pw, G = 32 / Pw;
    const int q = lane % Pw, grp = lane / Pw;
    const ScanGeom geom{P, Pw, prm.lev_f, prm.lev_b, prm.woff};
    const int rounds = (S + nwarps * G - 1) / (nwarps * G);
    // per-lane constants of the chunk-state scan (lane q of warp `warp` scans chunk q of systems (rr nwarps + warp) G + grp).
    // The one-system-per-thread instantiations, kept for A/B, have no registers for them and use the round-1 scan.
    ScanLane lane_tab;
    int scan_slot[SPT];
    if constexpr (SPT > 1) {
        lane_tab = make_scan_lane<T>(geom, wtab, q);
#pragma unroll
        for (int rr = 0; rr < SPT; ++rr) {
            const int sys = (rr * nwarps + warp) * G + grp;
            scan_slot[rr] = (sys < S && q < P) ? state_slot<S>(q, sys) : -1;
            asm volatile("" : "+r"(scan_slot[rr]));
        }
    }
    const T r = prm.r, sigma = prm.sigma;
    constexpr bool incr = (KIND == 2);       // KIND: 0 CH direct form, 2 CH increment form, 1 hyperdiffusion, 3 periodic
    constexpr bool PER = (KIND == 3);
    static_assert(!PER || SPT == 2, "the periodic step is built on the two-systems-per-thread shape");
    const T dg_edge = (prm.bc == 1) ? (T)-1 : (T)-2;
    auto ldc = [&](T (&o)[SPT], int k) {
        if ((unsigned)k < (unsigned)N) lds_sys<T, SPT>(o, cs + (size_t)k * S);
        else {
#pragma unroll
            for (int u = 0; u < SPT; ++u) o[u] = (T)0;
        }
    };
    auto Ld = [&](int k) -> T { return (k == 0 || k == N - 1) ? dg_edge : (T)-2; };
    // Warp-uniform choice: a warp that holds one boundary chunk (several chunks per warp) takes the
    // general path with ALL its lanes instead of executing both paths one after the other; that warp
    // is the straggler every block barrier waits for.
    const bool first = row0 == 0, last = row0 + C == N;
    const T dfirst = first ? dg_edge : (T)-2, dlast = last ? dg_edge : (T)-2;
    // (lanes beyond the last chunk execute neither path: they do not vote it down)
    const bool interior = __all_sync(0xffffffffu, !active || ((first || row0 >= 2) && (last || row0 + C + 2 <= N - 1) &&
                                                              C >= 4 && N >= 2 * C));
    uint32_t parity = 0;

    for (int64_t tile = prm.tile0 + (int64_t)blockIdx.x * NG + grp_id; tile < prm.ntiles; tile += (int64_t)gridDim.x * NG) {
        if (tid == 0) {
            mbar_expect_tx(bar_state, box_bytes * prm.nbox);
            for (int b = 0; b < prm.nbox; ++b)
                tma_load_2d(state + (size_t)b * prm.box_rows * S, &tm, (int)(tile * S), b * prm.box_rows, bar_state);
        }
        mbar_wait(bar_state, parity);
        // forcing amplitudes of system tid (threads 0..S-1) at step n -> amp[n & 1][tid]
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
            double sn, cs_;
            sincospi(2.0 * fm2 * (prm.t0 + (double)n * prm.dt), &sn, &cs_);
            const double am = prm.dt * fm1;
            T2 ab; ab.x = (T)(am * cs_); ab.y = (T)(am * sn);
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
            T v[SPT][C];
            if (active) {
                // ---- explicit right-hand side of rows row0 .. row0+C-1, in registers ----
                if constexpr (KIND == 0 || KIND == 2) {
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
                        const T* cw = cs + (size_t)row0 * S;          // cw[j*S + u] = c_{row0+j} of system u
                        T cl[SPT], cc[SPT], cr[SPT], u_prev[SPT], u_cur[SPT];
                        if (first) {
#pragma unroll
                            for (int u = 0; u < SPT; ++u) { cl[u] = 0; cc[u] = 0; }
                        } else {
                            lds_sys<T, SPT>(cl, cw - 2 * S);
                            lds_sys<T, SPT>(cc, cw - S);
                        }
                        lds_sys<T, SPT>(cr, cw);
#pragma unroll
                        for (int u = 0; u < SPT; ++u) {
                            u_prev[u] = first ? (T)0 : U(cl[u], cc[u], cr[u], (T)-2);        // u_{row0-1}
                            cl[u] = cc[u]; cc[u] = cr[u];
                        }
                        lds_sys<T, SPT>(cr, cw + S);
#pragma unroll
                        for (int u = 0; u < SPT; ++u) u_cur[u] = U(cl[u], cc[u], cr[u], dfirst);  // u_{row0}
#pragma unroll
                        for (int j = 0; j < C; ++j) {
#pragma unroll
                            for (int u = 0; u < SPT; ++u) { cl[u] = cc[u]; cc[u] = cr[u]; }    // cl = c_{row0+j}, cc = c_{row0+j+1}
                            if (j + 2 < C || !last) lds_sys<T, SPT>(cr, cw + (size_t)(j + 2) * S);
                            else {
#pragma unroll
                                for (int u = 0; u < SPT; ++u) cr[u] = (T)0;                    // rows N, N+1 do not exist
                            }
#pragma unroll
                            for (int u = 0; u < SPT; ++u) {
                                T u_next = U(cl[u], cc[u], cr[u], (j + 1 == C - 1) ? dlast : (T)-2);   // u_{row0+j+1}
                                if (j == C - 1 && last) u_next = 0;                                    // u_N
                                T Lu = u_prev[u] + fma(j == 0 ? dfirst : (j == C - 1 ? dlast : (T)-2), u_cur[u], u_next);
                                v[u][j] = incr ? Lu : fma(r, Lu, cl[u]);
                                u_prev[u] = u_cur[u]; u_cur[u] = u_next;
                            }
                        }
                    } else {
                        auto U = [&](int k, T cl, T cc, T cr) -> T {
                            if ((unsigned)k >= (unsigned)N) return (T)0;
                            T w = cc * cc * cc - cc;
                            if (!incr) return w;
                            return fma(-sigma, cl + fma(Ld(k), cc, cr), r * w);
                        };
                        T cl[SPT], cc[SPT], cr[SPT], u_prev[SPT], u_cur[SPT];
                        ldc(cl, row0 - 2); ldc(cc, row0 - 1); ldc(cr, row0);
#pragma unroll
                        for (int u = 0; u < SPT; ++u) {
                            u_prev[u] = U(row0 - 1, cl[u], cc[u], cr[u]);
                            cl[u] = cc[u]; cc[u] = cr[u];
                        }
                        ldc(cr, row0 + 1);
#pragma unroll
                        for (int u = 0; u < SPT; ++u) u_cur[u] = U(row0, cl[u], cc[u], cr[u]);
#pragma unroll
                        for (int j = 0; j < C; ++j) {
                            const int k = row0 + j;
#pragma unroll
                            for (int u = 0; u < SPT; ++u) { cl[u] = cc[u]; cc[u] = cr[u]; }    // window centred on k+1; cl = c_k
                            ldc(cr, k + 2);
#pragma unroll
                            for (int u = 0; u < SPT; ++u) {
                                T u_next = U(k + 1, cl[u], cc[u], cr[u]);
                                T Lu = u_prev[u] + fma(Ld(k), u_cur[u], u_next);
                                v[u][j] = incr ? Lu : fma(r, Lu, cl[u]);
                                u_prev[u] = u_cur[u]; u_cur[u] = u_next;
                            }
                        }
                    }
                } else {
                    // Crank-Nicolson hyperdiffusion, A c+ = (2I - A) c (Eq. 6 / 7c), evaluated as  c+ = 2 A^{-1} c - c
                    // (A^{-1} (2I - A) = 2 A^{-1} - I): the right-hand side of the solve is the state itself -- no stencil,
                    // no halo rows, none of the matrix's diagonals (which would have to come from L2: shared memory is
                    // full) -- and the write-back below forms 2 y - c.  Same scheme, another order of evaluation.
                    const T* cw = cs + (size_t)row0 * S;
                    if (row0 + C <= N) {
#pragma unroll
                        for (int j = 0; j < C; ++j) {
                            T cj[SPT];
                            lds_sys<T, SPT>(cj, cw + (size_t)j * S);
#pragma unroll
                            for (int u = 0; u < SPT; ++u) v[u][j] = cj[u];
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < C; ++j) {
                            T cj[SPT];
                            ldc(cj, row0 + j);
#pragma unroll
                            for (int u = 0; u < SPT; ++u) v[u][j] = cj[u];
                        }
                    }
                }
                if constexpr (FORCED) {
#pragma unroll
                    for (int u = 0; u < SPT; ++u) {
                        const T2 ab = amp[(step & 1) * S + sys0 + u];
                        T ph = fma(ab.x, fcx, ab.y * fsx), dph = fma(ab.x, fdcx, ab.y * fdsx);
                        if (row0 + C <= N) {
#pragma unroll
                            for (int j = 0; j < C; ++j) { v[u][j] += ph; ph += dph; dph = fma(-fkap, ph, dph); }
                        } else {
#pragma unroll
                            for (int j = 0; j < C; ++j) {
                                if (row0 + j < N) v[u][j] += ph;
                                ph += dph;
                                dph = fma(-fkap, ph, dph);
                            }
                        }
                    }
                }
                // ---- chunked solve, stages 1+2 ----  (periodic: of the block E; its rows N-2, N-1 have zero coefficients)
                T2 e[SPT], s[SPT];
                chunk_local_sweeps_n<T, SPT>(v, blk, e, s);
#pragma unroll
                for (int u = 0; u < SPT; ++u) { stE[slot[u]] = e[u]; stS[slot[u]] = s[u]; }
            }
            group_sync<NG>(grp_id, TG);
            if constexpr (FORCED) {
                if (tid < S && step + 1 < prm.nsteps) amp_for_step(step + 1);   // read after two more barriers
            }
            if (P > 1) {
                if (SPT > 1 && rounds == SPT) {   // (P a power of two) every scan lane carries SPT systems at once
                    chunk_state_scan_lean<T, SPT>(lane_tab, prm.so, P, Pw, prm.lev_f, prm.lev_b, q, stE, stS, scan_slot);
                } else {
                    for (int rr = 0; rr < rounds; ++rr) {
                        const int sys = (rr * nwarps + warp) * G + grp;
                        chunk_state_scan<T, S, false>(geom, wtab, stE, stS, sys, q, (sys < S) && (q < P), 0, 1,
                                                      nullptr, nullptr, bars, 0u, 0u, 0u);
                    }
                }
            }
            group_sync<NG>(grp_id, TG);
            T F0[SPT], F1[SPT], B0[SPT], B1[SPT];
            if (active) {
#pragma unroll
                for (int u = 0; u < SPT; ++u) {
                    F0[u] = 0; F1[u] = 0; B0[u] = 0; B1[u] = 0;
                    if (P > 1) { T2 fo = stE[slot[u]]; F0[u] = fo.x; F1[u] = fo.y; T2 bo = stS[slot[u]]; B0[u] = bo.x; B1[u] = bo.y; }
                }
                if constexpr (PER) {
                    // the first chunk publishes (y_0, y_1), the last one (y_{n-2}, y_{n-1}) (its rows C-4, C-3), each into
                    // its OWN stE slot (already read above; nobody else reads it before the barrier below)
                    if (first || last) {
                        const T* cr = blk + 5 * C + 4 * (first ? 0 : C - 4);
#pragma unroll
                        for (int u = 0; u < SPT; ++u) {
                            const T xa = first ? v[u][0] : v[u][C - 4], xb = first ? v[u][1] : v[u][C - 3];
                            T2 y;
                            y.x = fma(cr[3], B1[u], fma(cr[2], B0[u], fma(cr[1], F1[u], fma(cr[0], F0[u], xa))));
                            y.y = fma(cr[7], B1[u], fma(cr[6], B0[u], fma(cr[5], F1[u], fma(cr[4], F0[u], xb))));
                            stE[slot[u]] = y;
                        }
                        if (last) {   // ... and the right-hand side of the two tail rows, (c_{N-2}, c_{N-1}), into its stS slot
                            T fa[SPT], fb[SPT];
                            lds_sys<T, SPT>(fa, cs + (size_t)(N - 2) * S);
                            lds_sys<T, SPT>(fb, cs + (size_t)(N - 1) * S);
#pragma unroll
                            for (int u = 0; u < SPT; ++u) { T2 ft; ft.x = fa[u]; ft.y = fb[u]; stS[slot[u]] = ft; }
                        }
                    }
                }
            }
            T t0[SPT], t1[SPT];
            if constexpr (PER) {
                group_sync<NG>(grp_id, TG);
                if (active) {
                    // t = S2^{-1} [ (f_{N-2}, f_{N-1}) - h^T y ]  (Eq. 12), redundantly by every thread of the system, then
                    // Z folded into the chunk states: F - F^Z t, B - B^Z t
                    T fz[8];
#pragma unroll
                    for (int w = 0; w < 8; ++w) fz[w] = __ldg(prm.pfold + 8 * (size_t)p + w);
#pragma unroll
                    for (int u = 0; u < SPT; ++u) {
                        const T2 y0 = stE[state_slot<S>(0, sys0 + u)], yl = stE[state_slot<S>(P - 1, sys0 + u)];
                        const T2 ft = stS[state_slot<S>(P - 1, sys0 + u)];
                        const T r0 = ft.x - fma(prm.ph[2], yl.y, fma(prm.ph[1], yl.x, prm.ph[0] * y0.x));
                        const T r1 = ft.y - fma(prm.ph[5], yl.y, fma(prm.ph[4], y0.y, prm.ph[3] * y0.x));
                        t0[u] = fma(prm.pi[1], r1, prm.pi[0] * r0);
                        t1[u] = fma(prm.pi[3], r1, prm.pi[2] * r0);
                        F0[u] = fma(-fz[1], t1[u], fma(-fz[0], t0[u], F0[u]));
                        F1[u] = fma(-fz[3], t1[u], fma(-fz[2], t0[u], F1[u]));
                        B0[u] = fma(-fz[5], t1[u], fma(-fz[4], t0[u], B0[u]));
                        B1[u] = fma(-fz[7], t1[u], fma(-fz[6], t0[u], B1[u]));
                    }
                }
            }
            if (active) {
                T* co = cs + (size_t)row0 * S;
#pragma unroll
                for (int jg = 0; jg < C / 4; ++jg) {
                    T xv[SPT][4];
                    chunk_correct4_n<T, SPT>(xv, v, blk, jg, F0, F1, B0, B1);
                    if constexpr (PER) {
                        if (first || last) {        // the chunks that hold the non-zero rows of k: explicit rows of Z
#pragma unroll
                            for (int rr = 0; rr < 4; ++rr) {
                                const typename Vec<T>::T2 z = __ldg(prm.pzedge + (first ? 0 : C) + 4 * jg + rr);
#pragma unroll
                                for (int u = 0; u < SPT; ++u) xv[u][rr] = fma(-z.y, t1[u], fma(-z.x, t0[u], xv[u][rr]));
                            }
                        }
                    }
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr) {
                        T* o = co + (size_t)(4 * jg + rr) * S;
                        T nv[SPT];
                        if constexpr (PER) {
                            if (last && 4 * jg + rr >= C - 2) {      // rows N-2, N-1 of the solution are t (Eq. 12)
#pragma unroll
                                for (int u = 0; u < SPT; ++u) xv[u][rr] = (4 * jg + rr == C - 2) ? t0[u] : t1[u];
                            }
                        }
                        if (incr) {
                            lds_sys<T, SPT>(nv, o);
#pragma unroll
                            for (int u = 0; u < SPT; ++u) nv[u] += xv[u][rr];
                        } else if (KIND == 1 || KIND == 3) {
                            lds_sys<T, SPT>(nv, o);
#pragma unroll
                            for (int u = 0; u < SPT; ++u) nv[u] = fma((T)2, xv[u][rr], -nv[u]);
                        } else {
#pragma unroll
                            for (int u = 0; u < SPT; ++u) nv[u] = xv[u][rr];
                        }
                        sts_sys<T, SPT>(o, nv);
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

// Shape of a step launch: NG groups of TG threads, each with a tile of S systems, SPT systems per thread.
struct StepPlan {
    bool ok = false;
    ChunkPlan pl;
    int S = 0, NG = 1, TG = 0, SPT = 1;
    size_t smem = 0;
};

static StepPlan step_plan(const pent_handle* h, int64_t M, const void* c, int S, int NG, int SPT)
{
    StepPlan sp;
    if (!h || h->kind != 0 || h->periodic) return sp;
    const size_t esz = h->dtype == PENT_F64 ? 8 : 4;
    sp.pl = make_plan(h, M, c, 1, S, /*any_S=*/true);
    if (!sp.pl.ok || S % SPT != 0) return sp;
    sp.S = S; sp.NG = NG; sp.SPT = SPT;
    sp.TG = (sp.pl.Pl * S / SPT + 31) / 32 * 32;
    if (sp.TG * NG > CHUNK_MAX_THREADS / SPT) return sp;
    sp.smem = (size_t)NG * ((size_t)sp.pl.nbox * sp.pl.box_rows * S * esz + (size_t)4 * sp.pl.Pl * S * esz) +
              sp.pl.table_bytes + (size_t)(1 + NG) * sizeof(uint64_t) +
              (size_t)NG * 4 * S * esz;                                    // forcing amplitudes (used when FORCED)
    sp.ok = sp.smem <= SMEM_LIMIT;
    return sp;
}

// Default shapes, measured on cfg4 (1000 steps, profiles/r02_step_spt.md).  Two systems per thread halve the
// coefficient broadcasts per unknown, which is what bounds this kernel (shared-memory wavefronts).
// PENT_AB_STEP_SPT=1 (environment, measurement only) selects the one-system-per-thread shapes of round 1.
// Two thread groups of half-width tiles (S = 8 fp64 / 16 fp32, SPT = 2) measured slower: 26.7 against 22.9 us per
// step (fp32 13.4 against 11.5): a warp then spans 8 chunks and its coefficient loads are no longer broadcasts.
static StepPlan step_auto_plan(const pent_handle* h, int64_t M, const void* c)
{
    if (!h || !chunk_stitching_stable(h)) return StepPlan{};
    static const int spt = []() { const char* e = std::getenv("PENT_AB_STEP_SPT"); return e ? std::atoi(e) : 2; }();
    if (h->dtype == PENT_F64) {
        if (spt != 1) { StepPlan two = step_plan(h, M, c, 16, 1, 2); if (two.ok) return two; }
        return step_plan(h, M, c, 16, 1, 1);
    }
    if (spt != 1) { StepPlan w = step_plan(h, M, c, 32, 1, 2); if (w.ok) return w; }
    StepPlan two = step_plan(h, M, c, 16, 2, 1);
    if (two.ok) return two;
    return step_plan(h, M, c, 32, 1, 1);
}

// Systems [sys_lo, sys_hi) of the batch (sys_lo a multiple of S) in tiles of S.  KIND 3: hp = the periodic handle, h = its
// inner handle (the block E, whose tables the solve stages read); otherwise hp == h.
template <typename T, int S, int KIND, int NG, bool FORCED, int SPT>
static int launch_step_inst(const pent_handle* h, const StepPlan& sp, const pent_step_params* p, const pent_forcing* fg,
                            int64_t M, void* c, int nsteps, cudaStream_t s, int64_t sys_lo, int64_t sys_hi,
                            const pent_handle* hp = nullptr)
{
    if (!hp) hp = h;
    const ChunkPlan& pl = sp.pl;
    StepChunkParams<T> prm;
    prm.N = hp->N; prm.P = pl.Pl; prm.Pw = pl.Pw; prm.M = M;
    int lg = 0;
    while ((1 << lg) < pl.Pw) ++lg;
    prm.lev_f = h->lev_f[0] < lg ? h->lev_f[0] : lg;
    prm.lev_b = h->lev_b[0] < lg ? h->lev_b[0] : lg;
    for (int l = 0; l < W_LEVELS; ++l) prm.woff[l] = w_level_off(pl.Pl, l, 1);
    prm.so = make_scan_offsets<T>(pl.Pl, prm.woff);
    prm.box_rows = pl.box_rows; prm.nbox = pl.nbox;
    prm.tile0 = sys_lo / S;
    prm.ntiles = (sys_hi + S - 1) / S;
    prm.table = (const T*)h->cf[0];
    prm.table_bytes = (uint32_t)pl.table_bytes;
    prm.dg = (const T*)(KIND == 3 ? hp->dgp : h->dg);
    prm.nsteps = nsteps; prm.bc = p->bc;
    prm.r = (T)p->r; prm.sigma = (T)p->sigma;
    prm.pfold = nullptr; prm.pzedge = nullptr;
    for (int w = 0; w < 6; ++w) prm.ph[w] = (T)0;
    for (int w = 0; w < 4; ++w) prm.pi[w] = (T)0;
    if (KIND == 3) {
        prm.pfold = (const T*)hp->pfold; prm.pzedge = (const typename Vec<T>::T2*)hp->pzedge;
        for (int w = 0; w < 6; ++w) prm.ph[w] = (T)hp->pc[w];
        for (int w = 0; w < 4; ++w) prm.pi[w] = (T)hp->pc[6 + w];
    }
    prm.mu1 = prm.mu2 = nullptr; prm.dt = prm.t0 = 0.0;
    if (FORCED) { prm.mu1 = (const T*)fg->mu1; prm.mu2 = (const T*)fg->mu2; prm.dt = fg->dt; prm.t0 = fg->t0; }
    CUtensorMap tm;
    if (!encode_batch_map_cached(&tm, c, M, hp->N, S, prm.box_rows, sizeof(T) == 8)) {
        g_last_cuda_error = (int)cudaErrorInvalidValue;
        return PENT_ERR_CUDA;
    }
    auto kern = step_chunked_kernel<T, S, KIND, NG, FORCED, SPT>;
    static SmemOnce mark;
    PENT_CUDA(ensure_dynamic_smem(mark, kern, sp.smem));
    const int threads = sp.TG * NG;
    int dev = 0, nsm = 0, occ = 0;
    PENT_CUDA(cudaGetDevice(&dev));
    PENT_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    PENT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, sp.smem));
    if (occ < 1) return PENT_ERR_ARG;
    int64_t grid = (int64_t)nsm * occ;
    const int64_t need = (prm.ntiles - prm.tile0 + NG - 1) / NG;
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

template <typename T, int S, int NG, int SPT>
static int launch_step_kind(const pent_handle* h, const StepPlan& sp, const pent_step_params* p, const pent_forcing* fg,
                            int64_t M, void* c, int nsteps, cudaStream_t s, int64_t lo, int64_t hi)
{
    if (p->kind == 1) return launch_step_inst<T, S, 1, NG, false, SPT>(h, sp, p, nullptr, M, c, nsteps, s, lo, hi);
    if (fg) {
        if (p->form == 1) return launch_step_inst<T, S, 2, NG, true, SPT>(h, sp, p, fg, M, c, nsteps, s, lo, hi);
        return launch_step_inst<T, S, 0, NG, true, SPT>(h, sp, p, fg, M, c, nsteps, s, lo, hi);
    }
    if (p->form == 1) return launch_step_inst<T, S, 2, NG, false, SPT>(h, sp, p, nullptr, M, c, nsteps, s, lo, hi);
    return launch_step_inst<T, S, 0, NG, false, SPT>(h, sp, p, nullptr, M, c, nsteps, s, lo, hi);
}

// The tiles of a launch run in rounds of one tile per SM.  When the last round would fill at most half of the SMs,
// its systems go to a SECOND launch in tiles of half the width instead (twice the CTAs, each about half the time of a
// full tile): cfg4's 512 tiles of 16 systems are 3 full rounds on 148 SMs plus 68 tiles, i.e. 4 rounds; as 444 tiles
// of 16 and 136 tiles of 8 they are 3 rounds plus one short one.  The tile width does not enter the arithmetic of a
// system, so the result does not depend on the split.
int launch_step_chunked(const pent_handle* h, const pent_step_params* p, const pent_forcing* fg, int64_t M, void* c,
                        int nsteps, cudaStream_t s)
{
    const StepPlan sp = step_auto_plan(h, M, c);
    if (!sp.ok) return PENT_ERR_ARG;
    int64_t split = M;                       // systems [0, split) in full tiles, [split, M) in half-width tiles
    StepPlan half;
    if (sp.SPT == 2 && sp.NG == 1) {
        static const int no_split = []() { const char* e = std::getenv("PENT_AB_STEP_NOSPLIT"); return e ? std::atoi(e) : 0; }();
        int dev = 0, nsm = 0;
        PENT_CUDA(cudaGetDevice(&dev));
        PENT_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        const int64_t ntiles = (M + sp.S - 1) / sp.S, rem = ntiles % nsm;
        if (!no_split && ntiles > nsm && rem > 0 && 2 * rem <= nsm) {
            half = step_plan(h, M, c, sp.S / 2, 1, 2);
            if (half.ok) split = (ntiles - rem) * sp.S;
        }
    }
    int rc = PENT_OK;
    if (h->dtype == PENT_F64) {
        if (sp.SPT == 2) {
            rc = launch_step_kind<double, 16, 1, 2>(h, sp, p, fg, M, c, nsteps, s, 0, split);
            if (rc == PENT_OK && split < M) rc = launch_step_kind<double, 8, 1, 2>(h, half, p, fg, M, c, nsteps, s, split, M);
            return rc;
        }
        return launch_step_kind<double, 16, 1, 1>(h, sp, p, fg, M, c, nsteps, s, 0, M);
    }
    if (sp.SPT == 2) {
        rc = launch_step_kind<float, 32, 1, 2>(h, sp, p, fg, M, c, nsteps, s, 0, split);
        if (rc == PENT_OK && split < M) rc = launch_step_kind<float, 16, 1, 2>(h, half, p, fg, M, c, nsteps, s, split, M);
        return rc;
    }
    if (sp.NG == 2) return launch_step_kind<float, 16, 2, 1>(h, sp, p, fg, M, c, nsteps, s, 0, M);
    return launch_step_kind<float, 32, 1, 1>(h, sp, p, fg, M, c, nsteps, s, 0, M);
}

// ---- periodic handles: the paper's own loop with the state on chip, KIND 3 ----------------------------
// The tile holds all N rows of the state; the solve stages run on the tables of the inner handle (the (N-2) x (N-2)
// block E), whose last chunk ends with the two tail rows (zero coefficients).
static StepPlan step_periodic_plan(const pent_handle* h, int64_t M, const void* c, int S)
{
    StepPlan sp;
    if (!h || !h->periodic || !h->inner || !h->pfold || !h->pzedge) return sp;
    const pent_handle* hi = h->inner;
    const int C = h->dtype == PENT_F64 ? ChunkCfg<double>::C : ChunkCfg<float>::C;
    if (h->N % C != 0 || h->N < 2 * C || hi->cfP[0] != h->N / C || !chunk_stitching_stable(hi)) return sp;
    sp = step_plan(hi, M, c, S, 1, 2);     // rows per tile = Pl * C = N: the two tail rows are part of the boxes
    return sp;
}

bool step_chunked_periodic_supported(const pent_handle* h, int64_t M, const void* c)
{
    return step_periodic_plan(h, M, c, h && h->dtype == PENT_F64 ? 16 : 32).ok;
}

int launch_step_chunked_periodic(const pent_handle* h, int64_t M, void* c, int nsteps, cudaStream_t s)
{
    const int Sf = h->dtype == PENT_F64 ? 16 : 32;
    const StepPlan sp = step_periodic_plan(h, M, c, Sf);
    if (!sp.ok) return PENT_ERR_ARG;
    pent_step_params p = {};
    p.kind = 1;
    int64_t split = M;                       // leftover round in half-width tiles, as in launch_step_chunked
    StepPlan half;
    int dev = 0, nsm = 0;
    PENT_CUDA(cudaGetDevice(&dev));
    PENT_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    const int64_t ntiles = (M + sp.S - 1) / sp.S, rem = ntiles % nsm;
    if (ntiles > nsm && rem > 0 && 2 * rem <= nsm) {
        half = step_periodic_plan(h, M, c, Sf / 2);
        if (half.ok) split = (ntiles - rem) * sp.S;
    }
    int rc;
    if (h->dtype == PENT_F64) {
        rc = launch_step_inst<double, 16, 3, 1, false, 2>(h->inner, sp, &p, nullptr, M, c, nsteps, s, 0, split, h);
        if (rc == PENT_OK && split < M) rc = launch_step_inst<double, 8, 3, 1, false, 2>(h->inner, half, &p, nullptr, M, c, nsteps, s, split, M, h);
        return rc;
    }
    rc = launch_step_inst<float, 32, 3, 1, false, 2>(h->inner, sp, &p, nullptr, M, c, nsteps, s, 0, split, h);
    if (rc == PENT_OK && split < M) rc = launch_step_inst<float, 16, 3, 1, false, 2>(h->inner, half, &p, nullptr, M, c, nsteps, s, split, M, h);
    return rc;
}
}  // namespace pent
