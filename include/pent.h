/* pent.h -- C ABI of the B200 (sm_100a) batched pentadiagonal solver.
 *
 * The library solves A x_i = f_i, i = 0..M-1, for an N x N pentadiagonal A by the extended
 * Thomas algorithm of arXiv 1807.07382 ("cuPentBatch"): factor A = L R once
 * (section II.D steps 1-14), then per system a forward sweep L g = f
 * and a back substitution R x = g.  No pivoting is
 * ever attempted (valid for SPD or diagonally dominant A).
 *
 * LAYOUT ("interleaved"): a batch is ONE array of N*M elements in which
 * element k of system i is at index k*M + i.  Consecutive systems are consecutive in memory.
 *
 * DIAGONALS: five arrays indexed by ROW k = 0..N-1,
 *     a[k] = A[k][k-2], b[k] = A[k][k-1], c[k] = A[k][k], d[k] = A[k][k+1], e[k] = A[k][k+2].
 * a[0], a[1], b[0], d[N-1], e[N-2], e[N-1] lie outside the matrix and are NEVER READ.
 * The positional order (N, e, c, d, a, b) is the one BASELINE.json's north_star writes.
 *
 * POINTERS: "device" = CUDA device memory of the current device; "host" = ordinary host
 * memory; "host or device" = either (detected with cudaPointerGetAttributes).  The element
 * type of every data pointer is `double` for PENT_F64 and `float` for PENT_F32.
 * `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *
 * OWNERSHIP: the caller owns every array it passes; a handle owns device copies of whatever
 * it needs and never keeps a caller pointer.  Handles are immutable after creation and may
 * be used from several streams/threads at once.  No hidden global state (per-thread caches of
 * encoded tensor maps, occupancy answers and the staging buffers of pent_solve_batch_host hold no
 * results; pent_release_thread_cache frees the latter).
 *
 * DEVICE: a handle belongs to the CUDA device that was current when it was created; every call
 * that takes a handle returns PENT_ERR_ARG if another device is current.
 *
 * ASYNCHRONY: every *_batch call only enqueues work on `stream` and returns; it never
 * synchronises the host (pent_factor_batch included: `info` is device memory).
 * pent_factor / pent_factor_periodic run on a PRIVATE non-blocking stream and wait for that stream
 * only: they return with the handle complete, and they neither wait for nor stall any other
 * stream of the process (device-pointer diagonals must therefore be complete before the call).
 * pent_solve_batch_host returns when x_host is complete.  pent_destroy synchronises the device
 * (cudaFree): do not call it while work that uses the handle is in flight.
 *
 * ERRORS: every int function returns one of the codes below; nothing is printed, nothing
 * throws, and there is NO CPU fallback.
 */
#ifndef PENT_H_
#define PENT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pent_handle pent_handle;   /* opaque */

typedef enum { PENT_F64 = 0, PENT_F32 = 1 } pent_dtype;

enum {
    PENT_OK = 0,
    PENT_ERR_ARG = 1,      /* null pointer, N < 1, M < 0, bad dtype / params, handle of the wrong kind */
    PENT_ERR_PIVOT = 2,    /* zero or non-finite pivot alpha_k (shared-A factor only)                   */
    PENT_ERR_CUDA = 3,     /* a CUDA call failed; pent_last_cuda_error() holds its cudaError_t          */
    PENT_ERR_ALLOC = 4,    /* host or device allocation failed                                          */
    PENT_ERR_TOO_LARGE = 5 /* pent_factor_solve_batch_noalloc: the problem needs more scratch than the static
                              array holds (pent_noalloc_scratch_bytes)                                  */
};

/* Kernel choice for pent_solve_batch_v (measurement / tests).  AUTO is what pent_solve_batch uses. */
enum {
    PENT_KERNEL_AUTO = 0,
    PENT_KERNEL_THREAD_PER_SYSTEM = 1,  /* the paper's design: one thread per system,
                                           g round-trips through x in global memory (4 passes)         */
    PENT_KERNEL_CHUNKED = 2             /* k split into chunks across threads, g kept in registers,
                                           chunk coupling by the shared correction vectors (2 passes)  */
};
/* PENT_KERNEL_CHUNKED with an explicit shape (measurement): Q = CTAs of a thread-block cluster that
 * split k between them (1, 2, 4, 8, 16 -- 16 is CUDA's non-portable cluster size --; 0 = choose), S = systems per tile (16, 32 for fp64; 32, 64 for
 * fp32; 0 = choose).  PENT_ERR_ARG if that shape does not fit N / M / shared memory. */
#define PENT_KERNEL_CHUNKED_CFG(Q, S) (2 | ((Q) << 8) | ((S) << 16))

/* ---- shared A: factor once, solve many ("cuPentBatchConstant") -----------------
 * pent_factor: e,c,d,a,b: N elements each, host or device, element type per `dtype`.
 *   The factorisation itself runs in a device kernel in fp64 whatever the
 *   dtype (fp32 inputs are widened exactly; the fp32 solve kernel reads rounded factors).
 *   *out receives the handle.  If bad_row != NULL it receives -1, or the first 0-based row whose
 *   pivot is zero / non-finite when PENT_ERR_PIVOT is returned (no handle is created then). */
int pent_factor(int N, const void* e, const void* c, const void* d, const void* a, const void* b,
                pent_dtype dtype, pent_handle** out, int* bad_row);

/* pent_solve_batch: f, x: device, N*M elements, interleaved.  x == f (in place) is allowed;
 *   any other overlap is undefined.  M == 0 is a no-op.  Forward + backward sweeps
 *    for all M systems in one launch on `stream`. */
int pent_solve_batch(const pent_handle* h, int64_t M, const void* f, void* x, void* stream);
int pent_solve_batch_v(const pent_handle* h, int64_t M, const void* f, void* x, void* stream,
                       int kernel);

/* Same operation on a SYSTEM-MAJOR batch: f, x: device, M*N elements, element k of system i at i*N + k
 * ("one system per row", the layout of the paper's serial code; it is also what an ADI
 * sweep along the contiguous axis of a 2-D field needs: the sweep along the other axis is
 * pent_solve_batch itself).  x == f allowed.  Shared-A, non-periodic handles with N <= 16384;
 * PENT_ERR_ARG otherwise.  2 passes over the batch, no transpose: a system's run of rows moves global <-> shared memory
 * by 1-D bulk copies when N * sizeof(element) and the base addresses are 16-byte aligned; otherwise every thread reads and
 * writes its contiguous run of 32 (fp64) / 64 (fp32) elements itself, with 32-byte accesses when the run is 32-byte aligned
 * and element-wise accesses when it is not. */
int pent_solve_batch_rows(const pent_handle* h, int64_t M, const void* f, void* x, void* stream);
/* Same with an explicit shape / data path (measurement): kernel = PENT_KERNEL_AUTO or PENT_KERNEL_CHUNKED_CFG(Q, S),
 * optionally OR-ed with one of the flags below.  Default: one 1-D bulk copy (cp.async.bulk) per system and tile in
 * each direction, through padded shared-memory buffers; when the staging buffer does not fit, bulk loads with 32-byte
 * STG stores; when N * sizeof(element) or a base address is not 16-byte aligned, the per-thread LDG loader. */
#define PENT_ROWS_LDG   (1 << 24)   /* per-thread 32-byte LDG / STG accesses */
#define PENT_ROWS_STG   (1 << 25)   /* bulk loads, 32-byte STG stores */
#define PENT_ROWS_TMA2D (1 << 26)   /* swizzled tensor-tile TMA loads (128-byte rows), 32-byte STG stores (A/B baseline) */
int pent_solve_batch_rows_v(const pent_handle* h, int64_t M, const void* f, void* x, void* stream, int kernel);
/* What pent_solve_batch_rows runs for M systems: PENT_KERNEL_CHUNKED_CFG(Q, S) | (data path << 24), data path 6 = bulk
 * copies both ways, 5 = bulk loads + STG stores, 3 = swizzled TMA loads, 2 = per-thread LDG / STG; -1 if unsupported. */
int pent_solve_rows_kernel_choice(const pent_handle* h, int64_t M);

/* Same operation with HOST buffers (pageable or pinned): copies slabs of systems to the device,
 * solves, copies back, pipelined on internal streams; returns when x_host is complete.
 * M * sizeof(element) must be below 2^31 bytes (the pitch limit of the 2-D copies), else PENT_ERR_ARG.
 * The staging buffers (4 x 16 MiB of device memory, 4 streams) are cached per calling thread until
 * the thread exits or calls pent_release_thread_cache(). */
int pent_solve_batch_host(const pent_handle* h, int64_t M, const void* f_host, void* x_host);
void pent_release_thread_cache(void);

void pent_destroy(pent_handle* h);          /* NULL is allowed */

/* ---- periodic (cyclic) shared A: the matrix of the paper's own benchmark ------
 * a[k] = A[k][(k-2) mod N], b[k] = A[k][(k-1) mod N], c[k] = A[k][k], d[k] = A[k][(k+1) mod N],
 * e[k] = A[k][(k+2) mod N]: ALL N entries of every array are read (Eq. 7a with row-indexed
 * entries).  N >= 6.  Set-up = the reduction of Eqs. 8-12: factor the (N-2) x (N-2) block E,
 * E^{-1} k and the inverted 2 x 2 Schur complement are computed once and kept in the handle.
 * The handle is used with pent_solve_batch / _v / _host (f, x: N*M elements, interleaved) and with
 * pent_step_batch (kind 1 only: A c+ = (2I - A) c with the cyclic A, Eq. 6 / 7c = the paper's own time loop,
 * PAPER.md:281; ONE launch for all nsteps with the state on chip when N is a multiple of 32 (fp64) / 64 (fp32) and the
 * tile fits, evaluated as c+ = 2 A^{-1} c - c; otherwise a right-hand-side kernel and a fused periodic solve per step with
 * `scratch` = N*M elements or NULL).  PENT_ERR_PIVOT: *bad_row = failing row of E, or N-2 if the 2 x 2 Schur
 * complement is singular. */
int pent_factor_periodic(int N, const void* e, const void* c, const void* d, const void* a, const void* b,
                         pent_dtype dtype, pent_handle** out, int* bad_row);
/* pent_solve_batch on a periodic handle runs ONE fused kernel (solve of E, 2 x 2 tail, rank-2 update:
 * 2 passes over the batch) when the shape allows it, else three kernels (4 passes).
 * pent_periodic_fused: 1 / 0 = which of the two PENT_KERNEL_AUTO runs for M systems; -1 = not periodic.
 * pent_solve_batch_v(kernel = PENT_KERNEL_CHUNKED or PENT_KERNEL_THREAD_PER_SYSTEM) forces the
 * three-kernel path with that inner solve kernel. */
int pent_periodic_fused(const pent_handle* h, int64_t M);
int pent_handle_periodic(const pent_handle* h);          /* 1 for a periodic handle, 0 otherwise, -1 for NULL */

/* ---- per-system matrices ("cuPentBatchRewrite") ---------------------------------
 * e,c,d,a,b,f,x: device, N*M elements each, interleaved like f (diagonal entry k of system i at
 * k*M+i).  x == f (in place) is allowed; any other overlap is undefined.  info: device int[M] or NULL; info[i] = 0, or (first bad row + 1) if system i met a
 * zero / non-finite pivot (its x is then unspecified; other systems are unaffected).
 * pent_factor_solve_batch factors and solves in ONE kernel and keeps nothing.  For N >= 8 it cuts every system in the
 * middle and gives each half a thread (top-down LU of the leading block, the same recurrence bottom-up on the reversed
 * trailing block, a 4 x 4 interface system): x_i = A_i^{-1} f_i by a twisted factorisation without pivoting, which differs
 * from the paper's LU by rounding only; info[i] is then the first bad pivot of the top-down half, else of the bottom-up half.
 * pent_factor_batch keeps the M factorisations in the handle (5*N*M elements of device memory)
 * for repeated pent_solve_batch_multi calls (M is fixed by the handle). */
int pent_factor_solve_batch(int N, int64_t M, const void* e, const void* c, const void* d,
                            const void* a, const void* b, const void* f, void* x,
                            pent_dtype dtype, int* info, void* stream);
/* Same with a caller-owned workspace: device, 3*N*M' elements, M' = M rounded up to a multiple of 64
 * (gamma_k, delta_k, g_k of every system, in a block-contiguous layout),
 * or NULL (the library then allocates and frees a stream-ordered temporary on every call). */
int pent_factor_solve_batch_ws(int N, int64_t M, const void* e, const void* c, const void* d,
                               const void* a, const void* b, const void* f, void* x,
                               pent_dtype dtype, int* info, void* workspace, void* stream);
/* Same operation for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the scratch is a static device array inside the library, so the call makes NO cudaMalloc, cudaFree or
 * stream-ordered allocation.  Limit: 3 * N * M' * sizeof(element) <= pent_noalloc_scratch_bytes() = 32 MiB, M' = M rounded
 * up to a multiple of 64 (e.g. N = 1024: M <= 1344 fp64, 2688 fp32); beyond it PENT_ERR_TOO_LARGE and nothing is launched.
 * Every GPU that loads the library holds those 32 MiB until the process exits.  All calls share the array: calls that
 * overlap on the GPU (different streams, concurrent graph branches) RACE on it; calls ordered on one stream are safe and
 * nothing needs clearing between them.  The first call on a device looks the array's address up (cudaGetSymbolAddress)
 * and sets a function attribute: make one call before starting a graph capture.  Arguments as pent_factor_solve_batch. */
int pent_factor_solve_batch_noalloc(int N, int64_t M, const void* e, const void* c, const void* d,
                                    const void* a, const void* b, const void* f, void* x,
                                    pent_dtype dtype, int* info, void* stream);
int64_t pent_noalloc_scratch_bytes(void);
int pent_factor_batch(int N, int64_t M, const void* e, const void* c, const void* d,
                      const void* a, const void* b, pent_dtype dtype, pent_handle** out,
                      int* info, void* stream);
int pent_solve_batch_multi(const pent_handle* h, const void* f, void* x, void* stream);

/* ---- fused time stepping on a shared-A handle (BASELINE.json configs[3]) ----------------------
 * One step = explicit right-hand side built from the state + one solve, fused in one kernel.
 * Default (N*S*sizeof(T) <= 128 KiB per tile of S systems, i.e. N <= 1024, and M*sizeof(T) a
 * multiple of 16): ONE launch takes every tile of systems through all `nsteps` steps with the
 * state held in shared memory (HBM traffic: read c once, write c once, whatever nsteps is).
 * Otherwise one launch per step (thread per system, g through `scratch`).
 *  kind 0, Cahn-Hilliard (Eq. 2), L = second-difference matrix with boundary `bc`:
 *     form 0 (direct):     A c+ = c + r L (c^3 - c)
 *     form 1 (increment):  q = r (c^3 - c) - sigma L c;   A delta = L q;   c+ = c + delta
 *     (algebraically identical; form 1 conserves mean(c) to rounding when bc = 1).
 *  kind 1, hyperdiffusion Crank-Nicolson (PAPER.md:87-89 Eq. 6, :117 Eq. 7c):
 *     A c+ = (2I - A) c, with the handle's own diagonals (bc, form, r, sigma ignored).
 *     Evaluated as c+ = 2 A^{-1} c - c (the same scheme, no stencil): on chip for N <= 1024, else one chunked solve with a
 *     2x - f store stage per step (2 passes over the state, no scratch).
 *  bc 0: Dirichlet L (diag -2, off 1).  bc 1: zero-flux L (corner diagonal entries -1).
 *  kind 0, form 1 is the scheme of Eq. 2 only if the handle's A IS I + sigma L^2 with this sigma and bc:
 *  pent_factor records whether its matrix has that form (and which sigma, bc), and the call returns
 *  PENT_ERR_ARG on a mismatch (relative tolerance 1e-12 fp64, 1e-6 fp32).  form 0 takes any A.
 * c_inout: device, N*M, interleaved, updated in place.  scratch: device, N*M elements, or NULL
 * (the library then allocates and frees a stream-ordered temporary). */
typedef struct {
    int kind;
    int bc;
    int form;
    double r;       /* dt/dx^2 */
    double sigma;   /* gamma dt/dx^4 */
} pent_step_params;

int pent_step_batch(const pent_handle* h, const pent_step_params* p, int64_t M,
                    void* c_inout, void* scratch, int nsteps, void* stream);
/* Same with an explicit kernel (measurement / tests): PENT_KERNEL_AUTO, PENT_KERNEL_THREAD_PER_SYSTEM
 * or PENT_KERNEL_CHUNKED (= the on-chip kernel; PENT_ERR_ARG when the shape does not fit). */
int pent_step_batch_v(const pent_handle* h, const pent_step_params* p, int64_t M,
                      void* c_inout, void* scratch, int nsteps, void* stream, int kernel);
/* Which kernel pent_step_batch runs for M systems: PENT_KERNEL_CHUNKED or PENT_KERNEL_THREAD_PER_SYSTEM. */
int pent_step_kernel_choice(const pent_handle* h, int64_t M);

/* ---- forced Cahn-Hilliard, one parameter set per system (Remark 1, Eq. 3) -----------
 * "A parameter study based on the model (3) provides the motivation for batch programming in this work":
 * system i of the batch is the run with parameters (mu1[i], mu2[i]).  The paper names no Phi; this library
 * implements a zero-mean travelling wave (reading C-22)
 *     Phi(x, t; mu1, mu2) = mu1 cos(2 pi (x - mu2 t)),   x_k = (k + 1/2) / N   (cell centres of the unit interval),
 * treated explicitly like the other bracketed term of Eq. 2: step n of a call is taken at t_n = t0 + n dt and adds
 * dt * Phi(x_k, t_n) to row k of the right-hand side of pent_step_batch(kind 0) (either form).  sum_k Phi(x_k) = 0,
 * so the zero-flux scheme still conserves mean(c).  p->kind must be 0; g->kind 0 = no forcing (= pent_step_batch).
 * mu1, mu2: device, M elements of the handle's dtype.  Everything else as pent_step_batch; still ONE kernel for
 * all nsteps (the forcing is formed in registers from two per-system amplitudes per step). */
typedef struct {
    int kind;           /* 0 none, 1 travelling wave */
    double dt;          /* time step (the forcing enters the right-hand side as dt * Phi) */
    double t0;          /* time of the first step of this call */
    const void* mu1;    /* device, M: amplitude */
    const void* mu2;    /* device, M: wave speed */
} pent_forcing;
int pent_step_batch_forced(const pent_handle* h, const pent_step_params* p, const pent_forcing* g, int64_t M,
                           void* c_inout, void* scratch, int nsteps, void* stream);
int pent_step_batch_forced_v(const pent_handle* h, const pent_step_params* p, const pent_forcing* g, int64_t M,
                             void* c_inout, void* scratch, int nsteps, void* stream, int kernel);

/* ---- 2-D ADI time step built on the 1-D solves (section IV; reading C-23) ---------
 * Peaceman-Rachford splitting of u_t = D_x u + D_y u with A_x = I - (dt/2) D_x (handle hx, N = Nx) and
 * A_y = I - (dt/2) D_y (handle hy, N = Ny), e.g. the Remark-3 heat matrices:
 *     A_x u* = (2I - A_y) u^n  (explicit along y, implicit along x),   A_y u^{n+1} = (2I - A_x) u*.
 * u: device, Ny x Nx elements, row-major (u[y*Nx + x]), updated in place: its rows are solved as a system-major
 * batch (pent_solve_batch_rows), its columns as an interleaved batch (pent_solve_batch).  scratch: device,
 * Ny*Nx elements, or NULL (stream-ordered temporary).  After the first explicit half of a call every later one is formed
 * as 2 x - f in the store stage of the solve before it ((2I - A) A^{-1} f = 2 A^{-1} f - f): two launches and 4 passes over
 * the field per step, the same scheme in another order of evaluation.  hx, hy: shared-A, non-periodic, same dtype;
 * PENT_ERR_ARG otherwise, or when Nx is too long for the on-chip row solve.  Asynchronous on `stream`. */
int pent_adi_step_batch(const pent_handle* hx, const pent_handle* hy, void* u, void* scratch, int nsteps,
                        void* stream);

/* ---- introspection ------------------------------------------------------------------------ */
int pent_handle_n(const pent_handle* h);                 /* N, or -1 */
int pent_handle_dtype(const pent_handle* h);             /* pent_dtype, or -1 */
int64_t pent_handle_m(const pent_handle* h);             /* M of a per-system handle, 0 for shared A, -1 for NULL */
int pent_handle_device(const pent_handle* h);            /* CUDA device ordinal of the handle, or -1 */
/* Stability figures of the chunked evaluation (host, 3 doubles): max |Phi|, |X|, |Psi| = the largest response of the
 * forward recurrence, of its back substitution and of the backward recurrence to a unit incoming state inside one
 * chunk of 32 (fp64) / 64 (fp32) rows.  The on-chip kernels restart their local sweeps from a zero state, so their
 * intermediates (and rounding noise) exceed the serial sweep's by up to this factor; when it exceeds 1e6 (fp64) /
 * 1e3 (fp32) PENT_KERNEL_AUTO runs the serial thread-per-system kernels instead (pent_solve_kernel_choice says so).
 * SPD matrices I + sigma L^2: about 5 sqrt(sigma).  Shared-A handles (periodic: of the block E). */
int pent_handle_growth(const pent_handle* h, double* out3);
int pent_handle_band(const pent_handle* h);              /* shared A: 1 = tridiagonal (a == e == 0), 2 = pentadiagonal; -1 */
/* Cluster kernels (Q = 2, 4, 8, 16 CTAs split k): with how many neighbouring ranks on each side a CTA NEEDS to exchange its
 * block aggregates (the kernels use it for Q >= 8, where it pays).  1 when every block transfer product of the handle is below 1e-25 (a state entering a block of >= 32 chunks
 * has decayed to nothing by its end: the usual case for diagonally dominant matrices), else Q - 1 (every rank).  -1: no
 * tables for that cluster size. */
int pent_handle_exchange_depth(const pent_handle* h, int Q);
/* Copies the fp64 factor arrays (N doubles each; any pointer may be NULL) to HOST memory:
 * eps, beta, alpha = bands of L, gamma, delta = bands of R (Eq. 13).  Shared-A only. */
int pent_handle_factors(const pent_handle* h, double* eps, double* beta, double* alpha,
                        double* gamma, double* delta);
/* Which kernel PENT_KERNEL_AUTO picks for M systems on this handle: PENT_KERNEL_THREAD_PER_SYSTEM,
 * or PENT_KERNEL_CHUNKED_CFG(Q, S) with the chosen shape (low byte = PENT_KERNEL_CHUNKED). */
int pent_solve_kernel_choice(const pent_handle* h, int64_t M);
int pent_last_cuda_error(void);                         /* thread-local cudaError_t of the last PENT_ERR_CUDA */
/* Number of kernel launches the library has enqueued from this thread since the last call with
 * reset != 0 (used by bench.py for its gpu_launches field). */
int64_t pent_launch_count(int reset);
const char* pent_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PENT_H_ */
