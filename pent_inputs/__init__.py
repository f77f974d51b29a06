"""Seeded synthetic inputs for the batched pentadiagonal path (numpy only).

This module is the ONE thing the CPU oracle (`oracle/`) and the CUDA path
(`paper_1807_07382_b200/`) share.  It holds no arithmetic of the method
(no factorisation, no sweep, no RHS stencil): only

* a counter-based random generator, so a value depends on (seed, stream,
  element index) and never on generation order;
* the diagonals of the benchmark matrices A = I + sigma * L^2
  (BASELINE.json configs), which are *inputs*
  to `pent_factor`;
* the named workload configurations of BASELINE.json.

Array convention: five length-N arrays
indexed by ROW k,  a[k]=A[k][k-2], b[k]=A[k][k-1], c[k]=A[k][k],
d[k]=A[k][k+1], e[k]=A[k][k+2].  Entries that fall outside the matrix
(a[0], a[1], b[0], d[N-1], e[N-2], e[N-1]) are set to 0 and never read.

Batches are interleaved: a 2-D array of shape (N, M),
C-contiguous, so element k of system i sits at flat index k*M + i.
"""
from __future__ import annotations

import numpy as np

_U64 = np.uint64
_GOLDEN = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser (Steele, Lea, Flood 2014), vectorised on uint64."""
    z = (z ^ (z >> _U64(30))) * _M1
    z = (z ^ (z >> _U64(27))) * _M2
    return z ^ (z >> _U64(31))


def hash_u01(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """Uniform [0,1) doubles, one per element index (53-bit fractions).

    u = (mix64(mix64(key) + (index+1)*GOLDEN) >> 11) * 2^-53,
    key = seed * 2^32 + stream.
    """
    with np.errstate(over="ignore"):
        key = _U64((int(seed) << 32 | (int(stream) & 0xFFFFFFFF)) & 0xFFFFFFFFFFFFFFFF)
        k0 = _mix64(np.asarray([key], dtype=_U64))[0]
        idx = np.asarray(index, dtype=_U64)
        z = _mix64(k0 + (idx + _U64(1)) * _GOLDEN)
    return (z >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def _index_grid(N: int, M: int, col0: int = 0, Mtot: int | None = None) -> np.ndarray:
    """Flat element indices k*Mtot + (col0+i) for an (N, M) window of an (N, Mtot) batch."""
    Mtot = M if Mtot is None else Mtot
    k = np.arange(N, dtype=np.uint64)[:, None] * np.uint64(Mtot)
    i = np.arange(col0, col0 + M, dtype=np.uint64)[None, :]
    return k + i


def uniform_pm1(seed: int, stream: int, N: int, M: int, col0: int = 0,
                Mtot: int | None = None) -> np.ndarray:
    """(N, M) array, i.i.d. uniform[-1,1).  `col0`/`Mtot` select a window of
    systems of a larger batch (used to shard M across ranks: the values of
    system i do not depend on which rank generates it)."""
    out = np.empty((N, M), dtype=np.float64)
    rows = max(1, (1 << 22) // max(M, 1))
    for r0 in range(0, N, rows):
        r1 = min(N, r0 + rows)
        idx = _index_grid(r1 - r0, M, col0, Mtot) + np.uint64(r0) * np.uint64(M if Mtot is None else Mtot)
        out[r0:r1] = 2.0 * hash_u01(seed, stream, idx) - 1.0
    return out


def normal01(seed: int, stream: int, N: int, M: int, col0: int = 0,
             Mtot: int | None = None) -> np.ndarray:
    """(N, M) array, i.i.d. N(0,1) by Box-Muller on streams (stream, stream+1)."""
    out = np.empty((N, M), dtype=np.float64)
    rows = max(1, (1 << 22) // max(M, 1))
    for r0 in range(0, N, rows):
        r1 = min(N, r0 + rows)
        idx = _index_grid(r1 - r0, M, col0, Mtot) + np.uint64(r0) * np.uint64(M if Mtot is None else Mtot)
        u1 = 1.0 - hash_u01(seed, stream, idx)          # (0,1]
        u2 = hash_u01(seed, stream + 1, idx)
        out[r0:r1] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return out


def uniform_vec(seed: int, stream: int, M: int, lo: float, hi: float,
                col0: int = 0) -> np.ndarray:
    """Length-M vector uniform[lo,hi), one value per system."""
    idx = np.arange(col0, col0 + M, dtype=np.uint64)
    return lo + (hi - lo) * hash_u01(seed, stream, idx)


# ----------------------------------------------------------------------------
# benchmark matrices: diagonals of A = I + sigma * L^2
# ----------------------------------------------------------------------------
def second_difference(N: int, bc: str = "dirichlet") -> np.ndarray:
    """Dense N x N second-difference matrix L (diag -2, off-diagonals 1).
    bc='dirichlet': plain Toeplitz.  bc='zeroflux': corner diagonal entries -1,
    so 1^T L = 0.  Used by tests to build A densely."""
    L = np.zeros((N, N))
    for k in range(N):
        L[k, k] = -2.0
        if k > 0:
            L[k, k - 1] = 1.0
        if k + 1 < N:
            L[k, k + 1] = 1.0
    if bc == "zeroflux":
        L[0, 0] = -1.0
        L[N - 1, N - 1] = -1.0
    elif bc != "dirichlet":
        raise ValueError(bc)
    return L


def diagonals_I_plus_sigma_L2(N: int, sigma, bc: str = "dirichlet"):
    """Diagonals (a, b, c, d, e) of A = I + sigma*L^2, L = second_difference(N, bc).

    `sigma` may be a scalar (arrays of shape (N,)) or a length-M vector
    (arrays of shape (N, M), interleaved per-system diagonals, config 5b).
    The entries of L^2 are small integers, written out here (N >= 4):
      dirichlet: diag [5,6,...,6,5], first off-diagonals -4, second 1
      zeroflux : diag [2,6,...,6,2], first off-diagonals [-3,-4,...,-4,-3], second 1
    (BASELINE.json configs).
    """
    if N < 4:
        raise ValueError("N >= 4 required for the written-out L^2 pattern")
    l2c = np.full(N, 6.0)
    l2o1 = np.full(N - 1, -4.0)        # L2[k][k+1] = L2[k+1][k], k = 0..N-2
    l2o2 = np.ones(N - 2)              # L2[k][k+2] = L2[k+2][k]
    if bc == "dirichlet":
        l2c[0] = l2c[-1] = 5.0
    elif bc == "zeroflux":
        l2c[0] = l2c[-1] = 2.0
        l2c[1] = l2c[-2] = 6.0
        l2o1[0] = l2o1[-1] = -3.0
    else:
        raise ValueError(bc)
    s = np.asarray(sigma, dtype=np.float64)
    shape = (N,) + s.shape
    s = s[None, ...] if s.ndim else s
    ex = (slice(None),) + (None,) * (len(shape) - 1)
    a = np.zeros(shape); b = np.zeros(shape); c = np.zeros(shape)
    d = np.zeros(shape); e = np.zeros(shape)
    c[...] = 1.0 + s * l2c[ex]
    d[:-1] = s * l2o1[ex]
    b[1:] = s * l2o1[ex]
    e[:-2] = s * l2o2[ex]
    a[2:] = s * l2o2[ex]
    return a, b, c, d, e


def heat4_cn_diagonals(N: int, s_h: float, bc: str = "dirichlet"):
    """The pentadiagonal matrix of PAPER.md:96 (Remark 3): heat equation C_t = C_xx, Crank-Nicolson in time,
    fourth-order centred differences in space (nearest and next-nearest neighbours),
        C_xx ~ (-C_{i-2} + 16 C_{i-1} - 30 C_i + 16 C_{i+1} - C_{i+2}) / (12 dx^2) = (12 L - L^2) C / (12 dx^2),
    so  A = I - (dt/2) (12 L - L^2) / (12 dx^2) = I + s_h (L^2 - 12 L),   s_h = dt / (24 dx^2),
    and one step is A C+ = (2I - A) C (the library's kind-1 step).  Entries written out:
      interior rows  (s_h, -16 s_h, 1 + 30 s_h, -16 s_h, s_h);
      bc='dirichlet': L, L^2 formed exactly (corner diagonal 1 + 29 s_h), i.e. odd reflection at the walls;
      bc='periodic' : five constant length-N arrays, every entry used (cyclic matrix, like Eq. 7a).
    Returns (a, b, c, d, e), row-indexed like every other generator here."""
    if N < 4:
        raise ValueError("N >= 4 required")
    one = np.ones(N)
    if bc == "periodic":
        return s_h * one, -16.0 * s_h * one, (1.0 + 30.0 * s_h) * one, -16.0 * s_h * one, s_h * one
    if bc != "dirichlet":
        raise ValueError(bc)
    a = np.zeros(N); b = np.zeros(N); c = np.zeros(N); d = np.zeros(N); e = np.zeros(N)
    c[:] = 1.0 + 30.0 * s_h
    c[0] = c[-1] = 1.0 + 29.0 * s_h
    d[:-1] = -16.0 * s_h
    b[1:] = -16.0 * s_h
    e[:-2] = s_h
    a[2:] = s_h
    return a, b, c, d, e


def dense_from_diagonals(a, b, c, d, e) -> np.ndarray:
    """Assemble the dense N x N matrix from row-indexed diagonals (1 system)."""
    N = len(c)
    A = np.zeros((N, N))
    for k in range(N):
        A[k, k] = c[k]
        if k >= 1:
            A[k, k - 1] = b[k]
        if k >= 2:
            A[k, k - 2] = a[k]
        if k + 1 < N:
            A[k, k + 1] = d[k]
        if k + 2 < N:
            A[k, k + 2] = e[k]
    return A


def random_diag_dominant(seed: int, N: int, M: int | None = None):
    """Random NON-symmetric strictly diagonally dominant diagonals
    (off-diagonals uniform[-1,1), diagonal = 1.5 + sum|off| with random sign
    pattern fixed positive).  Shape (N,) or (N, M)."""
    shp = (N, 1 if M is None else M)
    a = uniform_pm1(seed, 11, *shp); b = uniform_pm1(seed, 12, *shp)
    d = uniform_pm1(seed, 13, *shp); e = uniform_pm1(seed, 14, *shp)
    a[:2] = 0.0; b[:1] = 0.0
    d[N - 1:] = 0.0
    e[max(N - 2, 0):] = 0.0
    c = 1.5 + np.abs(a) + np.abs(b) + np.abs(d) + np.abs(e)
    if M is None:
        return tuple(v[:, 0].copy() for v in (a, b, c, d, e))
    return a, b, c, d, e


def spd_banded_product(seed: int, N: int, rho: float):
    """Diagonals of A = B B^T, B lower banded with bandwidth 2 whose rows are ~(rho^2, -2 rho, 1) (jittered by
    +-5 %): symmetric positive definite by construction, NOT diagonally dominant for rho > 0.3, with
    cond(A) ~ (1 - rho)^-4.  PAPER.md:275-277 names SPD as one of the two classes the algorithm is stable for;
    the I + sigma L^2 family and the diagonally dominant generator above cover only the other."""
    j0 = 1.0 + 0.05 * uniform_pm1(seed, 31, N, 1)[:, 0]
    j1 = 1.0 + 0.05 * uniform_pm1(seed, 32, N, 1)[:, 0]
    j2 = 1.0 + 0.05 * uniform_pm1(seed, 33, N, 1)[:, 0]
    b0, b1, b2 = j0, -2.0 * rho * j1, rho * rho * j2          # B[k][k], B[k][k-1], B[k][k-2]
    b1[0] = 0.0
    b2[:2] = 0.0
    a = np.zeros(N); b = np.zeros(N); c = np.zeros(N); d = np.zeros(N); e = np.zeros(N)
    c[:] = b0 * b0 + b1 * b1 + b2 * b2
    b[1:] = b1[1:] * b0[:-1] + b2[1:] * b1[:-1]               # A[k][k-1] = B[k][k-1] B[k-1][k-1] + B[k][k-2] B[k-1][k-2]
    a[2:] = b2[2:] * b0[:-2]                                  # A[k][k-2] = B[k][k-2] B[k-2][k-2]
    d[:-1] = b[1:]
    e[:-2] = a[2:]
    return a, b, c, d, e


def transpose_diagonals(a, b, c, d, e):
    """Row-indexed diagonals of A^T (a column-diagonally-dominant matrix from a row-dominant one)."""
    N = len(c)
    at = np.zeros(N); bt = np.zeros(N); dt = np.zeros(N); et = np.zeros(N)
    at[2:] = np.asarray(e)[:-2]
    bt[1:] = np.asarray(d)[:-1]
    dt[:-1] = np.asarray(b)[1:]
    et[:-2] = np.asarray(a)[2:]
    return at, bt, np.array(c, dtype=np.float64), dt, et


# ----------------------------------------------------------------------------
# periodic (cyclic) matrices, Eq. 7a-7b
# ----------------------------------------------------------------------------
def periodic_hyperdiffusion_diagonals(N: int, sigma_x: float):
    """Constant diagonals of PAPER.md Eq. 7b: a = e = sigma_x, b = d = -4 sigma_x,
    c = 1 + 6 sigma_x, as five length-N arrays (every entry used: the matrix is cyclic)."""
    one = np.ones(N)
    return sigma_x * one, -4.0 * sigma_x * one, (1.0 + 6.0 * sigma_x) * one, -4.0 * sigma_x * one, sigma_x * one


def dense_from_periodic_diagonals(a, b, c, d, e) -> np.ndarray:
    """Dense N x N cyclic matrix: a[k] = A[k][(k-2)%N], b[k] = A[k][(k-1)%N], c[k] = A[k][k],
    d[k] = A[k][(k+1)%N], e[k] = A[k][(k+2)%N]  (Eq. 7a with row-indexed entries)."""
    N = len(c)
    A = np.zeros((N, N))
    for k in range(N):
        A[k, (k - 2) % N] += a[k]
        A[k, (k - 1) % N] += b[k]
        A[k, k] += c[k]
        A[k, (k + 1) % N] += d[k]
        A[k, (k + 2) % N] += e[k]
    return A


def random_periodic_diag_dominant(seed: int, N: int):
    """Random NON-symmetric strictly diagonally dominant cyclic diagonals (all entries used)."""
    a = uniform_pm1(seed, 21, N, 1)[:, 0]; b = uniform_pm1(seed, 22, N, 1)[:, 0]
    d = uniform_pm1(seed, 23, N, 1)[:, 0]; e = uniform_pm1(seed, 24, N, 1)[:, 0]
    c = 1.5 + np.abs(a) + np.abs(b) + np.abs(d) + np.abs(e)
    return a, b, c, d, e
