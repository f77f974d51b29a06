"""CPU oracle for the batched pentadiagonal path -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It shares no code with
`paper_1807_07382_b200/` and neither imports the other.

Thin ctypes wrapper around `pent_oracle.c` / `pent_oracle_step.c` (plain fp64 C,
PAPER.md:148-244 transcribed step by step).  The wrapper only marshals arrays and
transposes between the interleaved batch layout (N, M) used by the library
 and the serial "one system per row" layout (M, N) the paper's CPU
code uses; all arithmetic is in the C files.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "pent_oracle.c"), os.path.join(_HERE, "pent_oracle_step.c"),
        os.path.join(_HERE, "pent_oracle_periodic.c"), os.path.join(_HERE, "pent_oracle_ld.c"),
        os.path.join(_HERE, "pent_oracle_adi.c")]
_LIB = os.path.join(_HERE, "libpent_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (no FMA contraction: one reproducible definition)."""
    if not force and os.path.exists(_LIB) and all(
            os.path.getmtime(_LIB) >= os.path.getmtime(s) for s in _SRC):
        return _LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-fopenmp",
           "-o", _LIB] + _SRC + ["-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.pent_oracle_factor.restype = C.c_int
        _lib.pent_oracle_dense_ge.restype = C.c_int
        _lib.pent_oracle_periodic_setup.restype = C.c_int
        _lib.pent_oracle_ld_solve_rows.restype = C.c_int
        _lib.pent_oracle_ld_step_rows.restype = C.c_int
        _lib.pent_oracle_ld_periodic_solve_rows.restype = C.c_int
    return _lib


def _p(x: np.ndarray):
    assert x.dtype == np.float64 and x.flags.c_contiguous
    return x.ctypes.data_as(C.POINTER(C.c_double))


def _f64(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.float64)


@dataclass
class Factors:
    """L (eps, beta, alpha) and R (gamma, delta) of PAPER.md Eq. 13, plus the
    original diagonals (kept for residuals and for the (2I-A)C right-hand side)."""
    N: int
    eps: np.ndarray
    beta: np.ndarray
    alpha: np.ndarray
    gamma: np.ndarray
    delta: np.ndarray
    diags: tuple


class SingularPivot(ArithmeticError):
    def __init__(self, row: int):
        super().__init__(f"zero or non-finite pivot at row {row} (no pivoting, PAPER.md:275)")
        self.row = row


def factor(a, b, c, d, e) -> Factors:
    """A = L R.  Raises SingularPivot(row) on a bad pivot."""
    a, b, c, d, e = (_f64(v) for v in (a, b, c, d, e))
    N = c.shape[0]
    out = [np.zeros(N) for _ in range(5)]
    rc = _load().pent_oracle_factor(C.c_int(N), _p(a), _p(b), _p(c), _p(d), _p(e),
                                    *[_p(o) for o in out])
    if rc != 0:
        raise SingularPivot(rc - 1)
    return Factors(N, *out, diags=(a, b, c, d, e))


def solve(fac: Factors, f) -> np.ndarray:
    """One system, contiguous f of length N.  PAPER.md:223-242."""
    f = _f64(f)
    x = np.empty_like(f)
    _load().pent_oracle_solve(C.c_int(fac.N), _p(fac.eps), _p(fac.beta), _p(fac.alpha),
                              _p(fac.gamma), _p(fac.delta), _p(f), _p(x))
    return x


def to_rows(f_interleaved: np.ndarray) -> np.ndarray:
    """(N, M) interleaved -> (M, N) one system per row."""
    # always a fresh array: for M == 1 the transpose of a contiguous (N, 1) array is itself contiguous, and the
    # in-place C routines (step_rows) would then overwrite the caller's input
    return np.array(np.asarray(f_interleaved, dtype=np.float64).T, order="C", copy=True)


def solve_rows(fac: Factors, F_rows: np.ndarray, nthreads: int = 1) -> np.ndarray:
    """Batch solve in the serial layout (M, N); this is what the CPU baseline times."""
    F_rows = _f64(F_rows)
    M = F_rows.shape[0]
    X = np.empty_like(F_rows)
    _load().pent_oracle_solve_rows(C.c_int(fac.N), C.c_long(M), _p(fac.eps), _p(fac.beta),
                                   _p(fac.alpha), _p(fac.gamma), _p(fac.delta),
                                   _p(F_rows), _p(X), C.c_int(nthreads))
    return X


def solve_batch(fac: Factors, f_interleaved, nthreads: int = 1) -> np.ndarray:
    """Interleaved (N, M) in, interleaved (N, M) out (fp64)."""
    X = solve_rows(fac, to_rows(f_interleaved), nthreads)
    return np.ascontiguousarray(X.T)


def factor_solve_batch(a, b, c, d, e, f, nthreads: int = 1):
    """Per-system matrices (PAPER.md:289 'Rewrite' mode); every argument is an
    interleaved (N, M) array.  Returns (x (N, M), info (M,)): info[i] = 0 or
    first bad row + 1."""
    rows = [to_rows(v) for v in (a, b, c, d, e, f)]
    M, N = rows[5].shape
    X = np.zeros_like(rows[5])
    info = np.zeros(M, dtype=np.int32)
    _load().pent_oracle_factor_solve_rows(
        C.c_int(N), C.c_long(M), *[_p(r) for r in rows], _p(X),
        info.ctypes.data_as(C.POINTER(C.c_int)), C.c_int(nthreads))
    return np.ascontiguousarray(X.T), info


def dense_ge(A: np.ndarray, f: np.ndarray) -> np.ndarray:
    """Dense Gaussian elimination with partial pivoting (second, independent oracle)."""
    A = _f64(A).copy()
    f = _f64(f).copy()
    N = A.shape[0]
    x = np.zeros(N)
    rc = _load().pent_oracle_dense_ge(C.c_int(N), _p(A), _p(f), _p(x))
    if rc:
        raise ArithmeticError("singular")
    return x


def rhs(fac: Factors, kind: int, bc: int, form: int, r: float, sigma: float, Cvec) -> np.ndarray:
    """Right-hand side of one time step for one system (see pent_oracle_step.c)."""
    Cvec = _f64(Cvec)
    N = fac.N
    out = np.empty(N)
    work = np.empty(2 * N)
    _load().pent_oracle_rhs(C.c_int(N), C.c_int(kind), C.c_int(bc), C.c_int(form),
                            C.c_double(r), C.c_double(sigma), *[_p(v) for v in fac.diags],
                            _p(Cvec), _p(out), _p(work))
    return out


def step_batch(fac: Factors, kind: int, bc: int, form: int, r: float, sigma: float,
               c_interleaved, nsteps: int, nthreads: int = 1) -> np.ndarray:
    """nsteps fused steps on an interleaved (N, M) state; returns the new state."""
    Crows = to_rows(c_interleaved)
    M = Crows.shape[0]
    _load().pent_oracle_step_rows(
        C.c_int(fac.N), C.c_long(M), C.c_int(kind), C.c_int(bc), C.c_int(form),
        C.c_double(r), C.c_double(sigma), *[_p(v) for v in fac.diags],
        _p(fac.eps), _p(fac.beta), _p(fac.alpha), _p(fac.gamma), _p(fac.delta),
        _p(Crows), C.c_int(nsteps), C.c_int(nthreads))
    return np.ascontiguousarray(Crows.T)


def forcing(N: int, t: float, mu1: float, mu2: float) -> np.ndarray:
    """Phi(x_k, t; mu1, mu2) of the forced Cahn-Hilliard equation (reading C-22)."""
    out = np.empty(N)
    _load().pent_oracle_forcing(C.c_int(N), C.c_double(t), C.c_double(mu1), C.c_double(mu2), _p(out))
    return out


def step_forced_batch(fac: Factors, bc: int, form: int, r: float, sigma: float, dt: float, t0: float,
                      mu1, mu2, c_interleaved, nsteps: int, nthreads: int = 1) -> np.ndarray:
    """nsteps forced Cahn-Hilliard steps (Eq. 3) with per-system parameters mu1[i], mu2[i]."""
    Crows = to_rows(c_interleaved)
    M = Crows.shape[0]
    mu1, mu2 = _f64(mu1), _f64(mu2)
    assert mu1.shape == (M,) and mu2.shape == (M,)
    _load().pent_oracle_step_forced_rows(
        C.c_int(fac.N), C.c_long(M), C.c_int(bc), C.c_int(form), C.c_double(r), C.c_double(sigma),
        C.c_double(dt), C.c_double(t0), _p(mu1), _p(mu2), *[_p(v) for v in fac.diags],
        _p(fac.eps), _p(fac.beta), _p(fac.alpha), _p(fac.gamma), _p(fac.delta),
        _p(Crows), C.c_int(nsteps), C.c_int(nthreads))
    return np.ascontiguousarray(Crows.T)


# ---- periodic (cyclic) pentadiagonal systems, PAPER.md:104-146 (pent_oracle_periodic.c) -----------
@dataclass
class PeriodicFactors:
    """Set-up of the periodic reduction (Eqs. 8-12): factors of E, the stored
    h^T E^{-1} (Y, shape (2, N-2)), the columns k (shape (2, N-2)) and the inverted 2x2 matrix."""
    N: int
    facE: np.ndarray
    Y: np.ndarray
    kk: np.ndarray
    s2inv: np.ndarray
    diags: tuple


def factor_periodic(a, b, c, d, e) -> PeriodicFactors:
    """Diagonals are length-N, row-indexed and wrapped cyclically (every entry is used)."""
    a, b, c, d, e = (_f64(v) for v in (a, b, c, d, e))
    N = c.shape[0]
    if N < 6:
        raise ValueError("periodic reduction needs N >= 6")
    n = N - 2
    facE, Y, kk, s2 = np.zeros(5 * n), np.zeros(2 * n), np.zeros(2 * n), np.zeros(4)
    rc = _load().pent_oracle_periodic_setup(C.c_int(N), _p(a), _p(b), _p(c), _p(d), _p(e),
                                            _p(facE), _p(Y), _p(kk), _p(s2))
    if rc != 0:
        raise SingularPivot(rc - 1)
    return PeriodicFactors(N, facE, Y.reshape(2, n), kk.reshape(2, n), s2.reshape(2, 2),
                           (a, b, c, d, e))


def solve_periodic_batch(pf: PeriodicFactors, f_interleaved, nthreads: int = 1) -> np.ndarray:
    """Interleaved (N, M) in, interleaved (N, M) out."""
    F = to_rows(f_interleaved)
    X = np.empty_like(F)
    _load().pent_oracle_periodic_solve_rows(
        C.c_int(pf.N), C.c_long(F.shape[0]), _p(pf.facE), _p(np.ascontiguousarray(pf.Y.ravel())),
        _p(np.ascontiguousarray(pf.kk.ravel())), _p(np.ascontiguousarray(pf.s2inv.ravel())),
        _p(F), _p(X), C.c_int(nthreads))
    return np.ascontiguousarray(X.T)


def step_periodic_batch(pf: PeriodicFactors, c_interleaved, nsteps: int, nthreads: int = 1) -> np.ndarray:
    """nsteps Crank-Nicolson steps A c+ = (2I - A) c with the cyclic A (Eq. 6, 7c)."""
    Crows = to_rows(c_interleaved)
    _load().pent_oracle_periodic_step_rows(
        C.c_int(pf.N), C.c_long(Crows.shape[0]), *[_p(v) for v in pf.diags], _p(pf.facE),
        _p(np.ascontiguousarray(pf.Y.ravel())), _p(np.ascontiguousarray(pf.kk.ravel())),
        _p(np.ascontiguousarray(pf.s2inv.ravel())), _p(Crows), C.c_int(nsteps), C.c_int(nthreads))
    return np.ascontiguousarray(Crows.T)


# ---- the same transcription in long double (pent_oracle_ld.c): the "truth" that measured tolerances refer to ----
def ld_solve_batch(diags, f_interleaved, nthreads: int = 1) -> np.ndarray:
    """A^{-1} f in 80-bit long double, rounded once to fp64.  Interleaved (N, M) in and out."""
    a, b, c, d, e = (_f64(v) for v in diags)
    F = to_rows(f_interleaved)
    X = np.empty_like(F)
    rc = _load().pent_oracle_ld_solve_rows(C.c_int(c.shape[0]), C.c_long(F.shape[0]), _p(a), _p(b), _p(c),
                                           _p(d), _p(e), _p(F), _p(X), C.c_int(nthreads))
    if rc != 0:
        raise SingularPivot(rc - 1)
    return np.ascontiguousarray(X.T)


def ld_factor_solve_batch(a, b, c, d, e, f, nthreads: int = 1):
    """Per-system matrices in long double; arguments interleaved (N, M)."""
    rows = [to_rows(v) for v in (a, b, c, d, e, f)]
    M, N = rows[5].shape
    X = np.zeros_like(rows[5])
    info = np.zeros(M, dtype=np.int32)
    _load().pent_oracle_ld_factor_solve_rows(C.c_int(N), C.c_long(M), *[_p(r) for r in rows], _p(X),
                                             info.ctypes.data_as(C.POINTER(C.c_int)), C.c_int(nthreads))
    return np.ascontiguousarray(X.T), info


def ld_step_batch(diags, kind: int, bc: int, form: int, r: float, sigma: float, c_interleaved, nsteps: int,
                  nthreads: int = 1) -> np.ndarray:
    """nsteps time steps with every intermediate (and the state between steps) in long double."""
    a, b, c, d, e = (_f64(v) for v in diags)
    Crows = to_rows(c_interleaved)
    rc = _load().pent_oracle_ld_step_rows(C.c_int(c.shape[0]), C.c_long(Crows.shape[0]), C.c_int(kind), C.c_int(bc),
                                          C.c_int(form), C.c_double(r), C.c_double(sigma), _p(a), _p(b), _p(c),
                                          _p(d), _p(e), _p(Crows), C.c_int(nsteps), C.c_int(nthreads))
    if rc != 0:
        raise SingularPivot(rc - 1)
    return np.ascontiguousarray(Crows.T)


def ld_solve_periodic_batch(diags, f_interleaved, nthreads: int = 1) -> np.ndarray:
    """Periodic (cyclic) solve, set-up and Eqs. 12 / 11 in long double."""
    a, b, c, d, e = (_f64(v) for v in diags)
    F = to_rows(f_interleaved)
    X = np.empty_like(F)
    rc = _load().pent_oracle_ld_periodic_solve_rows(C.c_int(c.shape[0]), C.c_long(F.shape[0]), _p(a), _p(b), _p(c),
                                                    _p(d), _p(e), _p(F), _p(X), C.c_int(nthreads))
    if rc != 0:
        raise SingularPivot(rc - 1)
    return np.ascontiguousarray(X.T)


# ---- 2-D ADI time step on top of the 1-D solver (pent_oracle_adi.c, reading C-23) ----
def adi_steps(fac_x: Factors, fac_y: Factors, u, nsteps: int, nthreads: int = 1) -> np.ndarray:
    """nsteps Peaceman-Rachford steps on a field u of shape (Ny, Nx) (row-major): A_x u* = (2I - A_y) u,
    A_y u+ = (2I - A_x) u*.  fac_x / fac_y: factors of A_x (N = Nx) and A_y (N = Ny)."""
    U = np.array(u, dtype=np.float64, order="C", copy=True)
    Ny, Nx = U.shape
    assert fac_x.N == Nx and fac_y.N == Ny
    W = np.empty_like(U)
    pack = lambda vs: np.ascontiguousarray(np.concatenate([_f64(v) for v in vs]))
    dx, dy = pack(fac_x.diags), pack(fac_y.diags)
    fx = pack((fac_x.eps, fac_x.beta, fac_x.alpha, fac_x.gamma, fac_x.delta))
    fy = pack((fac_y.eps, fac_y.beta, fac_y.alpha, fac_y.gamma, fac_y.delta))
    _load().pent_oracle_adi_steps(C.c_int(Nx), C.c_int(Ny), _p(dx), _p(fx), _p(dy), _p(fy), _p(U), _p(W),
                                  C.c_int(nsteps), C.c_int(nthreads))
    return U
