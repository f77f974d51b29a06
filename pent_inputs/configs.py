"""The named workloads of BASELINE.json `configs`.

Each entry only *describes* inputs; `make_*` functions draw them with the
counter-based generator of `pent_inputs`.  No method arithmetic here, with
one documented exception: config 2's manufactured right-hand side f = A x is
a banded matrix-vector product with the ORIGINAL diagonals (it is part of the
input recipe, BASELINE.json configs[1]; it uses no factor and no sweep).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from . import (diagonals_I_plus_sigma_L2, normal01, uniform_pm1, uniform_vec)


@dataclass(frozen=True)
class Workload:
    name: str
    N: int
    M: int
    sigma: float
    bc: str
    seed: int
    rhs: str            # 'uniform' | 'manufactured' | 'ch_state'
    note: str = ""


# sigma of config 4: gamma*dt/dx^4 = 1e-2 * 1e-6 * 1024^4
SIGMA_CH = 1e-2 * 1e-6 * 1024.0 ** 4
R_CH = 1e-6 * 1024.0 ** 2           # dt/dx^2

WORKLOADS = {
    "cfg1":  Workload("cfg1", 64, 256, 0.1, "dirichlet", 1, "uniform"),
    "cfg2":  Workload("cfg2", 512, 16384, 1.0, "dirichlet", 2, "manufactured"),
    "cfg3":  Workload("cfg3", 1024, 65536, 10.0, "dirichlet", 3, "uniform",
                      "headline: N=1024, M=65536"),
    "cfg4":  Workload("cfg4", 1024, 8192, SIGMA_CH, "zeroflux", 4, "ch_state",
                      "Cahn-Hilliard, 1000 steps"),
    "cfg5a": Workload("cfg5a", 4096, 32768, 0.5, "dirichlet", 5, "uniform"),
    # the paper's own benchmark shape: a batch of identical periodic
    # hyperdiffusion systems, Crank-Nicolson, N=1024, batch 8192, dt=1e-8 (sigma_x = dt/(2 dx^4))
    "paper_hd": Workload("paper_hd", 1024, 8192, 1e-8 / (2.0 * (1.0 / 1024) ** 4), "periodic", 7, "cos_mode",
                         "periodic hyperdiffusion, identical systems, 250 steps"),
    # cfg3's shape with the paper's periodic matrix (Eq. 7a-7b), for the periodic solve on its own
    "cfg3p": Workload("cfg3p", 1024, 65536, 10.0, "periodic", 8, "uniform", "periodic solve, N=1024, M=65536"),
    "cfg5b": Workload("cfg5b", 1024, 16384, float("nan"), "dirichlet", 6, "uniform",
                      "per-system sigma_i ~ U[0.1,10]"),
    # cfg3's shape with a TRIDIAGONAL matrix (a = e = 0): A = I - sigma L, the second-order
    # Crank-Nicolson heat matrix of cuThomasBatch's use case; runs the BAND = 1 instantiation
    "cfg3t": Workload("cfg3t", 1024, 65536, 10.0, "tridiagonal", 9, "uniform", "tridiagonal, N=1024, M=65536"),
    # 2-D ADI on a 4096 x 4096 field, heat equation with the Remark-3
    # fourth-order matrices along both axes, dt/(24 dx^2) = sigma
    "adi2d": Workload("adi2d", 4096, 4096, 40.0, "heat4", 10, "uniform", "Peaceman-Rachford ADI, 4096 x 4096 field"),
}


def banded_matvec(a, b, c, d, e, x: np.ndarray) -> np.ndarray:
    """y = A x for interleaved x of shape (N, M); diagonals shape (N,) or (N, M).
    Plain definition of the banded product, original diagonals only."""
    def col(v):
        return v[:, None] if v.ndim == 1 else v
    a, b, c, d, e = (col(np.asarray(v)) for v in (a, b, c, d, e))
    y = c * x
    y[1:] += b[1:] * x[:-1]
    y[2:] += a[2:] * x[:-2]
    y[:-1] += d[:-1] * x[1:]
    y[:-2] += e[:-2] * x[2:]
    return y


def make_matrix(w: Workload, M: int | None = None, col0: int = 0):
    """Diagonals for workload `w`.  cfg5b returns (N, M) per-system arrays."""
    if w.name == "cfg5b":
        M = w.M if M is None else M
        sig = uniform_vec(w.seed, 1, M, 0.1, 10.0, col0)
        return diagonals_I_plus_sigma_L2(w.N, sig, w.bc)
    if w.bc == "periodic":
        from . import periodic_hyperdiffusion_diagonals
        return periodic_hyperdiffusion_diagonals(w.N, w.sigma)
    if w.bc == "tridiagonal":          # I - sigma L (Dirichlet L): diag 1 + 2 sigma, off-diagonals -sigma
        z = np.zeros(w.N)
        b = np.full(w.N, -w.sigma); b[0] = 0.0
        d = np.full(w.N, -w.sigma); d[-1] = 0.0
        return z, b, np.full(w.N, 1.0 + 2.0 * w.sigma), d, z.copy()
    if w.bc == "heat4":
        from . import heat4_cn_diagonals
        return heat4_cn_diagonals(w.N, w.sigma)
    return diagonals_I_plus_sigma_L2(w.N, w.sigma, w.bc)


def make_rhs(w: Workload, M: int | None = None, col0: int = 0):
    """Right-hand sides f of shape (N, M) (interleaved).  For 'manufactured'
    returns (f, x_true); for 'ch_state' returns the initial concentration c0.
    `M`/`col0` select a window of the systems of the full batch (sharding)."""
    M = w.M if M is None else M
    if w.rhs == "uniform":
        return uniform_pm1(w.seed, 0, w.N, M, col0, w.M)
    if w.rhs == "manufactured":
        x = normal01(w.seed, 2, w.N, M, col0, w.M)
        f = banded_matvec(*make_matrix(w), x)
        return f, x
    if w.rhs == "ch_state":
        m = uniform_vec(w.seed, 5, M, -0.5, 0.5, col0)
        return m[None, :] + 0.05 * uniform_pm1(w.seed, 0, w.N, M, col0, w.M)
    raise ValueError(w.rhs)


def sine_modes(N: int) -> np.ndarray:
    """(N, N) interleaved batch whose system j-1 is the sine mode
    sin(pi*j*(k+1)/(N+1)), k = 0..N-1 (BASELINE.json configs[0], north_star)."""
    k = np.arange(1, N + 1)[:, None]
    j = np.arange(1, N + 1)[None, :]
    return np.sin(np.pi * k * j / (N + 1))
