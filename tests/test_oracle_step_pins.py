"""Pins for the time-step oracle (oracle/pent_oracle_step.c) and the input recipes.
CPU only.  The step oracle is pinned by dense linear algebra (numpy matmul / LAPACK solve
on the assembled matrices), by the algebraic identity between the direct and increment
forms, by exact conservation of the mean under the zero-flux operator, and by the exact
per-mode amplification factor of the Crank-Nicolson hyperdiffusion step.
Citations: PAPER.md:53 (Eq. 2), :81-92 (Eqs. 5-6), :117 (Eq. 7c); SURVEY.md C-13..C-18, P10.
"""
import numpy as np
import pytest

import oracle
import pent_inputs as pin
from pent_inputs.configs import (R_CH, SIGMA_CH, WORKLOADS, banded_matvec, make_matrix,
                                 make_rhs, sine_modes)


# ---- input recipes -----------------------------------------------------------------------
@pytest.mark.parametrize("bc", ["dirichlet", "zeroflux"])
@pytest.mark.parametrize("N", [4, 5, 12])
def test_diagonals_match_dense_L_squared(N, bc):
    sigma = 0.37
    L = pin.second_difference(N, bc)
    A = np.eye(N) + sigma * (L @ L)
    assert np.allclose(pin.dense_from_diagonals(*pin.diagonals_I_plus_sigma_L2(N, sigma, bc)),
                       A, atol=1e-15)
    assert np.allclose(A, A.T)
    if bc == "zeroflux":
        assert np.allclose(L.sum(axis=0), 0.0)          # 1^T L = 0  (C-13)
        assert np.allclose(A.sum(axis=0), 1.0, atol=1e-15)


def test_per_system_diagonals_broadcast():
    sig = np.array([0.1, 3.0, 10.0])
    d3 = pin.diagonals_I_plus_sigma_L2(9, sig)
    for i, s in enumerate(sig):
        for v3, v1 in zip(d3, pin.diagonals_I_plus_sigma_L2(9, float(s))):
            assert np.array_equal(v3[:, i], v1)


def test_generator_is_counter_based():
    """A window of systems drawn alone equals the same window of the full batch."""
    full = pin.uniform_pm1(3, 0, 16, 40)
    part = pin.uniform_pm1(3, 0, 16, 10, col0=20, Mtot=40)
    assert np.array_equal(full[:, 20:30], part)
    g = pin.normal01(2, 2, 64, 512)
    assert abs(g.mean()) < 0.02 and abs(g.std() - 1.0) < 0.02
    u = pin.uniform_pm1(5, 0, 64, 512)
    assert u.min() >= -1.0 and u.max() < 1.0 and abs(u.mean()) < 0.02
    assert not np.array_equal(pin.uniform_pm1(5, 1, 4, 4), pin.uniform_pm1(5, 0, 4, 4))


def test_workload_recipes():
    w = WORKLOADS["cfg2"]
    f, x = make_rhs(w, M=8)
    A = pin.dense_from_diagonals(*make_matrix(w))
    assert np.allclose(A @ x, f, rtol=0, atol=1e-12)
    assert np.allclose(banded_matvec(*pin.random_diag_dominant(1, 9), np.eye(9)),
                       pin.dense_from_diagonals(*pin.random_diag_dominant(1, 9)))
    c0 = make_rhs(WORKLOADS["cfg4"], M=16)
    assert np.all(np.abs(c0.mean(axis=0)) < 0.52) and np.all(np.abs(c0 - c0.mean(axis=0)) < 0.11)
    assert abs(SIGMA_CH - 10995.11627776) < 1e-6 and abs(R_CH - 1.048576) < 1e-12
    s = sine_modes(8)
    assert np.allclose(s.T @ s, 4.5 * np.eye(8), atol=1e-12)    # orthogonal modes


# ---- right-hand sides against dense linear algebra ---------------------------------------------
@pytest.mark.parametrize("bc,bcname", [(0, "dirichlet"), (1, "zeroflux")])
def test_rhs_against_dense(bc, bcname):
    N, sigma, r = 24, 3.7, 0.9
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, bcname)
    fac = oracle.factor(*diags)
    L = pin.second_difference(N, bcname)
    C = 0.3 + 0.5 * pin.uniform_pm1(40, 0, N, 1)[:, 0]
    w = C ** 3 - C
    direct = oracle.rhs(fac, 0, bc, 0, r, sigma, C)
    assert np.max(np.abs(direct - (C + r * (L @ w)))) <= 1e-14
    incr = oracle.rhs(fac, 0, bc, 1, r, sigma, C)
    assert np.max(np.abs(incr - L @ (r * w - sigma * (L @ C)))) <= 1e-12
    hyper = oracle.rhs(fac, 1, bc, 0, 0.0, 0.0, C)
    A = pin.dense_from_diagonals(*diags)
    assert np.max(np.abs(hyper - (2 * np.eye(N) - A) @ C)) <= 1e-13


def test_hyper_rhs_uses_general_nonsymmetric_diagonals():
    N = 17
    diags = pin.random_diag_dominant(8, N)
    fac = oracle.factor(*diags)
    C = pin.uniform_pm1(41, 0, N, 1)[:, 0]
    A = pin.dense_from_diagonals(*diags)
    assert np.max(np.abs(oracle.rhs(fac, 1, 0, 0, 0, 0, C) - (2 * np.eye(N) - A) @ C)) <= 1e-14


# ---- one full step against a dense LAPACK solve ------------------------------------------------
@pytest.mark.parametrize("bc,bcname", [(0, "dirichlet"), (1, "zeroflux")])
@pytest.mark.parametrize("form", [0, 1])
def test_ch_step_against_dense_solve(bc, bcname, form):
    N, M, sigma, r = 32, 5, 40.0, 1.05
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, bcname)
    fac = oracle.factor(*diags)
    L = pin.second_difference(N, bcname)
    A = np.eye(N) + sigma * (L @ L)
    c0 = 0.2 + 0.05 * pin.uniform_pm1(42, 0, N, M)
    ref = np.linalg.solve(A, c0 + r * (L @ (c0 ** 3 - c0)))       # the scheme's definition
    got = oracle.step_batch(fac, 0, bc, form, r, sigma, c0, 1)
    assert np.max(np.abs(got - ref)) <= 5e-12
    two = oracle.step_batch(fac, 0, bc, form, r, sigma, c0, 2)
    ref2 = np.linalg.solve(A, ref + r * (L @ (ref ** 3 - ref)))
    assert np.max(np.abs(two - ref2)) <= 1e-11


def test_hyperdiffusion_cn_amplification():
    """Dirichlet sine mode k is an eigenvector: one CN step multiplies it by
    (2 - lam_k)/lam_k,  lam_k = 1 + 16 sigma sin^4(pi k/(2(N+1)))."""
    N, sigma = 48, 0.8
    fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(N, sigma))
    modes = sine_modes(N)
    out = oracle.step_batch(fac, 1, 0, 0, 0.0, 0.0, modes, 3)
    k = np.arange(1, N + 1)
    lam = 1 + 16 * sigma * np.sin(np.pi * k / (2 * (N + 1))) ** 4
    assert np.max(np.abs(out - modes * ((2 - lam) / lam)[None, :] ** 3)) <= 1e-13


# ---- P10: conservation of the mean (zero-flux, increment form) -----------------------------------
def test_p10_mean_conservation_and_positive_pivots():
    N, M = 256, 6
    sigma = 1e-2 * 1e-6 * N ** 4
    r = 1e-6 * N ** 2
    fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(N, sigma, "zeroflux"))
    assert np.all(fac.alpha > 0)
    m = pin.uniform_vec(4, 5, M, -0.5, 0.5)
    c0 = m[None, :] + 0.05 * pin.uniform_pm1(4, 0, N, M)
    c = oracle.step_batch(fac, 0, 1, 1, r, sigma, c0, 200)
    import math
    for i in range(M):
        m0 = math.fsum(c0[:, i]) / N
        m1 = math.fsum(c[:, i]) / N
        assert abs(m1 - m0) <= 1e-12
    # the state really evolved
    assert np.max(np.abs(c - c0)) > 1e-3
