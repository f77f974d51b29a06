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


# ---- forced Cahn-Hilliard, PAPER.md:63-67 (Remark 1, Eq. 3); reading C-22 -------------------------
def test_forcing_definition_and_zero_mean():
    """Phi = mu1 cos(2 pi (x - mu2 t)) at the cell centres x_k = (k + 1/2)/N: retyped here from the reading,
    zero discrete mean (so the zero-flux scheme still conserves mean(C)), period 1/mu2 in time."""
    N = 48
    x = (np.arange(N) + 0.5) / N
    for t, mu1, mu2 in ((0.0, 1.0, 0.0), (0.3, 2.5, 1.75), (1e-3, -0.4, 20.0)):
        phi = oracle.forcing(N, t, mu1, mu2)
        assert np.max(np.abs(phi - mu1 * np.cos(2 * np.pi * x - 2 * np.pi * mu2 * t))) <= 1e-14 * max(1.0, abs(mu1))
        assert abs(phi.sum()) <= 1e-13 * abs(mu1) * N
    assert np.allclose(oracle.forcing(N, 0.25, 1.0, 2.0), oracle.forcing(N, 0.75, 1.0, 2.0), atol=1e-14)


def test_forced_step_dense_definition_one_step():
    """One forced step = the dense-matrix definition A c+ = c + r L (c^3 - c) + dt Phi(t0) (LAPACK solve)."""
    N, M = 24, 5
    sigma, r, dt, t0 = 3.0, 0.8, 2e-3, 0.37
    for bc, bcname in ((1, "zeroflux"), (0, "dirichlet")):
        diags = pin.diagonals_I_plus_sigma_L2(N, sigma, bcname)
        A = pin.dense_from_diagonals(*diags)
        L = pin.second_difference(N, bcname)
        c0 = 0.2 + 0.05 * pin.uniform_pm1(60, 0, N, M)
        mu1 = pin.uniform_vec(60, 1, M, 0.5, 5.0)
        mu2 = pin.uniform_vec(60, 2, M, -3.0, 3.0)
        x = (np.arange(N) + 0.5) / N
        want = np.empty_like(c0)
        for i in range(M):
            phi = mu1[i] * np.cos(2 * np.pi * (x - mu2[i] * t0))
            want[:, i] = np.linalg.solve(A, c0[:, i] + r * (L @ (c0[:, i] ** 3 - c0[:, i])) + dt * phi)
        fac = oracle.factor(*diags)
        for form in (0, 1):
            got = oracle.step_forced_batch(fac, bc, form, r, sigma, dt, t0, mu1, mu2, c0, 1)
            assert np.max(np.abs(got - want)) <= 1e-13


def test_forced_step_reduces_to_unforced_and_time_advances():
    N, M = 40, 3
    sigma, r = 2.0, 0.5
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, "zeroflux")
    fac = oracle.factor(*diags)
    c0 = 0.1 + 0.05 * pin.uniform_pm1(61, 0, N, M)
    z = np.zeros(M)
    a = oracle.step_forced_batch(fac, 1, 1, r, sigma, 1e-3, 0.0, z, z + 7.0, c0, 4)
    assert np.array_equal(a, oracle.step_batch(fac, 0, 1, 1, r, sigma, c0, 4))          # mu1 = 0: no forcing
    # 5 steps from t0 == 2 steps from t0, then 3 steps from t0 + 2 dt (step n is taken at t0 + n dt)
    mu1, mu2, dt = z + 3.0, z + 11.0, 1e-3
    five = oracle.step_forced_batch(fac, 1, 1, r, sigma, dt, 0.2, mu1, mu2, c0, 5)
    two = oracle.step_forced_batch(fac, 1, 1, r, sigma, dt, 0.2, mu1, mu2, c0, 2)
    assert np.array_equal(five, oracle.step_forced_batch(fac, 1, 1, r, sigma, dt, 0.2 + 2 * dt, mu1, mu2, two, 3))


def test_forced_step_exact_quadrature_when_the_pde_terms_are_off():
    """sigma = 0, r = 0 => A = I and the scheme is c_{n+1} = c_n + dt Phi(t_n): after K steps
    c_K = c_0 + dt sum_n Phi(x, t0 + n dt), and the sum of the cosines has the closed form
    sum_{n<K} cos(th - n ph) = sin(K ph / 2) / sin(ph / 2) * cos(th - (K - 1) ph / 2)."""
    N, M, K = 32, 4, 200
    one, zero = np.ones(N), np.zeros(N)
    fac = oracle.factor(zero, zero, one, zero, zero)            # A = I
    c0 = pin.uniform_pm1(62, 0, N, M)
    mu1 = np.array([1.0, -2.0, 0.5, 3.0])
    mu2 = np.array([0.7, 5.0, -13.0, 40.0])
    dt, t0 = 2.5e-3, 0.1
    got = oracle.step_forced_batch(fac, 1, 0, 0.0, 0.0, dt, t0, mu1, mu2, c0, K)
    x = (np.arange(N) + 0.5) / N
    for i in range(M):
        th = 2 * np.pi * (x - mu2[i] * t0)
        ph = 2 * np.pi * mu2[i] * dt
        s = np.sin(K * ph / 2) / np.sin(ph / 2) * np.cos(th - (K - 1) * ph / 2)
        assert np.max(np.abs(got[:, i] - (c0[:, i] + dt * mu1[i] * s))) <= 1e-13


def test_forced_step_steady_cosine_mode_closed_form():
    """r = 0, mu2 = 0, c_0 = 0: Phi = mu1 cos(2 pi x_k) is the k = 2 zero-flux cosine mode, an eigenvector of
    A = I + sigma L_N^2 with lambda = 1 + 16 sigma sin^4(pi / N); so c_n = mu1 dt cos(2 pi x) sum_{j=1..n} lambda^-j."""
    N, n, sigma, dt, mu1 = 64, 12, 40.0, 1e-2, 1.5
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, "zeroflux")
    fac = oracle.factor(*diags)
    got = oracle.step_forced_batch(fac, 1, 0, 0.0, sigma, dt, 0.0, np.array([mu1]), np.array([0.0]), np.zeros((N, 1)), n)
    lam = 1.0 + 16.0 * sigma * np.sin(np.pi / N) ** 4
    x = (np.arange(N) + 0.5) / N
    want = mu1 * dt * np.cos(2 * np.pi * x) * sum(lam ** -j for j in range(1, n + 1))
    assert np.max(np.abs(got[:, 0] - want)) <= 1e-13 * np.max(np.abs(want)) * (1 + 16 * sigma)


def test_forced_zero_flux_step_conserves_the_mean():
    import math
    N, M = 128, 6
    sigma, r = 1e-2 * 1e-6 * N ** 4, 1e-6 * N ** 2
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, "zeroflux")
    c0 = pin.uniform_vec(63, 5, M, -0.5, 0.5)[None, :] + 0.05 * pin.uniform_pm1(63, 0, N, M)
    mu1 = pin.uniform_vec(63, 1, M, 10.0, 1000.0)
    mu2 = pin.uniform_vec(63, 2, M, -1e4, 1e4)
    c1 = oracle.step_forced_batch(oracle.factor(*diags), 1, 1, r, sigma, 1e-6, 0.0, mu1, mu2, c0, 300)
    for i in range(M):
        assert abs(math.fsum(c1[:, i]) - math.fsum(c0[:, i])) / N <= 1e-13
    assert np.max(np.abs(c1 - oracle.step_batch(oracle.factor(*diags), 0, 1, 1, r, sigma, c0, 300))) > 1e-6   # the forcing acts
