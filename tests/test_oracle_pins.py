"""Pins for the CPU oracle (oracle/pent_oracle.c): each test ties it to something
other than itself -- brute force, exact rational arithmetic, closed forms, a LAPACK
routine, algebraic invariants.  A dropped term, wrong sign/index or transposed
operand in the oracle fails at least one of them.  CPU only.

Citations: PAPER.md:167-242 (algorithm), north_star (dense GE, sine-mode closed form,
manufactured f = A x), SURVEY.md §8(c) pins P1-P10.
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import pent_inputs as pin
from pent_inputs.configs import banded_matvec


def _normwise(x, ref):
    return np.max(np.abs(x - ref)) / np.max(np.abs(ref))


def _fraction_solve(A, f):
    """Exact Gauss-Jordan elimination in rational arithmetic (row swaps on zero pivot)."""
    n = len(f)
    M = [[Fraction(float(A[i][j])) for j in range(n)] + [Fraction(float(f[i]))] for i in range(n)]
    for k in range(n):
        p = next(i for i in range(k, n) if M[i][k] != 0)
        M[k], M[p] = M[p], M[k]
        piv = M[k][k]
        M[k] = [v / piv for v in M[k]]
        for i in range(n):
            if i != k and M[i][k] != 0:
                m = M[i][k]
                M[i] = [vi - m * vk for vi, vk in zip(M[i], M[k])]
    return np.array([float(M[i][n]) for i in range(n)])


# ---- P1: brute force on tiny N, non-symmetric matrices (catches b<->d, a<->e swaps) -----
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 7, 8, 16, 33])
def test_p1_dense_ge_and_exact_rational(N):
    a, b, c, d, e = pin.random_diag_dominant(100 + N, N)
    A = pin.dense_from_diagonals(a, b, c, d, e)
    f = pin.uniform_pm1(200 + N, 0, N, 1)[:, 0]
    fac = oracle.factor(a, b, c, d, e)
    x = oracle.solve(fac, f)
    x_ge = oracle.dense_ge(A, f)
    assert np.max(np.abs(x - x_ge)) <= 4e-15
    if N <= 8:
        x_exact = _fraction_solve(A, f)
        assert np.max(np.abs(x - x_exact)) <= 4e-15
        assert np.max(np.abs(x_ge - x_exact)) <= 4e-15
    # and against numpy's LAPACK dgesv, a third party
    assert np.max(np.abs(x - np.linalg.solve(A, f))) <= 4e-15


def test_p1_dense_ge_needs_pivoting():
    """The second oracle really pivots: a matrix with a zero leading entry."""
    A = np.array([[0.0, 2.0, 1.0], [1.0, 1.0, 0.0], [3.0, 0.0, 1.0]])
    f = np.array([1.0, 2.0, 3.0])
    assert np.allclose(oracle.dense_ge(A, f), np.linalg.solve(A, f), atol=1e-15)


# ---- P2: L R == A ------------------------------------------------------------------------
@pytest.mark.parametrize("N", [4, 5, 9, 64])
def test_p2_reconstruction(N):
    a, b, c, d, e = pin.random_diag_dominant(7 + N, N)
    fac = oracle.factor(a, b, c, d, e)
    L = np.zeros((N, N)); R = np.eye(N)
    for k in range(N):
        L[k, k] = fac.alpha[k]
        if k >= 1: L[k, k - 1] = fac.beta[k]
        if k >= 2: L[k, k - 2] = fac.eps[k]
        if k + 1 < N: R[k, k + 1] = fac.gamma[k]
        if k + 2 < N: R[k, k + 2] = fac.delta[k]
    A = pin.dense_from_diagonals(a, b, c, d, e)
    assert np.max(np.abs(L @ R - A)) <= 2e-15 * np.max(np.abs(A))


# ---- P3: closed-form eigenpairs (north_star) ------------------------------------------------
@pytest.mark.parametrize("N,sigma", [(64, 0.1), (33, 10.0), (128, 1.0)])
def test_p3_sine_modes_dirichlet(N, sigma):
    """A = I + sigma L^2 (Dirichlet): sin(pi k j/(N+1)) is an eigenvector with eigenvalue
    1 + 16 sigma sin^4(pi k / (2(N+1)))."""
    fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(N, sigma, "dirichlet"))
    j = np.arange(1, N + 1)
    for k in range(1, N + 1):
        f = np.sin(np.pi * ((k * j) % (2 * (N + 1))) / (N + 1))   # exact argument reduction
        lam = 1.0 + 16.0 * sigma * np.sin(np.pi * k / (2 * (N + 1))) ** 4
        # forward-error bound ~ cond(A) * eps, cond(A) <= 1 + 16 sigma (the eigenvalue range)
        assert _normwise(oracle.solve(fac, f), f / lam) <= (8 * (1 + 16 * sigma) + 100) * 1.2e-16
    if (N, sigma) == (64, 0.1):   # SURVEY.md P3 values
        assert abs(1 + 16 * sigma * np.sin(np.pi / 130) ** 4 - 1.0000005454776684) < 1e-15


@pytest.mark.parametrize("N,sigma", [(64, 0.1), (48, 1.0e4)])
def test_p3prime_cosine_modes_zeroflux(N, sigma):
    """Zero-flux L_N: cos(pi k (j+1/2)/N) is an eigenvector of I + sigma L_N^2 with
    eigenvalue 1 + 16 sigma sin^4(pi k/(2N)), k = 0..N-1 (k=0: constants, eigenvalue 1)."""
    fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(N, sigma, "zeroflux"))
    j = np.arange(N)
    for k in range(N):
        f = np.cos(np.pi * ((k * (2 * j + 1)) % (4 * N)) / (2 * N))   # = cos(pi k (j+1/2)/N)
        lam = 1.0 + 16.0 * sigma * np.sin(np.pi * k / (2 * N)) ** 4
        assert _normwise(oracle.solve(fac, f), f / lam) <= (8 * (1 + 16 * sigma) + 100) * 1.2e-16


# ---- P4: manufactured solution -------------------------------------------------------------
def test_p4_manufactured():
    N, M, sigma = 512, 8, 1.0
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma)
    x = pin.normal01(2, 2, N, M)
    f = banded_matvec(*diags, x)
    xs = oracle.solve_batch(oracle.factor(*diags), f)
    for i in range(M):
        assert _normwise(xs[:, i], x[:, i]) <= 1e-14


# ---- P5: reductions to textbook routines -----------------------------------------------------
def _thomas(b, c, d, f):
    """Independent 3-term Thomas algorithm (b sub, c main, d super; row-indexed)."""
    n = len(c)
    cp = np.zeros(n); fp = np.zeros(n)
    cp[0] = d[0] / c[0]; fp[0] = f[0] / c[0]
    for k in range(1, n):
        m = c[k] - b[k] * cp[k - 1]
        cp[k] = d[k] / m if k + 1 < n else 0.0
        fp[k] = (f[k] - b[k] * fp[k - 1]) / m
    x = np.zeros(n); x[-1] = fp[-1]
    for k in range(n - 2, -1, -1):
        x[k] = fp[k] - cp[k] * x[k + 1]
    return x


def test_p5_tridiagonal_and_diagonal():
    N = 40
    a, b, c, d, e = pin.random_diag_dominant(5, N)
    z = np.zeros(N)
    f = pin.uniform_pm1(6, 0, N, 1)[:, 0]
    x = oracle.solve(oracle.factor(z, b, c, d, z), f)
    assert np.max(np.abs(x - _thomas(b, c, d, f))) <= 1e-15
    x = oracle.solve(oracle.factor(z, z, c, z, z), f)
    assert np.max(np.abs(x - f / c)) == 0.0


# ---- P6: LAPACK banded solver (pivoted) at full N -------------------------------------------
@pytest.mark.parametrize("N,sigma,bc", [(64, 0.1, "dirichlet"), (512, 1.0, "dirichlet"),
                                        (1024, 10.0, "dirichlet"), (4096, 0.5, "dirichlet"),
                                        (1024, 10995.11627776, "zeroflux")])
def test_p6_lapack_banded(N, sigma, bc):
    from scipy.linalg import solve_banded
    a, b, c, d, e = pin.diagonals_I_plus_sigma_L2(N, sigma, bc)
    ab = np.zeros((5, N))
    ab[0, 2:] = e[:-2]; ab[1, 1:] = d[:-1]; ab[2] = c; ab[3, :-1] = b[1:]; ab[4, :-2] = a[2:]
    f = pin.uniform_pm1(9, 0, N, 4)
    ref = solve_banded((2, 2), ab, f)
    xs = oracle.solve_batch(oracle.factor(a, b, c, d, e), f)
    tol = 1e-11 if sigma > 100 else 2e-14
    for i in range(4):
        assert _normwise(xs[:, i], ref[:, i]) <= tol


def test_p6_lapack_banded_nonsymmetric():
    from scipy.linalg import solve_banded
    N = 257
    a, b, c, d, e = pin.random_diag_dominant(31, N)
    ab = np.zeros((5, N))
    ab[0, 2:] = e[:-2]; ab[1, 1:] = d[:-1]; ab[2] = c; ab[3, :-1] = b[1:]; ab[4, :-2] = a[2:]
    f = pin.uniform_pm1(32, 0, N, 1)[:, 0]
    x = oracle.solve(oracle.factor(a, b, c, d, e), f)
    assert _normwise(x, solve_banded((2, 2), ab, f)) <= 1e-14


# ---- P7: LDL^T structure for symmetric A ----------------------------------------------------
def test_p7_symmetric_invariants():
    fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(300, 10.0))
    al, be, ep, ga, de = fac.alpha, fac.beta, fac.eps, fac.gamma, fac.delta
    assert np.max(np.abs(be[1:] - al[:-1] * ga[:-1])) <= 1e-13 * np.max(np.abs(be))
    assert np.max(np.abs(ep[2:] - al[:-2] * de[:-2])) <= 1e-13 * np.max(np.abs(ep))
    assert np.all(al > 0)          # SPD => positive pivots


# ---- P8: Toeplitz-interior fixed point -------------------------------------------------------
def test_p8_toeplitz_fixed_point():
    """Mid-array factors of I + sigma L^2 converge to the solution of
    alpha*delta = sigma, alpha*gamma*(1+delta) = -4 sigma, alpha(1+gamma^2+delta^2) = 1+6 sigma.
    For sigma = 1/2: alpha = 3/2 + sqrt 2, gamma = sqrt 2 - 2, delta = 3 - 2 sqrt 2,
    beta = -(1 + sqrt 2 / 2)   (closed form)."""
    fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(4096, 0.5))
    m = 2048
    s2 = np.sqrt(2.0)
    assert abs(fac.alpha[m] - (1.5 + s2)) <= 1e-14
    assert abs(fac.gamma[m] - (s2 - 2.0)) <= 1e-14
    assert abs(fac.delta[m] - (3.0 - 2.0 * s2)) <= 1e-14
    assert abs(fac.beta[m] + (1.0 + s2 / 2.0)) <= 1e-14
    for sigma in (10.0, 0.1):
        fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(1024, sigma))
        al, ga, de = fac.alpha[512], fac.gamma[512], fac.delta[512]
        assert abs(al * de - sigma) <= 1e-13 * sigma
        assert abs(al * ga * (1 + de) + 4 * sigma) <= 1e-12 * sigma
        assert abs(al * (1 + ga * ga + de * de) - (1 + 6 * sigma)) <= 1e-12 * (1 + 6 * sigma)


def test_p9_first_rows_rational():
    """First factor rows of the cfg1 matrix (sigma = 1/10) from exact rationals:
    alpha_0 = 1+5s = 3/2, gamma_0 = -4s/alpha_0 = -4/15, delta_0 = s/alpha_0 = 1/15,
    beta_1 = -4s, alpha_1 = 1+6s - beta_1*gamma_0 = 8/5 - 8/75 = 112/75."""
    fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(64, 0.1))
    assert abs(fac.alpha[0] - 1.5) <= 1e-16
    assert abs(fac.gamma[0] + 4.0 / 15.0) <= 1e-16
    assert abs(fac.delta[0] - 1.0 / 15.0) <= 1e-16
    assert abs(fac.beta[1] + 0.4) <= 1e-16
    assert abs(fac.alpha[1] - 112.0 / 75.0) <= 3e-16


# ---- error behaviour -------------------------------------------------------------------------
def test_zero_pivot_reported():
    N = 8
    a, b, c, d, e = pin.random_diag_dominant(3, N)
    c = c.copy(); c[0] = 0.0
    with pytest.raises(oracle.SingularPivot) as ei:
        oracle.factor(a, b, c, d, e)
    assert ei.value.row == 0
    # a pivot that cancels exactly at row 1: alpha_1 = c_1 - b_1 d_0 / c_0
    a, b, c, d, e = (np.array(v, dtype=float) for v in
                     ([0, 0, 1, 1], [0, 2, 1, 1], [4, 1, 5, 5], [2, 1, 1, 0], [1, 1, 0, 0]))
    with pytest.raises(oracle.SingularPivot) as ei:
        oracle.factor(a, b, c, d, e)
    assert ei.value.row == 1


def test_batch_layout_and_threads():
    """Interleaved wrapper == per-system solves; OpenMP variant is bit-identical."""
    N, M = 37, 19
    diags = pin.random_diag_dominant(77, N)
    fac = oracle.factor(*diags)
    f = pin.uniform_pm1(78, 0, N, M)
    x1 = oracle.solve_batch(fac, f, nthreads=1)
    x4 = oracle.solve_batch(fac, f, nthreads=4)
    assert np.array_equal(x1, x4)
    for i in (0, 7, M - 1):
        assert np.array_equal(x1[:, i], oracle.solve(fac, f[:, i].copy()))


def test_per_system_variant_matches_shared():
    N, M = 64, 12
    sig = pin.uniform_vec(6, 1, M, 0.1, 10.0)
    diags = pin.diagonals_I_plus_sigma_L2(N, sig)
    f = pin.uniform_pm1(6, 0, N, M)
    x, info = oracle.factor_solve_batch(*diags, f)
    assert not info.any()
    for i in (0, 5, M - 1):
        fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(N, float(sig[i])))
        assert np.array_equal(x[:, i], oracle.solve(fac, f[:, i].copy()))
    # a singular system is flagged and the others are unaffected
    diags2 = [v.copy() for v in diags]
    diags2[2][0, 3] = 0.0
    x2, info2 = oracle.factor_solve_batch(*diags2, f)
    assert info2[3] == 1 and info2.sum() == 1
    assert np.array_equal(np.delete(x2, 3, axis=1), np.delete(x, 3, axis=1))
