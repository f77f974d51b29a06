"""PAPER.md:96 (Remark 3): "A finite-difference approximation of the Heat Equation with Crank-Nicolson temporal
discretisation and high-order accurate spatial discretisation (nearest and next-nearest neighbours) also produces a
pentadiagonal problem that can be solved with the methods developed herein."  SURVEY.md section 8(f) NEXT-4.
The generator pent_inputs.heat4_cn_diagonals writes that matrix out; these CPU tests pin it and the oracle on it by
closed forms: A = I + s_h (L^2 - 12 L), so the Dirichlet sine modes / periodic Fourier modes are eigenvectors."""
import numpy as np
import pytest

import oracle
import pent_inputs as pin


def _normwise(x, ref):
    return float(np.max(np.abs(x - ref)) / np.max(np.abs(ref)))


def test_generator_is_the_fourth_order_stencil():
    N, s = 11, 0.37
    L = pin.second_difference(N, "dirichlet")
    A = np.eye(N) + s * (L @ L - 12.0 * L)
    assert np.allclose(pin.dense_from_diagonals(*pin.heat4_cn_diagonals(N, s)), A, atol=1e-14)
    # interior row = I - (dt/2) * (-1, 16, -30, 16, -1)/(12 dx^2), s = dt/(24 dx^2)
    assert np.allclose(A[5, 3:8], [s, -16 * s, 1 + 30 * s, -16 * s, s])
    Ap = pin.dense_from_periodic_diagonals(*pin.heat4_cn_diagonals(N, s, "periodic"))
    assert np.allclose(Ap[0, [N - 2, N - 1, 0, 1, 2]], [s, -16 * s, 1 + 30 * s, -16 * s, s])
    # the stencil differentiates x^2, x^3, x^4 exactly to fourth order: (12L - L^2)/12 applied to k^4 gives 12 k^2
    k = np.arange(N, dtype=float)
    D = (12.0 * L - L @ L) / 12.0
    assert np.allclose((D @ k ** 4)[3:-3], 12.0 * k[3:-3] ** 2)


@pytest.mark.parametrize("N,s", [(64, 0.8), (255, 40.0)])
def test_solve_sine_modes_closed_form(N, s):
    """lambda_k = 1 + s (mu_k^2 + 12 mu_k), mu_k = 4 sin^2(pi k / (2(N+1))) (eigenvalue of -L)."""
    fac = oracle.factor(*pin.heat4_cn_diagonals(N, s))
    j = np.arange(1, N + 1)
    for k in (1, 2, N // 3, N - 1, N):
        f = np.sin(np.pi * ((k * j) % (2 * (N + 1))) / (N + 1))
        mu = 4.0 * np.sin(np.pi * k / (2 * (N + 1))) ** 2
        lam = 1.0 + s * (mu * mu + 12.0 * mu)
        assert _normwise(oracle.solve(fac, f), f / lam) <= 50 * (1 + 64 * s) * 1.2e-16


def test_crank_nicolson_amplification_and_fourth_order_convergence():
    """One step multiplies sine mode k by (2 - lambda_k)/lambda_k; with dt tiny, the decay of mode 1 over T
    approaches exp(-pi^2 T) like dx^4 (the stencil's order; the paper's hyperdiffusion scheme is dx^2)."""
    T, errs, Ns = 0.05, [], [8, 16, 32, 64]
    for N in Ns:
        dx = 1.0 / (N + 1)
        steps = 2000
        dt = T / steps
        s = dt / (24.0 * dx * dx)
        diags = pin.heat4_cn_diagonals(N, s)
        fac = oracle.factor(*diags)
        x = np.arange(1, N + 1) * dx
        c0 = np.sin(np.pi * x)[:, None]
        c = oracle.step_batch(fac, 1, 0, 0, 0.0, 0.0, c0, steps)
        mu = 4.0 * np.sin(np.pi / (2 * (N + 1))) ** 2
        lam = 1.0 + s * (mu * mu + 12.0 * mu)
        assert _normwise(c[:, 0], ((2.0 - lam) / lam) ** steps * c0[:, 0]) <= 1e-11
        errs.append(np.max(np.abs(c[:, 0] - np.exp(-np.pi ** 2 * T) * c0[:, 0])))
    slope = np.polyfit(np.log(Ns), np.log(errs), 1)[0]
    assert -4.4 <= slope <= -3.7, slope


def test_periodic_heat_matrix_circulant_spectrum():
    N, s = 48, 3.0
    diags = pin.heat4_cn_diagonals(N, s, "periodic")
    pf = oracle.factor_periodic(*diags)
    j = np.arange(N)
    for m in (0, 1, 5, N // 2):
        th = 2 * np.pi * m / N
        f = np.cos(th * j + 0.3)[:, None]
        lam = 1.0 + s * (30.0 - 32.0 * np.cos(th) + 2.0 * np.cos(2 * th))
        assert _normwise(oracle.solve_periodic_batch(pf, f)[:, 0], f[:, 0] / lam) <= 1e-12
