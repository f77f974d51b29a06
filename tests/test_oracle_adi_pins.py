"""Pins for the 2-D ADI oracle (oracle/pent_oracle_adi.c, reading C-23).  CPU only.
* the dense definition on a tiny grid: one Peaceman-Rachford step equals
  (A_y (x) A_x)^{-1} ((2I - A_y) (x) (2I - A_x)) u, assembled with Kronecker products and solved by LAPACK
  (non-symmetric A_x != A_y, Nx != Ny: catches any axis / transpose mix-up);
* the product of the two 1-D Crank-Nicolson amplification factors on a tensor-product eigenmode;
* the 2-D heat equation u_t = u_xx + u_yy with the Remark-3 matrices: decay exp(-2 pi^2 t) of
  sin(pi x) sin(pi y), second order in time."""
import numpy as np
import pytest

import oracle
import pent_inputs as pin


def test_adi_step_dense_kronecker_definition():
    Nx, Ny = 7, 5
    dgx, dgy = pin.random_diag_dominant(901, Nx), pin.random_diag_dominant(902, Ny)
    Ax, Ay = pin.dense_from_diagonals(*dgx), pin.dense_from_diagonals(*dgy)
    u = pin.uniform_pm1(903, 0, Ny, Nx)
    Ix, Iy = np.eye(Nx), np.eye(Ny)
    # vec index = y * Nx + x: an operator along x is I_y (x) A_x, along y it is A_y (x) I_x
    lhs = np.kron(Ay, Ix) @ np.kron(Iy, Ax)
    rhs = np.kron(2 * Iy - Ay, Ix) @ np.kron(Iy, 2 * Ix - Ax)
    for steps in (1, 3):
        want = u.reshape(-1).copy()
        for _ in range(steps):
            want = np.linalg.solve(lhs, rhs @ want)
        got = oracle.adi_steps(oracle.factor(*dgx), oracle.factor(*dgy), u, steps)
        assert np.max(np.abs(got.reshape(-1) - want)) <= 1e-13


def test_adi_half_steps_in_the_stated_order():
    """Half step 1 is explicit along y / implicit along x (not the other way round): for A_y = I the step
    reduces to the 1-D kind-1 step along every row, for A_x = I to the 1-D step along every column."""
    Nx, Ny = 12, 9
    dgx, dgy = pin.random_diag_dominant(904, Nx), pin.random_diag_dominant(905, Ny)
    ident = lambda N: (np.zeros(N), np.zeros(N), np.ones(N), np.zeros(N), np.zeros(N))
    u = pin.uniform_pm1(906, 0, Ny, Nx)
    fx, fy = oracle.factor(*dgx), oracle.factor(*dgy)
    got = oracle.adi_steps(fx, oracle.factor(*ident(Ny)), u, 2)
    want = oracle.step_batch(fx, 1, 0, 0, 0.0, 0.0, np.ascontiguousarray(u.T), 2).T      # rows of u = systems
    assert np.max(np.abs(got - want)) <= 1e-14
    got = oracle.adi_steps(oracle.factor(*ident(Nx)), fy, u, 2)
    want = oracle.step_batch(fy, 1, 0, 0, 0.0, 0.0, u, 2)                                 # columns of u = systems
    assert np.max(np.abs(got - want)) <= 1e-14


def test_adi_amplification_factor_and_heat_equation_decay():
    Nx, Ny = 48, 40
    hx, hy = 1.0 / (Nx + 1), 1.0 / (Ny + 1)
    x = np.arange(1, Nx + 1) * hx
    y = np.arange(1, Ny + 1) * hy
    u0 = np.outer(np.sin(np.pi * y), np.sin(np.pi * x))
    T, errs = 0.02, []
    for steps in (10, 20, 40):
        dt = T / steps
        sx, sy = dt / (24 * hx * hx), dt / (24 * hy * hy)
        fx, fy = oracle.factor(*pin.heat4_cn_diagonals(Nx, sx)), oracle.factor(*pin.heat4_cn_diagonals(Ny, sy))
        got = oracle.adi_steps(fx, fy, u0, steps)
        mux, muy = 4 * np.sin(np.pi * hx / 2) ** 2, 4 * np.sin(np.pi * hy / 2) ** 2
        lx, ly = 1 + sx * (mux * mux + 12 * mux), 1 + sy * (muy * muy + 12 * muy)
        amp = ((2 - lx) / lx * (2 - ly) / ly) ** steps
        assert np.max(np.abs(got - amp * u0)) <= 1e-13
        errs.append(abs(amp - np.exp(-2 * np.pi ** 2 * T)))
    # Peaceman-Rachford is second order in time (the spatial error of the fourth-order stencil is far below)
    assert 3.5 <= errs[0] / errs[1] <= 4.5 and 3.5 <= errs[1] / errs[2] <= 4.5
