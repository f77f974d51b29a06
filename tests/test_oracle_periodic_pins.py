"""Pins of the PERIODIC oracle (oracle/pent_oracle_periodic.c; Eqs. 7a-12, and the
validation of section II.E).  None of them re-types the oracle's formula: dense
LAPACK solves of the assembled cyclic matrix, the closed-form spectrum of a circulant matrix, the
Crank-Nicolson amplification factor, the analytic solution Eq. 14 and the slope the paper prints."""
import os

import numpy as np
import pytest

import oracle
import pent_inputs as pin

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_fig2_slope.txt")


def normwise(x, ref):
    return float(np.max(np.max(np.abs(x - ref), axis=0) / np.max(np.abs(ref), axis=0)))


@pytest.mark.parametrize("N", [6, 7, 8, 9, 16, 33, 40])
def test_dense_lapack_nonsymmetric(N):
    dg = pin.random_periodic_diag_dominant(100 + N, N)
    A = pin.dense_from_periodic_diagonals(*dg)
    f = pin.uniform_pm1(200 + N, 0, N, 7)
    x = oracle.solve_periodic_batch(oracle.factor_periodic(*dg), f)
    assert normwise(x, np.linalg.solve(A, f)) <= 1e-14


def test_own_dense_elimination_tiny():
    N = 6
    dg = pin.random_periodic_diag_dominant(3, N)
    A = pin.dense_from_periodic_diagonals(*dg)
    f = pin.uniform_pm1(4, 0, N, 1)
    x = oracle.solve_periodic_batch(oracle.factor_periodic(*dg), f)[:, 0]
    assert np.max(np.abs(x - oracle.dense_ge(A, f[:, 0]))) <= 1e-15


def test_corner_entries_are_what_makes_it_periodic():
    """With the wrapped entries set to zero the cyclic matrix IS the strict pentadiagonal one."""
    N, M = 50, 9
    a, b, c, d, e = (v.copy() for v in pin.random_periodic_diag_dominant(11, N))
    a[:2] = 0.0; b[0] = 0.0; d[-1] = 0.0; e[-2:] = 0.0
    f = pin.uniform_pm1(12, 0, N, M)
    xp = oracle.solve_periodic_batch(oracle.factor_periodic(a, b, c, d, e), f)
    xs = oracle.solve_batch(oracle.factor(a, b, c, d, e), f)
    assert normwise(xp, xs) <= 1e-14
    # and with them present the two differ (the wrap is really used)
    a2, b2, c2, d2, e2 = pin.random_periodic_diag_dominant(11, N)
    xq = oracle.solve_periodic_batch(oracle.factor_periodic(a2, b2, c2, d2, e2), f)
    assert normwise(xq, xs) > 1e-3


@pytest.mark.parametrize("N,sigma_x", [(64, 0.1), (128, 10.0), (31, 2.5)])
def test_circulant_spectrum_closed_form(N, sigma_x):
    """Eq. 7a/7b is circulant: cos/sin(2 pi m j/N) are eigenvectors with
    lambda_m = c + 2 b cos(th) + 2 a cos(2 th) = 1 + 16 sigma_x sin^4(pi m/N), th = 2 pi m/N."""
    pf = oracle.factor_periodic(*pin.periodic_hyperdiffusion_diagonals(N, sigma_x))
    j = np.arange(N)[:, None]
    m = np.arange(N)[None, :]
    f = np.cos(2 * np.pi * m * j / N) + 0.5 * np.sin(2 * np.pi * m * j / N)
    lam = 1.0 + 16.0 * sigma_x * np.sin(np.pi * np.arange(N) / N) ** 4
    x = oracle.solve_periodic_batch(pf, f)
    assert normwise(x, f / lam[None, :]) <= 5e-14 * (1 + 16 * sigma_x)


def test_crank_nicolson_amplification_factor():
    """A c+ = (2I - A) c on an eigenmode: c+ = G c, G = (1 - s)/(1 + s), s = 16 sigma_x sin^4(pi m/N)."""
    N, sigma_x, steps = 48, 0.37, 25
    pf = oracle.factor_periodic(*pin.periodic_hyperdiffusion_diagonals(N, sigma_x))
    j = np.arange(N)[:, None]
    ms = np.array([0, 1, 2, 5, 11, 24])
    c0 = np.cos(2 * np.pi * ms[None, :] * j / N + 0.3)
    s = 16.0 * sigma_x * np.sin(np.pi * ms / N) ** 4
    G = (1.0 - s) / (1.0 + s)
    c = oracle.step_periodic_batch(pf, c0, steps)
    assert np.max(np.abs(c - c0 * (G ** steps)[None, :])) <= 1e-13
    # mode 0 (the mean) is invariant: the scheme conserves mass on a periodic grid
    assert np.max(np.abs(c[:, 0] - c0[:, 0])) <= 1e-13        # 25 steps of rounding


def _fig2_errors(Ns, T=1e-4, dt=1e-8, n=2):
    """gamma = D = L = 1, A = 1, phi = 0, n = 2; eps_N(T) of Eq. 15."""
    steps = int(round(T / dt))
    out = []
    for N in Ns:
        dx = 1.0 / N
        pf = oracle.factor_periodic(*pin.periodic_hyperdiffusion_diagonals(N, dt / (2.0 * dx ** 4)))
        xg = np.arange(1, N + 1) * dx
        c = oracle.step_periodic_batch(pf, np.cos(2 * np.pi * n * xg)[:, None], steps)[:, 0]
        exact = np.exp(-((2 * np.pi * n) ** 4) * T) * np.cos(2 * np.pi * n * xg)      # Eq. 14
        out.append(np.sqrt(np.mean((c - exact) ** 2)))                                 # Eq. 15
    return np.array(out)


def test_paper_validation_decay_and_printed_slope():
    """The paper's own validation (section II.E): the numerical solution follows Eq. 14 and the
    error falls like N^-2; the fitted slope the paper prints is -2.0162 (tests/golden)."""
    with open(GOLDEN) as fh:
        printed = [float(l.split()[1]) for l in fh if l.startswith("slope")][0]
    assert printed == -2.0162
    Ns = np.array([16, 32, 64, 128, 256, 512])
    eps = _fig2_errors(Ns)
    assert np.all(eps[1:] < eps[:-1])
    slope = np.polyfit(np.log(Ns), np.log(eps), 1)[0]
    # the paper's range of N is not printed; over 16..512 the fit is -2.019, over 64..512 -2.002
    assert abs(slope - printed) <= 0.02
    assert abs(slope + 2.0) <= 0.03
    # leading error term of the centred 5-point fourth difference: k^4 -> k^4 (1 - (k dx)^2/6)
    # => eps ~ amplitude/sqrt(2) * T k^6 dx^2 / 6 * exp(-k^4 T)
    k = 2 * np.pi * 2
    pred = (1 / np.sqrt(2)) * 1e-4 * k ** 6 / (6.0 * 512.0 ** 2) * np.exp(-(k ** 4) * 1e-4)
    assert abs(eps[-1] / pred - 1.0) <= 0.02


def test_singular_and_small_n_errors():
    with pytest.raises(ValueError):
        oracle.factor_periodic(*(np.ones(5),) * 5)
    N = 8
    a, b, c, d, e = (v.copy() for v in pin.random_periodic_diag_dominant(2, N))
    c[0] = 0.0
    a[2] = 0.0   # keep row 0 the failing pivot
    with pytest.raises(oracle.SingularPivot) as ei:
        oracle.factor_periodic(a, b, c, d, e)
    assert ei.value.row == 0
