"""Pins for the long-double oracle (oracle/pent_oracle_ld.c).  It is the "truth" behind the measured
parity tolerances on stiff matrices (reading C-15), so it must be tied to something other
than itself AND shown to carry more precision than the fp64 oracle:

* exact rational arithmetic (fractions.Fraction) on tiny N, stiff and non-symmetric matrices;
* manufactured solutions whose data are exactly representable (integer x, dyadic sigma), at the
  full size and stiffness of config 4: the exact answer is known to the last bit;
* the algebraic identity direct form == increment form of the Cahn-Hilliard step;
* agreement with the (independently pinned) fp64 oracle within cond(A) * 2^-53.
CPU only.
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import pent_inputs as pin
from pent_inputs.configs import banded_matvec


def _normwise(x, ref):
    return float(np.max(np.max(np.abs(x - ref), axis=0) / np.max(np.abs(ref), axis=0)))


def _fraction_solve(A, f):
    """Exact Gauss-Jordan elimination in rational arithmetic; A, f hold Fractions or floats."""
    n = len(f)
    M = [[Fraction(A[i][j]) for j in range(n)] + [Fraction(f[i])] for i in range(n)]
    for k in range(n):
        p = next(i for i in range(k, n) if M[i][k] != 0)
        M[k], M[p] = M[p], M[k]
        piv = M[k][k]
        M[k] = [v / piv for v in M[k]]
        for i in range(n):
            if i != k and M[i][k] != 0:
                m = M[i][k]
                M[i] = [vi - m * vk for vi, vk in zip(M[i], M[k])]
    return [M[i][n] for i in range(n)]


def _ulps(x, exact):
    """max over entries of |x - exact| in units of the spacing of fp64 at |exact|."""
    ex = np.array([float(v) for v in exact])
    return float(np.max(np.abs(x - ex) / np.spacing(np.maximum(np.abs(ex), 1e-300))))


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 8])
def test_ld_solve_exact_rational_nonsymmetric(N):
    a, b, c, d, e = pin.random_diag_dominant(300 + N, N)
    A = pin.dense_from_diagonals(a, b, c, d, e)
    f = pin.uniform_pm1(301 + N, 0, N, 3)
    x = oracle.ld_solve_batch((a, b, c, d, e), f)
    for i in range(3):
        exact = _fraction_solve([[float(v) for v in row] for row in A], [float(v) for v in f[:, i]])
        assert _ulps(x[:, i], exact) <= 1.0      # correctly rounded up to a tie


def test_ld_solve_exact_rational_stiff_beats_fp64():
    """I + sigma L_N^2 with sigma = 1e4 (cond ~ 1.5e5), N = 8: the long-double result is within
    cond * 2^-64 of the exact rational solution; the fp64 oracle is >= 50 x further away (the extra digits are real)."""
    N, sigma = 8, 1.0e4
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, "zeroflux")
    A = pin.dense_from_diagonals(*diags)
    f = pin.uniform_pm1(311, 0, N, 4)
    x_ld = oracle.ld_solve_batch(diags, f)
    x_64 = oracle.solve_batch(oracle.factor(*diags), f)
    worst_ld = worst_64 = 0.0
    for i in range(4):
        exact = _fraction_solve([[float(v) for v in row] for row in A], [float(v) for v in f[:, i]])
        ex = np.array([float(v) for v in exact])
        worst_ld = max(worst_ld, float(np.max(np.abs(x_ld[:, i] - ex)) / np.max(np.abs(ex))))
        worst_64 = max(worst_64, float(np.max(np.abs(x_64[:, i] - ex)) / np.max(np.abs(ex))))
    assert worst_ld <= 1e-14                # cond(A) * 2^-64 = 8e-15
    assert worst_64 >= 50 * worst_ld        # cond(A) * 2^-53: the fp64 oracle is visibly further away


@pytest.mark.parametrize("bc", ["zeroflux", "dirichlet"])
def test_ld_solve_exact_manufactured_full_size_stiff(bc):
    """Config-4 size and stiffness with exactly representable data: sigma = 10995 + 1/8 (dyadic), x has
    small integer entries, so f = A x is computed without any rounding and A^{-1} f = x EXACTLY.
    Long double recovers x to 4e-15; the fp64 oracle is ~cond * 2^-53 away."""
    N, M, sigma = 1024, 16, 10995.125
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, bc)
    x = np.round(8.0 * pin.uniform_pm1(312, 0, N, M))
    f = banded_matvec(*diags, x)
    # every product is an integer multiple of 1/8 below 2^24: the sums are exact
    assert np.all(f * 8.0 == np.round(f * 8.0))
    x_ld = oracle.ld_solve_batch(diags, f)
    x_64 = oracle.solve_batch(oracle.factor(*diags), f)
    err_ld = float(np.max(np.abs(x_ld - x)) / 8.0)
    err_64 = float(np.max(np.abs(x_64 - x)) / 8.0)
    assert err_ld <= 4e-15
    assert 1e-14 <= err_64 <= 1e-10          # two orders of magnitude and more between the two


def test_ld_solve_matches_fp64_oracle_on_config_matrices():
    for N, sigma, bc in ((64, 0.1, "dirichlet"), (512, 1.0, "dirichlet"), (1024, 10.0, "dirichlet"),
                         (1024, 10995.11627776, "zeroflux")):
        diags = pin.diagonals_I_plus_sigma_L2(N, sigma, bc)
        f = pin.uniform_pm1(313, 0, N, 8)
        got = _normwise(oracle.solve_batch(oracle.factor(*diags), f), oracle.ld_solve_batch(diags, f))
        assert got <= 4.0 * (1.0 + 16.0 * sigma) * 2.0 ** -53


def test_ld_per_system_exact_rational_and_matches_shared():
    N, M = 6, 5
    diags = pin.random_diag_dominant(320, N, M)
    f = pin.uniform_pm1(321, 0, N, M)
    x, info = oracle.ld_factor_solve_batch(*diags, f)
    assert not info.any()
    for i in range(M):
        A = pin.dense_from_diagonals(*(v[:, i] for v in diags))
        exact = _fraction_solve([[float(v) for v in row] for row in A], [float(v) for v in f[:, i]])
        assert _ulps(x[:, i], exact) <= 1.0
        one = oracle.ld_solve_batch(tuple(np.ascontiguousarray(v[:, i]) for v in diags), f[:, i:i + 1])
        assert np.array_equal(one[:, 0], x[:, i])


# ---- time step ---------------------------------------------------------------------------------
def _exact_ch_step(diags, bc, r, sigma, c0):
    """One Cahn-Hilliard step A c+ = c + r L (c^3 - c) in exact rational arithmetic."""
    N = len(c0)
    c = [Fraction(float(v)) for v in c0]
    w = [v * v * v - v for v in c]
    Ld = [Fraction(-2)] * N
    if bc == 1:
        Ld[0] = Ld[-1] = Fraction(-1)
    Lw = [Ld[k] * w[k] + (w[k - 1] if k > 0 else 0) + (w[k + 1] if k + 1 < N else 0) for k in range(N)]
    rhs = [c[k] + Fraction(float(r)) * Lw[k] for k in range(N)]
    A = pin.dense_from_diagonals(*diags)
    return _fraction_solve([[float(v) for v in row] for row in A], rhs)


@pytest.mark.parametrize("bc,bcname", [(1, "zeroflux"), (0, "dirichlet")])
@pytest.mark.parametrize("form", [0, 1])
def test_ld_ch_step_exact_rational(bc, bcname, form):
    """Both forms of the step equal the exact rational step (they are algebraically identical,
    DESIGN.md reading C-14) to within one rounding of the result."""
    N, sigma, r = 7, 300.0, 0.75
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, bcname)
    c0 = 0.3 + 0.05 * pin.uniform_pm1(330, 0, N, 2)
    got = oracle.ld_step_batch(diags, 0, bc, form, r, sigma, c0, 1)
    for i in range(2):
        assert _ulps(got[:, i], _exact_ch_step(diags, bc, r, sigma, c0[:, i])) <= 1.0


def test_ld_ch_step_forms_agree_at_config4_where_fp64_forms_do_not():
    """The identity c + r L w - A c = L (r w - sigma L c) needs A = I + sigma L^2 EXACTLY, so sigma is dyadic
    here (the fp64 entries fl(1 + 6 sigma) of config 4's own sigma are off by 1e-16 relative, which moves the
    two forms 7e-12 apart even in exact arithmetic: they are then two different, equally valid schemes)."""
    N, M = 1024, 32
    sigma, r = 10995.125, 1e-6 * N ** 2
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, "zeroflux")
    c0 = pin.uniform_vec(4, 5, M, -0.5, 0.5)[None, :] + 0.05 * pin.uniform_pm1(4, 0, N, M)
    ld0 = oracle.ld_step_batch(diags, 0, 1, 0, r, sigma, c0, 1)
    ld1 = oracle.ld_step_batch(diags, 0, 1, 1, r, sigma, c0, 1)
    assert _normwise(ld0, ld1) <= 2e-14
    fac = oracle.factor(*diags)
    o0 = oracle.step_batch(fac, 0, 1, 0, r, sigma, c0, 1)
    o1 = oracle.step_batch(fac, 0, 1, 1, r, sigma, c0, 1)
    assert _normwise(o0, o1) >= 1e-12                       # fp64: the two forms differ by ~cond * eps
    assert _normwise(o0, ld0) <= 1e-11 and _normwise(o1, ld1) <= 1e-10


def test_ld_hyperdiffusion_step_matches_fp64_and_exact():
    N = 6
    diags = pin.random_diag_dominant(340, N)
    c0 = pin.uniform_pm1(341, 0, N, 2)
    got = oracle.ld_step_batch(diags, 1, 0, 0, 0.0, 0.0, c0, 1)
    A = pin.dense_from_diagonals(*diags)
    for i in range(2):
        c = [Fraction(float(v)) for v in c0[:, i]]
        Af = [[Fraction(float(v)) for v in row] for row in A]
        rhs = [2 * c[k] - sum(Af[k][j] * c[j] for j in range(N)) for k in range(N)]
        assert _ulps(got[:, i], _fraction_solve(Af, rhs)) <= 1.0
    N = 300
    diags = pin.random_diag_dominant(342, N)
    c0 = pin.uniform_pm1(343, 0, N, 4)
    o = oracle.step_batch(oracle.factor(*diags), 1, 0, 0, 0.0, 0.0, c0, 3)
    assert _normwise(o, oracle.ld_step_batch(diags, 1, 0, 0, 0.0, 0.0, c0, 3)) <= 1e-14


# ---- periodic ------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [6, 7, 9])
def test_ld_periodic_exact_rational(N):
    diags = pin.random_periodic_diag_dominant(350 + N, N)
    A = pin.dense_from_periodic_diagonals(*diags)
    f = pin.uniform_pm1(351 + N, 0, N, 2)
    x = oracle.ld_solve_periodic_batch(diags, f)
    for i in range(2):
        exact = _fraction_solve([[float(v) for v in row] for row in A], [float(v) for v in f[:, i]])
        assert _ulps(x[:, i], exact) <= 1.0


def test_ld_periodic_matches_fp64_oracle_on_the_papers_matrix():
    for N, sx in ((40, 10.0), (1024, 10.0), (1024, 1e-8 / (2.0 * (1.0 / 1024) ** 4))):
        diags = pin.periodic_hyperdiffusion_diagonals(N, sx)
        f = pin.uniform_pm1(360, 0, N, 8)
        ref = oracle.solve_periodic_batch(oracle.factor_periodic(*diags), f)
        assert _normwise(ref, oracle.ld_solve_periodic_batch(diags, f)) <= 4.0 * (1.0 + 16.0 * sx) * 2.0 ** -53
