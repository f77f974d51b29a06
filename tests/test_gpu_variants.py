"""GPU parity for the per-system-matrix variant (BASELINE.json configs[4]) and the
fused time-step path (PAPER.md:53 Eq. 2, :87-89 Eq. 6; BASELINE.json configs[3])."""
import math

import numpy as np
import pytest
import torch

import oracle
import pent_inputs as pin
from gpu_helpers import Guarded, check_all, chunked_order_solve_fp64, envelope_tol, guarded, normwise, pinned_tol
from pent_inputs.configs import R_CH, SIGMA_CH, WORKLOADS, banded_matvec, make_matrix, make_rhs

pytestmark = pytest.mark.gpu


def _pent():
    import paper_1807_07382_b200 as pent
    return pent


def residual(diags, x, f):
    r = banded_matvec(*diags, x.astype(np.float64)) - f
    return float(np.max(np.linalg.norm(r, axis=0) / np.linalg.norm(f, axis=0)))


def _dev(v, dtype=torch.float64):
    return torch.tensor(np.ascontiguousarray(v), dtype=dtype, device="cuda")


# ---- per-system matrices ------------------------------------------------------------------
@pytest.mark.parametrize("N,M", [(64, 100), (1024, 2048 + 37), (5, 3), (3, 70), (8, 33), (9, 40), (1023, 130), (2001, 64)])
def test_factor_solve_batch_parity(N, M):
    pent = _pent()
    if N >= 4:
        sig = pin.uniform_vec(6, 1, M, 0.1, 10.0)
        diags = pin.diagonals_I_plus_sigma_L2(N, sig)
    else:
        diags = pin.random_diag_dominant(60 + N, N, M)
    f = pin.uniform_pm1(6, 0, N, M)
    gs = [guarded(v) for v in diags]
    a, b, c, d, e = (g.t for g in gs)
    fg, xg = guarded(f), Guarded((N, M))
    ig = Guarded((M,), torch.int32)
    wg = Guarded((3 * N * ((M + 63) // 64 * 64),))
    x, info = pent.pent_factor_solve_batch(N, M, e, c, d, a, b, fg.t, xg.t, ig.t, workspace=wg.t)
    check_all(fg, xg, ig, wg, *gs)
    ref, rinfo = oracle.factor_solve_batch(*diags, f, nthreads=8)
    assert not info.cpu().numpy().any() and not rinfo.any()
    assert normwise(x.cpu().numpy(), ref) <= 1e-11
    assert residual(diags, x.cpu().numpy(), f) <= 1e-12
    # stored-factor route gives the same answers
    ig2, xg2 = Guarded((M,), torch.int32), Guarded((N, M))
    h, info2 = pent.pent_factor_batch(N, M, e, c, d, a, b, ig2.t)
    x2 = pent.pent_solve_batch_multi(h, fg.t, xg2.t)
    check_all(fg, xg2, ig2, *gs)
    assert not info2.cpu().numpy().any()
    assert normwise(x2.cpu().numpy(), ref) <= 1e-11


@pytest.mark.parametrize("N,M", [(257, 96), (64, 31), (12, 200)])
def test_factor_solve_batch_nonsymmetric_two_threads_per_system(N, M):
    """Non-symmetric per-system matrices (nothing of the twisted factorisation may rely on symmetry: the bottom half is
    factored bottom-up with a <-> e, b <-> d), plus a singular pivot in the BOTTOM half of one system."""
    pent = _pent()
    diags = pin.random_diag_dominant(66 + N, N, M)
    f = pin.uniform_pm1(67, 0, N, M)
    gs = [guarded(v) for v in diags]
    a, b, c, d, e = (g.t for g in gs)
    fg, xg, ig = guarded(f), Guarded((N, M)), Guarded((M,), torch.int32)
    x, info = pent.pent_factor_solve_batch(N, M, e, c, d, a, b, fg.t, xg.t, ig.t)
    check_all(fg, xg, ig, *gs)
    ref, rinfo = oracle.factor_solve_batch(*diags, f)
    assert not info.cpu().numpy().any() and not rinfo.any()
    assert normwise(x.cpu().numpy(), ref) <= 1e-11
    assert residual(diags, x.cpu().numpy(), f) <= 1e-12
    # in place (x == f, which include/pent.h allows): every read of f precedes the first write of x within a system
    fi = fg.t.clone()
    xi, _ = pent.pent_factor_solve_batch(N, M, e, c, d, a, b, fi, fi)
    assert np.array_equal(xi.cpu().numpy(), x.cpu().numpy())
    # the last row is the FIRST pivot of the bottom-up thread: c[N-1] = 0 makes it exactly zero
    c2 = c.clone(); c2[N - 1, 5] = 0.0
    x2, info2 = pent.pent_factor_solve_batch(N, M, e, c2, d, a, b, fg.t)
    info2 = info2.cpu().numpy()
    assert info2[5] == N and np.count_nonzero(info2) == 1
    keep = np.arange(M) != 5
    assert np.array_equal(x2.cpu().numpy()[:, keep], x.cpu().numpy()[:, keep])


def test_cfg5b_full_size():
    pent = _pent()
    w = WORKLOADS["cfg5b"]
    diags = make_matrix(w)
    f = make_rhs(w)
    a, b, c, d, e = (_dev(v) for v in diags)
    ws = torch.empty(3 * w.N * ((w.M + 63) // 64 * 64), dtype=torch.float64, device="cuda")
    x, info = pent.pent_factor_solve_batch(w.N, w.M, e, c, d, a, b, _dev(f), workspace=ws)
    x = x.cpu().numpy()
    assert not info.cpu().numpy().any()
    ref, _ = oracle.factor_solve_batch(*diags, f, nthreads=8)
    assert normwise(x, ref) <= 1e-11
    assert residual(diags, x, f) <= 1e-12


def test_per_system_fp32_and_singular_flag():
    pent = _pent()
    N, M = 256, 300
    sig = pin.uniform_vec(6, 1, M, 0.1, 10.0)
    diags = [np.asarray(v, dtype=np.float32) for v in pin.diagonals_I_plus_sigma_L2(N, sig)]
    f = pin.uniform_pm1(6, 0, N, M).astype(np.float32)
    a, b, c, d, e = (_dev(v, torch.float32) for v in diags)
    x, info = pent.pent_factor_solve_batch(N, M, e, c, d, a, b, _dev(f, torch.float32))
    d64 = [v.astype(np.float64) for v in diags]
    ref, _ = oracle.factor_solve_batch(*d64, f.astype(np.float64))
    assert normwise(x.cpu().numpy().astype(np.float64), ref) <= 2e-5
    assert residual(d64, x.cpu().numpy(), f.astype(np.float64)) <= 1e-5
    # one singular system: flagged with first bad row + 1, the others untouched
    c2 = c.clone(); c2[0, 7] = 0.0
    x2, info2 = pent.pent_factor_solve_batch(N, M, e, c2, d, a, b, _dev(f, torch.float32))
    info2 = info2.cpu().numpy()
    assert info2[7] == 1 and info2.sum() == 1
    keep = np.arange(M) != 7
    assert np.array_equal(x2.cpu().numpy()[:, keep], x.cpu().numpy()[:, keep])


# ---- fused time step ------------------------------------------------------------------------
def _ch_setup(N, M, bcname, seed=4):
    sigma = 1e-2 * 1e-6 * N ** 4
    r = 1e-6 * N ** 2
    diags = pin.diagonals_I_plus_sigma_L2(N, sigma, bcname)
    m = pin.uniform_vec(seed, 5, M, -0.5, 0.5)
    c0 = m[None, :] + 0.05 * pin.uniform_pm1(seed, 0, N, M)
    return diags, sigma, r, c0


STEP_KERNELS = [1, 2]      # thread per system (one launch per step), on-chip chunked (one launch)


@pytest.mark.parametrize("kernel", STEP_KERNELS)
@pytest.mark.parametrize("bc,bcname", [(1, "zeroflux"), (0, "dirichlet")])
@pytest.mark.parametrize("form", [1, 0])
@pytest.mark.parametrize("N,M", [(1024, 300), (64, 34), (4, 6), (1000, 130), (37, 18)])
def test_ch_one_step_parity(kernel, bc, bcname, form, N, M):
    pent = _pent()
    diags, sigma, r, c0 = _ch_setup(N, M, bcname)
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    h = pent.pent_factor(N, e, c, d, a, b)
    cg = guarded(c0)
    sg = Guarded((N, M))
    pent.pent_step_batch(h, M, cg.t, 1, kind=0, bc=bc, form=form, r=r, sigma=sigma, kernel=kernel, scratch=sg.t)
    check_all(cg, sg)
    ref = oracle.step_batch(oracle.factor(*diags), 0, bc, form, r, sigma, c0, 1)
    # The error is measured against the same step evaluated in long double (oracle/pent_oracle_ld.c).  Bar:
    # north_star's 1e-11, or twice what a plain fp64 CPU evaluation of the step leaves on this input when that
    # is larger (C-15): the fp64 oracle (serial sweep) for the thread-per-system kernel; for the
    # on-chip kernel also the same right-hand side solved in the chunked evaluation ORDER on the CPU
    # (gpu_helpers.chunked_order_solve_fp64).  At N >= 1000, sigma = 1.1e4, increment form, the oracle is
    # 1.2e-11 and the chunked order 4e-11 from the truth; everywhere else all of them are below 2e-12.
    truth = oracle.ld_step_batch(diags, 0, bc, form, r, sigma, c0, 1)
    got = cg.numpy()
    evals = [ref]
    if kernel == 2 and N >= 1000:
        fac = oracle.factor(*diags)
        rhs = np.stack([oracle.rhs(fac, 0, bc, form, r, sigma, c0[:, i]) for i in range(M)], axis=1)
        sol = chunked_order_solve_fp64(fac, rhs)
        evals.append(c0 + sol if form == 1 else sol)
    err_gpu = normwise(got, truth)
    if N >= 1000:
        print(f"CH one step N={N} bc={bc} form={form} kernel={kernel}: vs long double: GPU {err_gpu:.3e}, "
              + ", ".join(f"fp64 CPU[{j}] {normwise(v, truth):.3e}" for j, v in enumerate(evals)))
    assert err_gpu <= envelope_tol(1e-11, truth, *evals)


@pytest.mark.parametrize("kernel,N,M", [(1, 300, 129), (2, 300, 130), (2, 1024, 64), (2, 33, 20), (0, 300, 129)])
def test_hyperdiffusion_step_parity_general_matrix(kernel, N, M):
    pent = _pent()
    diags = pin.random_diag_dominant(21, N)
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    h = pent.pent_factor(N, e, c, d, a, b)
    c0 = pin.uniform_pm1(22, 0, N, M)
    cg, sg = guarded(c0), Guarded((N, M))
    pent.pent_step_batch(h, M, cg.t, 3, kind=1, kernel=kernel, scratch=sg.t)
    check_all(cg, sg)
    ref = oracle.step_batch(oracle.factor(*diags), 1, 0, 0, 0.0, 0.0, c0, 3)
    assert normwise(cg.numpy(), ref) <= 1e-11


@pytest.mark.parametrize("N,M,dtype", [(2048, 200, torch.float64), (4096, 96, torch.float64), (3000, 64, torch.float64),
                                       (4096, 130, torch.float32), (1500, 37, torch.float64)])
def test_hyperdiffusion_step_beyond_the_on_chip_size(N, M, dtype):
    """N > 1024: the state does not fit on chip; a Crank-Nicolson step is then one chunked solve with the 2x - f epilogue
    (c+ = 2 A^-1 c - c), in place, against the oracle's (2I - A) c followed by a solve.  M = 37: the LDG loader."""
    pent = _pent()
    f32 = dtype == torch.float32
    diags = pin.random_diag_dominant(23, N)
    c0 = pin.uniform_pm1(24, 0, N, M)
    if f32:
        diags = tuple(np.asarray(v, dtype=np.float32).astype(np.float64) for v in diags)
        c0 = c0.astype(np.float32).astype(np.float64)
    a, b, c, d, e = (torch.tensor(v, dtype=dtype) for v in diags)
    h = pent.pent_factor(N, e, c, d, a, b)
    assert pent.lib().pent_step_kernel_choice(h.ptr, M) == pent.KERNEL_THREAD_PER_SYSTEM      # = "not the on-chip step kernel"
    cg = guarded(c0, dtype)
    n0 = pent.launch_count(reset=True)
    pent.pent_step_batch(h, M, cg.t, 3, kind=1)
    assert pent.launch_count() == 3                      # one solve launch per step, no scratch
    cg.check()
    ref = oracle.step_batch(oracle.factor(*diags), 1, 0, 0, 0.0, 0.0, c0, 3, nthreads=4)
    assert normwise(cg.numpy().astype(np.float64), ref) <= (2e-5 if f32 else 1e-11)
    # the thread-per-system kernel (4 passes) still answers the same question
    c2 = guarded(c0, dtype)
    pent.pent_step_batch(h, M, c2.t, 3, kind=1, kernel=1)
    assert normwise(c2.numpy().astype(np.float64), ref) <= (2e-5 if f32 else 1e-11)


def test_multi_step_on_chip_equals_repeated_single_steps():
    """The on-chip kernel keeps the state in shared memory across steps: n steps in one launch must
    give bit-identical results to n launches of one step (same arithmetic, same order)."""
    pent = _pent()
    N, M = 512, 96
    diags, sigma, r, c0 = _ch_setup(N, M, "zeroflux")
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    h = pent.pent_factor(N, e, c, d, a, b)
    assert pent.lib().pent_step_kernel_choice(h.ptr, M) == pent.KERNEL_CHUNKED
    c1, c2 = _dev(c0), _dev(c0)
    pent.pent_step_batch(h, M, c1, 7, kind=0, bc=1, form=1, r=r, sigma=sigma, kernel=2)
    for _ in range(7):
        pent.pent_step_batch(h, M, c2, 1, kind=0, bc=1, form=1, r=r, sigma=sigma, kernel=2)
    assert torch.equal(c1, c2)
    ref = oracle.step_batch(oracle.factor(*diags), 0, 1, 1, r, sigma, c0, 7)
    truth = oracle.ld_step_batch(diags, 0, 1, 1, r, sigma, c0, 7)
    assert normwise(c1.cpu().numpy(), truth) <= pinned_tol(7e-11, ref, truth)     # 7 steps of the 1e-11 bar


@pytest.mark.parametrize("kernel", STEP_KERNELS)
def test_cfg4_thousand_steps_conservation_and_trajectory(kernel):
    """BASELINE.json configs[3]: N=1024, M=8192, 1000 fused steps, zero-flux L, increment form.
    mean(c) per run conserved to 1e-12 on EVERY system (fsum on the host); trajectory parity with
    the oracle after 1000 nonlinear steps on 1024 systems (every eighth) to 1e-9."""
    pent = _pent()
    w = WORKLOADS["cfg4"]
    diags = make_matrix(w)
    c0 = make_rhs(w)
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    h = pent.pent_factor(w.N, e, c, d, a, b)
    cg, sg = guarded(c0), Guarded((w.N, w.M))
    pent.pent_step_batch(h, w.M, cg.t, 1000, kind=0, bc=1, form=1, r=R_CH, sigma=SIGMA_CH,
                         scratch=sg.t, kernel=kernel)
    check_all(cg, sg)
    c1 = cg.numpy()
    assert np.isfinite(c1).all()
    c1r, c0r = np.ascontiguousarray(c1.T), np.ascontiguousarray(c0.T)
    drift = max(abs(math.fsum(c1r[i]) - math.fsum(c0r[i])) / w.N for i in range(w.M))
    assert drift <= 1e-12
    cols = np.arange(0, w.M, 8)
    ref = oracle.step_batch(oracle.factor(*diags), 0, 1, 1, R_CH, SIGMA_CH,
                            np.ascontiguousarray(c0[:, cols]), 1000, nthreads=8)
    assert normwise(c1[:, cols], ref) <= 1e-9
    assert np.max(np.abs(c1 - c0)) > 1e-3          # the state evolved


@pytest.mark.parametrize("kernel", STEP_KERNELS)
def test_step_fp32_one_step(kernel):
    pent = _pent()
    N, M = 256, 200
    diags, sigma, r, c0 = _ch_setup(N, M, "zeroflux")
    d32 = [np.asarray(v, dtype=np.float32) for v in diags]
    a, b, c, d, e = (torch.tensor(v) for v in d32)
    h = pent.pent_factor(N, e, c, d, a, b)
    cd = _dev(c0, torch.float32)
    pent.pent_step_batch(h, M, cd, 1, kind=0, bc=1, form=0, r=r, sigma=sigma, kernel=kernel)
    d64 = [v.astype(np.float64) for v in d32]
    ref = oracle.step_batch(oracle.factor(*d64), 0, 1, 0, float(np.float32(r)),
                            float(np.float32(sigma)), c0.astype(np.float32).astype(np.float64), 1)
    assert normwise(cd.cpu().numpy().astype(np.float64), ref) <= 2e-5


# ---- forced Cahn-Hilliard with per-system parameters (Remark 1 / Eq. 3) ----
def _forcing_params(M, seed=70, dtype=torch.float64):
    mu1 = pin.uniform_vec(seed, 1, M, 50.0, 5000.0)         # dt * mu1 ~ 5e-5 .. 5e-3 per step
    mu2 = pin.uniform_vec(seed, 2, M, -2e4, 2e4)            # up to 20 periods over 1000 steps of dt = 1e-6
    return mu1, mu2, guarded(mu1, dtype), guarded(mu2, dtype)


@pytest.mark.parametrize("kernel", STEP_KERNELS)
@pytest.mark.parametrize("form", [1, 0])
@pytest.mark.parametrize("N,M,nsteps", [(256, 200, 3), (1024, 130, 2), (100, 38, 5), (64, 16, 1)])
def test_forced_ch_parity(kernel, form, N, M, nsteps):
    pent = _pent()
    diags, sigma, r, c0 = _ch_setup(N, M, "zeroflux")
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    h = pent.pent_factor(N, e, c, d, a, b)
    mu1, mu2, g1, g2 = _forcing_params(M)
    dt, t0 = 1e-6, 3.5e-5
    cg, sg = guarded(c0), Guarded((N, M))
    pent.pent_step_batch(h, M, cg.t, nsteps, kind=0, bc=1, form=form, r=r, sigma=sigma, kernel=kernel, scratch=sg.t,
                         forcing=(g1.t, g2.t, dt, t0))
    check_all(cg, sg, g1, g2)
    fac = oracle.factor(*diags)
    ref = oracle.step_forced_batch(fac, 1, form, r, sigma, dt, t0, mu1, mu2, c0, nsteps)
    unforced = oracle.step_batch(fac, 0, 1, form, r, sigma, c0, nsteps)
    assert normwise(ref, unforced) > 1e-6                                    # the forcing is visible at this scale
    tol = 1e-11 * nsteps
    if N >= 1000:   # stiff matrix: same measured envelope as the unforced step (the forcing adds nothing to it)
        truth = oracle.ld_step_batch(diags, 0, 1, form, r, sigma, c0, 1)
        one = oracle.step_batch(fac, 0, 1, form, r, sigma, c0, 1)
        rhs = np.stack([oracle.rhs(fac, 0, 1, form, r, sigma, c0[:, i]) for i in range(M)], axis=1)
        sol = chunked_order_solve_fp64(fac, rhs)
        tol = nsteps * envelope_tol(1e-11, truth, one, c0 + sol if form == 1 else sol)
    assert normwise(cg.numpy(), ref) <= tol


def test_forced_ch_multi_step_launch_equals_single_step_launches_and_conserves_mean():
    """n forced steps in one launch == n launches of one step with t0 advanced by the caller (bit for bit), and the
    zero-mean forcing leaves mean(c) invariant (zero-flux operator, increment form)."""
    pent = _pent()
    N, M, n = 512, 96, 9
    diags, sigma, r, c0 = _ch_setup(N, M, "zeroflux")
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    h = pent.pent_factor(N, e, c, d, a, b)
    mu1, mu2, g1, g2 = _forcing_params(M)
    dt, t0 = 1e-6, 0.0
    c1, c2 = _dev(c0), _dev(c0)
    kw = dict(kind=0, bc=1, form=1, r=r, sigma=sigma, kernel=2)
    pent.pent_step_batch(h, M, c1, n, forcing=(g1.t, g2.t, dt, t0), **kw)
    for k in range(n):
        pent.pent_step_batch(h, M, c2, 1, forcing=(g1.t, g2.t, dt, t0 + k * dt), **kw)
    assert torch.equal(c1, c2)
    got = c1.cpu().numpy()
    drift = max(abs(math.fsum(got[:, i]) - math.fsum(c0[:, i])) / N for i in range(M))
    assert drift <= 1e-13
    ref = oracle.step_forced_batch(oracle.factor(*diags), 1, 1, r, sigma, dt, t0, mu1, mu2, c0, n)
    assert normwise(got, ref) <= 1e-11 * n


def test_forced_ch_cfg4_shape_conservation_and_cost():
    """cfg4's shape (N=1024, M=8192), 200 forced steps in one launch: mean(c) of every run conserved to 1e-12, parity
    with the oracle on every 16th system, and the forced step costs about what the unforced one does."""
    pent = _pent()
    w = WORKLOADS["cfg4"]
    diags = make_matrix(w)
    c0 = make_rhs(w)
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    h = pent.pent_factor(w.N, e, c, d, a, b)
    mu1, mu2, g1, g2 = _forcing_params(w.M)
    n, dt = 200, 1e-6
    cg = guarded(c0)
    kw = dict(kind=0, bc=1, form=1, r=R_CH, sigma=SIGMA_CH)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    pent.pent_step_batch(h, w.M, cg.t, n, forcing=(g1.t, g2.t, dt, 0.0), **kw)      # also the warm-up
    cg.check()
    c1 = cg.numpy()
    c1r, c0r = np.ascontiguousarray(c1.T), np.ascontiguousarray(c0.T)
    assert max(abs(math.fsum(c1r[i]) - math.fsum(c0r[i])) / w.N for i in range(w.M)) <= 1e-12
    cols = np.arange(0, w.M, 16)
    ref = oracle.step_forced_batch(oracle.factor(*diags), 1, 1, R_CH, SIGMA_CH, dt, 0.0, mu1[cols], mu2[cols],
                                   np.ascontiguousarray(c0[:, cols]), n, nthreads=8)
    assert normwise(c1[:, cols], ref) <= 1e-9
    cd = _dev(c0)
    pent.pent_step_batch(h, w.M, cd, n, **kw)
    torch.cuda.synchronize()
    ev[0].record(); pent.pent_step_batch(h, w.M, cd, n, **kw); ev[1].record()
    ev[2].record(); pent.pent_step_batch(h, w.M, cd, n, forcing=(g1.t, g2.t, dt, 0.0), **kw); ev[3].record()
    torch.cuda.synchronize()
    t_plain, t_forced = ev[0].elapsed_time(ev[1]) / n * 1e3, ev[2].elapsed_time(ev[3]) / n * 1e3
    print(f"cfg4 shape: unforced {t_plain:.2f} us per step, forced {t_forced:.2f} us per step ({t_forced / t_plain:.3f} x)")
    assert t_forced <= 1.25 * t_plain


@pytest.mark.parametrize("kernel", STEP_KERNELS)
def test_forced_ch_fp32(kernel):
    pent = _pent()
    N, M, n = 256, 200, 4
    diags, sigma, r, c0 = _ch_setup(N, M, "zeroflux")
    d32 = [np.asarray(v, dtype=np.float32) for v in diags]
    a, b, c, d, e = (torch.tensor(v) for v in d32)
    h = pent.pent_factor(N, e, c, d, a, b)
    mu1, mu2, g1, g2 = _forcing_params(M, dtype=torch.float32)
    dt, t0 = 1e-6, 2e-5
    cg = guarded(c0, torch.float32)
    pent.pent_step_batch(h, M, cg.t, n, kind=0, bc=1, form=0, r=r, sigma=sigma, kernel=kernel,
                         forcing=(g1.t, g2.t, dt, t0))
    check_all(cg, g1, g2)
    d64 = [v.astype(np.float64) for v in d32]
    f32 = lambda v: np.asarray(v, dtype=np.float32).astype(np.float64)
    ref = oracle.step_forced_batch(oracle.factor(*d64), 1, 0, float(np.float32(r)), float(np.float32(sigma)), dt, t0,
                                   f32(mu1), f32(mu2), f32(c0), n)
    assert normwise(cg.numpy().astype(np.float64), ref) <= 2e-5 * n
