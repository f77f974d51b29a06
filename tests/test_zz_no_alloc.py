"""pent_factor_solve_batch_noalloc: the per-system factor + solve with its scratch in a static device array of the
library (no allocation inside the call) against the existing allocating path, on two calls in a row.  Collected last on
purpose (the suite runs with pytest -x).  Runs alone in a fresh process as well as after the other tests."""
import numpy as np
import pytest
import torch

import oracle
import pent_inputs as pin
from gpu_helpers import Guarded, check_all, guarded, normwise

pytestmark = pytest.mark.gpu


def _pent():
    import paper_1807_07382_b200 as pent
    return pent


def _case(pent, N, M, seed, dtype=torch.float64):
    sig = pin.uniform_vec(seed, 1, M, 0.1, 10.0)
    diags = pin.diagonals_I_plus_sigma_L2(N, sig) if N >= 4 else pin.random_diag_dominant(seed, N, M)
    f = pin.uniform_pm1(seed, 0, N, M)
    if dtype == torch.float32:
        diags = [np.asarray(v, dtype=np.float32).astype(np.float64) for v in diags]
        f = f.astype(np.float32).astype(np.float64)
    gs = [guarded(v, dtype) for v in diags]
    a, b, c, d, e = (g.t for g in gs)
    fg, xg, ig = guarded(f, dtype), Guarded((N, M), dtype), Guarded((M,), torch.int32)
    ig.t.fill_(7)                                     # the call must overwrite every entry
    pent.pent_factor_solve_batch_noalloc(N, M, e, c, d, a, b, fg.t, xg.t, ig.t)
    torch.cuda.synchronize()
    check_all(fg, xg, ig, *gs)
    x_ref, info_ref = pent.pent_factor_solve_batch(N, M, e, c, d, a, b, fg.t)          # the existing (allocating) path
    got, want = xg.numpy().astype(np.float64), x_ref.cpu().numpy().astype(np.float64)
    tol = 1e-11 if dtype == torch.float64 else 2e-5
    assert normwise(got, want) <= tol
    assert np.array_equal(ig.numpy(), info_ref.cpu().numpy()) and not ig.numpy().any()
    ref, _ = oracle.factor_solve_batch(*diags, f, nthreads=4)                          # and the oracle
    assert normwise(got, ref) <= tol


def test_noalloc_matches_the_allocating_path_on_two_calls_in_a_row():
    pent = _pent()
    assert pent.pent_noalloc_scratch_bytes() == 32 << 20
    # second call: smaller problem, other data -- the array still holds the first call's gamma, delta, g
    _case(pent, 1024, 1300, seed=91)
    _case(pent, 1024, 200 + 37, seed=92)
    _case(pent, 1024, 1300, seed=91)                  # and the first one again


@pytest.mark.parametrize("N,M,dtype", [(257, 2000, torch.float32), (5, 70, torch.float64), (64, 1, torch.float64)])
def test_noalloc_other_shapes(N, M, dtype):
    _case(_pent(), N, M, seed=93, dtype=dtype)


def test_noalloc_rejects_sizes_beyond_the_static_array():
    pent = _pent()
    N = 1024
    m_max = (32 << 20) // (3 * 8 * N) // 64 * 64       # 1344 systems of N = 1024 in fp64
    assert m_max == 1344
    for M, ok in ((m_max, True), (m_max + 1, False), (65536, False)):
        t = [torch.ones((N, M), dtype=torch.float64, device="cuda") for _ in range(2)]
        z = torch.zeros((N, M), dtype=torch.float64, device="cuda")
        info = torch.zeros(M, dtype=torch.int32, device="cuda")
        x = torch.full((N, M), -3.0, dtype=torch.float64, device="cuda")
        if ok:
            pent.pent_factor_solve_batch_noalloc(N, M, z, t[0], z, z, z, t[1], x, info)      # A = I: x = f
            torch.cuda.synchronize()
            assert bool((x == 1.0).all())
        else:
            with pytest.raises(pent.PentError) as ei:
                pent.pent_factor_solve_batch_noalloc(N, M, z, t[0], z, z, z, t[1], x, info)
            assert ei.value.code == 5
            torch.cuda.synchronize()
            assert bool((x == -3.0).all())              # nothing was launched
