"""GPU tests of the C-ABI boundary contract stated in include/pent.h: no call stalls
another stream, handles are usable from several threads, caches never change results, contract
violations are refused."""
import threading
import time

import numpy as np
import pytest
import torch

import oracle
import pent_inputs as pin
from gpu_helpers import Guarded, guarded, normwise

pytestmark = pytest.mark.gpu


def _pent():
    import paper_1807_07382_b200 as pent
    return pent


def _handle(diags, dtype=torch.float64):
    pent = _pent()
    a, b, c, d, e = (torch.tensor(v, dtype=dtype) for v in diags)
    return pent.pent_factor(len(diags[2]), e, c, d, a, b)


def _periodic_handle(diags):
    pent = _pent()
    a, b, c, d, e = (torch.tensor(v) for v in diags)
    return pent.pent_factor_periodic(len(diags[2]), e, c, d, a, b)


def test_factor_runs_on_a_private_stream_and_stalls_nobody():
    """pent_factor / pent_factor_periodic while a long kernel runs on another stream: the call returns long
    before that kernel ends (it neither waits for it nor synchronises the device)."""
    pent = _pent()
    N, M = 1024, 64 * 16          # 64 persistent CTAs: the long kernel leaves 84 SMs free for the factor kernels
    diags = pin.diagonals_I_plus_sigma_L2(N, 10.0, "zeroflux")
    h = _handle(diags)
    _periodic_handle(pin.periodic_hyperdiffusion_diagonals(64, 1.0))          # warm-up: module load, lazy init
    c = torch.tensor(0.1 + 0.05 * pin.uniform_pm1(1, 0, N, M), device="cuda")
    sB = torch.cuda.Stream()
    done = torch.cuda.Event()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    pent.pent_step_batch(h, M, c, 40000, kind=1, stream=sB)         # a few hundred ms of one kernel on stream B
    done.record(sB)
    d2 = pin.diagonals_I_plus_sigma_L2(2048, 3.0)
    t1 = time.perf_counter()
    h2 = _handle(d2)
    dp = pin.periodic_hyperdiffusion_diagonals(1024, 10.0)
    hp = _periodic_handle(dp)
    t2 = time.perf_counter()
    still_running = not done.query()
    done.synchronize()
    t3 = time.perf_counter()
    print(f"long kernel {t3 - t0:.3f} s; two factor calls issued during it took {t2 - t1:.3f} s")
    assert still_running, "pent_factor waited for the kernel on the other stream"
    assert (t2 - t1) < 0.5 * (t3 - t0)
    # and the handles made meanwhile are complete and correct
    f = pin.uniform_pm1(2, 0, 2048, 64)
    x = pent.pent_solve_batch(h2, 64, torch.tensor(f, device="cuda")).cpu().numpy()
    assert normwise(x, oracle.solve_batch(oracle.factor(*d2), f)) <= 1e-11
    fp = pin.uniform_pm1(3, 0, 1024, 64)
    xp = pent.pent_solve_batch(hp, 64, torch.tensor(fp, device="cuda")).cpu().numpy()
    assert normwise(xp, oracle.solve_periodic_batch(oracle.factor_periodic(*dp), fp)) <= 1e-11


def test_two_threads_same_kernel_instance_different_shared_memory():
    """cudaFuncAttributeMaxDynamicSharedMemorySize is process-wide.  Thread A launches the
    fp64 S=16 instance with an N=1024 handle (~200 KB of dynamic shared memory), thread B the same instance
    with N=256 (~60 KB), then A again: every launch must succeed and be correct."""
    pent = _pent()
    cases = {}
    for name, N in (("A", 1024), ("B", 256)):
        diags = pin.diagonals_I_plus_sigma_L2(N, 2.0)
        f = pin.uniform_pm1(10 + N, 0, N, 160)
        cases[name] = (_handle(diags), N, torch.tensor(f, device="cuda"),
                       oracle.solve_batch(oracle.factor(*diags), f))
    turn = threading.Semaphore(1), threading.Semaphore(0)
    errors = []

    def worker(name, mine, other):
        try:
            torch.cuda.set_device(0)
            h, N, fd, ref = cases[name]
            for _ in range(3):
                mine.acquire()
                x = pent.pent_solve_batch(h, 160, fd, kernel=pent.KERNEL_CHUNKED_CFG(1, 16))
                torch.cuda.synchronize()
                if normwise(x.cpu().numpy(), ref) > 1e-11:
                    errors.append(f"{name}: wrong result")
                other.release()
        except Exception as ex:                      # a failed launch surfaces here as PentError
            errors.append(f"{name}: {ex!r}")
            other.release()

    ta = threading.Thread(target=worker, args=("A", turn[0], turn[1]))
    tb = threading.Thread(target=worker, args=("B", turn[1], turn[0]))
    ta.start(); tb.start(); ta.join(60); tb.join(60)
    assert not errors, errors


def test_step_contract_is_enforced():
    pent = _pent()
    N, M = 128, 32
    h = _handle(pin.diagonals_I_plus_sigma_L2(N, 2.0, "zeroflux"))
    c = torch.tensor(0.1 + 0.05 * pin.uniform_pm1(5, 0, N, M), device="cuda")
    pent.pent_step_batch(h, M, c, 1, kind=0, bc=1, form=1, r=0.3, sigma=2.0)              # matches
    with pytest.raises(pent.PentError) as ei:                                             # wrong sigma
        pent.pent_step_batch(h, M, c, 1, kind=0, bc=1, form=1, r=0.3, sigma=3.0)
    assert ei.value.code == 1
    with pytest.raises(pent.PentError):                                                   # wrong boundary
        pent.pent_step_batch(h, M, c, 1, kind=0, bc=0, form=1, r=0.3, sigma=2.0)
    pent.pent_step_batch(h, M, c, 1, kind=0, bc=1, form=0, r=0.3, sigma=123.0)            # direct form: any A
    hg = _handle(pin.random_diag_dominant(6, N))
    with pytest.raises(pent.PentError):                                                   # not I + sigma L^2 at all
        pent.pent_step_batch(hg, M, c, 1, kind=0, bc=1, form=1, r=0.3, sigma=2.0)
    pent.pent_step_batch(hg, M, c, 1, kind=1)                                             # (2I - A) c takes any A


def test_introspection_and_binding_validation():
    pent = _pent()
    L = pent.lib()
    assert L.pent_handle_m(None) == -1 and L.pent_handle_device(None) == -1 and L.pent_handle_band(None) == -1
    N, M = 96, 40
    diags = pin.random_diag_dominant(7, N)
    h = _handle(diags)
    assert L.pent_handle_device(h.ptr) == torch.cuda.current_device()
    assert L.pent_handle_band(h.ptr) == 2 and L.pent_handle_m(h.ptr) == 0
    a, b, c, d, e = diags
    ht = _handle((np.zeros(N), b, c, d, np.zeros(N)))
    assert L.pent_handle_band(ht.ptr) == 1
    f = torch.tensor(pin.uniform_pm1(8, 0, N, M), device="cuda")
    with pytest.raises(ValueError):
        pent.pent_solve_batch(h, M, f, torch.empty((N, M + 1), dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):
        pent.pent_solve_batch(h, M, f, torch.empty((N, M), dtype=torch.float32, device="cuda"))
    with pytest.raises(ValueError):
        pent.pent_solve_batch(h, M, f, torch.empty((N, M), dtype=torch.float64))          # CPU tensor
    with pytest.raises(ValueError):
        pent.pent_solve_batch_host(h, M, f.cpu(), torch.empty((N, M), dtype=torch.float64, device="cuda"))
    dv = [torch.tensor(np.repeat(v[:, None], M, axis=1), device="cuda") for v in diags]
    with pytest.raises(ValueError):                                                       # info of the wrong dtype
        pent.pent_factor_solve_batch(N, M, dv[4], dv[2], dv[3], dv[0], dv[1], f,
                                     info=torch.zeros(M, dtype=torch.int64, device="cuda"))
    with pytest.raises(ValueError):                                                       # workspace too small
        pent.pent_factor_solve_batch(N, M, dv[4], dv[2], dv[3], dv[0], dv[1], f,
                                     workspace=torch.empty(10, dtype=torch.float64, device="cuda"))
    with pytest.raises(ValueError):                                                       # scratch too small
        pent.pent_step_batch(h, M, f.clone(), 1, kind=1, scratch=torch.empty(3, dtype=torch.float64, device="cuda"))
    L.pent_release_thread_cache()


def test_cached_tensor_maps_never_change_results():
    """The per-thread cache of encoded tensor maps is keyed by (base, M, N, tile, box, dtype): alternate
    buffers, shapes on the same base pointer and in-place calls, and compare every result with the oracle."""
    pent = _pent()
    N = 512
    diags = pin.diagonals_I_plus_sigma_L2(N, 1.0)
    h = _handle(diags)
    fac = oracle.factor(*diags)
    big = Guarded((N * 1024,))
    other = Guarded((N * 1024,))
    for rep in range(3):
        for M, buf in ((1024, big), (512, big), (1024, other), (256, big), (512, other)):
            f = pin.uniform_pm1(100 + rep, M, N, M)
            fd = buf.t[:N * M].view(N, M)
            fd.copy_(torch.tensor(f))
            x = pent.pent_solve_batch(h, M, fd, fd)
            assert normwise(x.cpu().numpy(), oracle.solve_batch(fac, f, nthreads=8)) <= 1e-11
    big.check(); other.check()
