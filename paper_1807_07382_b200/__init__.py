"""paper_1807_07382_b200 -- thin Python binding of libpent (include/pent.h).

Argument marshalling only: every step of the path (factor, sweeps, fused time step) runs in
the hand-written sm_100a kernels of `csrc/`.  PyTorch is used for device memory and streams.
There is NO CPU fallback: if the CUDA library cannot be built or loaded, importing the
compute entry points raises.  Names follow include/pent.h and the paper's notation
(PAPER.md:152 a..e diagonals, :162-165 eps/beta/alpha/gamma/delta, :267 interleaved layout).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

from . import build as _build

PENT_F64, PENT_F32 = 0, 1
KERNEL_AUTO, KERNEL_THREAD_PER_SYSTEM, KERNEL_CHUNKED = 0, 1, 2


def KERNEL_CHUNKED_CFG(Q: int = 0, S: int = 0) -> int:
    """PENT_KERNEL_CHUNKED_CFG of include/pent.h: explicit cluster size Q and tile width S."""
    return 2 | (Q << 8) | (S << 16)


def kernel_choice(h: "Handle", M: int) -> dict:
    """What PENT_KERNEL_AUTO runs for M systems: {'kernel': name, 'Q': .., 'S': ..}."""
    v = lib().pent_solve_kernel_choice(h.ptr, M)
    if (v & 0xff) == KERNEL_CHUNKED:
        return {"kernel": "solve_chunked_kernel", "Q": (v >> 8) & 0xff, "S": (v >> 16) & 0xff}
    return {"kernel": "solve_tps_kernel", "Q": 0, "S": 0}
def rows_kernel_choice(h: "Handle", M: int) -> dict:
    """What pent_solve_batch_rows runs for M systems: cluster size, tile width and data path."""
    v = lib().pent_solve_rows_kernel_choice(h.ptr, M)
    if v < 0:
        return {"kernel": None, "Q": 0, "S": 0, "path": None}
    path = {6: "1-D bulk copies both ways", 5: "bulk loads + STG.256 stores", 3: "swizzled TMA loads + STG.256 stores",
            2: "LDG.256 / STG.256"}.get(v >> 24, str(v >> 24))
    return {"kernel": "solve_chunked_kernel", "Q": (v >> 8) & 0xff, "S": (v >> 16) & 0xff, "path": path}


_ERR = {1: "invalid argument", 2: "zero or non-finite pivot", 3: "CUDA error", 4: "allocation failure",
        5: "problem needs more scratch than the library's static array holds (pent_noalloc_scratch_bytes)"}

_lib = None


class PentError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        super().__init__(f"libpent error {code} ({_ERR.get(code, '?')}){detail}")
        self.code = code


class SingularPivot(PentError):
    def __init__(self, row: int):
        super().__init__(2, f" at row {row}")
        self.row = row


class pent_step_params(C.Structure):
    _fields_ = [("kind", C.c_int), ("bc", C.c_int), ("form", C.c_int),
                ("r", C.c_double), ("sigma", C.c_double)]


class pent_forcing(C.Structure):
    _fields_ = [("kind", C.c_int), ("dt", C.c_double), ("t0", C.c_double),
                ("mu1", C.c_void_p), ("mu2", C.c_void_p)]


def lib() -> C.CDLL:
    """Load (building if needed) libpent.so.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.needs_build():
        path = _build.build()
    L = C.CDLL(path)
    vp, i64, ci = C.c_void_p, C.c_int64, C.c_int
    L.pent_factor.argtypes = [ci, vp, vp, vp, vp, vp, ci, C.POINTER(vp), C.POINTER(ci)]
    L.pent_factor_periodic.argtypes = [ci, vp, vp, vp, vp, vp, ci, C.POINTER(vp), C.POINTER(ci)]
    L.pent_handle_periodic.argtypes = [vp]
    L.pent_periodic_fused.argtypes = [vp, i64]
    L.pent_solve_batch.argtypes = [vp, i64, vp, vp, vp]
    L.pent_solve_batch_v.argtypes = [vp, i64, vp, vp, vp, ci]
    L.pent_solve_batch_host.argtypes = [vp, i64, vp, vp]
    L.pent_solve_batch_rows.argtypes = [vp, i64, vp, vp, vp]
    L.pent_solve_batch_rows_v.argtypes = [vp, i64, vp, vp, vp, ci]
    L.pent_destroy.argtypes = [vp]
    L.pent_destroy.restype = None
    L.pent_factor_solve_batch.argtypes = [ci, i64, vp, vp, vp, vp, vp, vp, vp, ci, vp, vp]
    L.pent_factor_solve_batch_ws.argtypes = [ci, i64, vp, vp, vp, vp, vp, vp, vp, ci, vp, vp, vp]
    L.pent_factor_solve_batch_noalloc.argtypes = [ci, i64, vp, vp, vp, vp, vp, vp, vp, ci, vp, vp]
    L.pent_noalloc_scratch_bytes.argtypes = []
    L.pent_noalloc_scratch_bytes.restype = i64
    L.pent_factor_batch.argtypes = [ci, i64, vp, vp, vp, vp, vp, ci, C.POINTER(vp), vp, vp]
    L.pent_solve_batch_multi.argtypes = [vp, vp, vp, vp]
    L.pent_step_batch.argtypes = [vp, C.POINTER(pent_step_params), i64, vp, vp, ci, vp]
    L.pent_step_batch_v.argtypes = [vp, C.POINTER(pent_step_params), i64, vp, vp, ci, vp, ci]
    L.pent_step_kernel_choice.argtypes = [vp, i64]
    L.pent_step_batch_forced.argtypes = [vp, C.POINTER(pent_step_params), C.POINTER(pent_forcing), i64, vp, vp, ci, vp]
    L.pent_step_batch_forced_v.argtypes = [vp, C.POINTER(pent_step_params), C.POINTER(pent_forcing), i64, vp, vp, ci,
                                           vp, ci]
    L.pent_adi_step_batch.argtypes = [vp, vp, vp, vp, ci, vp]
    L.pent_handle_n.argtypes = [vp]
    L.pent_handle_dtype.argtypes = [vp]
    L.pent_handle_m.argtypes = [vp]
    L.pent_handle_m.restype = i64
    L.pent_handle_device.argtypes = [vp]
    L.pent_handle_band.argtypes = [vp]
    L.pent_handle_exchange_depth.argtypes = [vp, ci]
    L.pent_handle_growth.argtypes = [vp, C.POINTER(C.c_double)]
    L.pent_release_thread_cache.argtypes = []
    L.pent_release_thread_cache.restype = None
    L.pent_handle_factors.argtypes = [vp] * 6
    L.pent_solve_kernel_choice.argtypes = [vp, i64]
    L.pent_solve_rows_kernel_choice.argtypes = [vp, i64]
    L.pent_launch_count.argtypes = [ci]
    L.pent_launch_count.restype = i64
    L.pent_version.restype = C.c_char_p
    _lib = L
    return L


def _check(rc: int):
    if rc != 0:
        detail = f", cudaError={lib().pent_last_cuda_error()}" if rc == 3 else ""
        raise PentError(rc, detail)


def _dt(t: torch.Tensor) -> int:
    if t.dtype == torch.float64:
        return PENT_F64
    if t.dtype == torch.float32:
        return PENT_F32
    raise TypeError("fp64 or fp32 tensors only")


def _stream(stream) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


def _batch(t: torch.Tensor, name: str, shape=None, dtype=None):
    """Every tensor whose pointer crosses the C ABI: contiguous, 2-D, on the CURRENT CUDA device (that is
    where the kernel is launched and where the handle's memory lives), and of the expected shape / dtype."""
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dim() == 2):
        raise ValueError(f"{name}: contiguous CUDA tensor of shape (N, M) expected (interleaved layout)")
    if t.device.index != torch.cuda.current_device():
        raise ValueError(f"{name}: tensor is on {t.device}, the current device is cuda:{torch.cuda.current_device()}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)}, expected {tuple(shape)}")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"{name}: dtype {t.dtype}, expected {dtype}")


def _vec(t: torch.Tensor, name: str, numel_min: int, dtype):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dtype
            and t.numel() >= numel_min and t.device.index == torch.cuda.current_device()):
        raise ValueError(f"{name}: contiguous {dtype} tensor of >= {numel_min} elements on the current CUDA device expected")


@dataclass
class Handle:
    """Owner of a pent_handle*.  Shared-A (from pent_factor) or per-system (pent_factor_batch)."""
    ptr: int
    N: int
    dtype: torch.dtype
    M: int = 0

    def __del__(self):
        if getattr(self, "ptr", 0) and _lib is not None:
            _lib.pent_destroy(self.ptr)
            self.ptr = 0

    def factors(self):
        """(eps, beta, alpha, gamma, delta) as fp64 CPU tensors (shared-A only)."""
        out = [torch.empty(self.N, dtype=torch.float64) for _ in range(5)]
        _check(lib().pent_handle_factors(self.ptr, *[o.data_ptr() for o in out]))
        return tuple(out)


def pent_factor(N: int, e, c, d, a, b) -> Handle:
    """Factor A = L R once.  e,c,d,a,b: 1-D tensors of length N (CPU or CUDA,
    fp64 or fp32), row-indexed diagonals in north_star's argument order."""
    ts = [torch.as_tensor(v) for v in (e, c, d, a, b)]
    dt = _dt(ts[1])
    ts = [t.to(ts[1].dtype).contiguous() for t in ts]
    if any(t.numel() != N for t in ts):
        raise ValueError("each diagonal must have N entries")
    if not torch.cuda.is_available():
        raise RuntimeError("pent_factor needs a CUDA device (no CPU fallback)")
    out = C.c_void_p()
    bad = C.c_int(-1)
    rc = lib().pent_factor(N, *[t.data_ptr() for t in ts], dt, C.byref(out), C.byref(bad))
    if rc == 2:
        raise SingularPivot(bad.value)
    _check(rc)
    return Handle(out.value, N, ts[1].dtype)


def pent_factor_periodic(N: int, e, c, d, a, b) -> Handle:
    """Set-up of the periodic (cyclic) solve, Eqs. 7a-12: every entry of every length-N
    diagonal is used (a[k] = A[k][(k-2) mod N], ...).  The handle works with pent_solve_batch,
    pent_solve_batch_host and pent_step_batch(kind=1)."""
    ts = [torch.as_tensor(v) for v in (e, c, d, a, b)]
    dt = _dt(ts[1])
    ts = [t.to(ts[1].dtype).contiguous() for t in ts]
    if any(t.numel() != N for t in ts):
        raise ValueError("each diagonal must have N entries")
    if not torch.cuda.is_available():
        raise RuntimeError("pent_factor_periodic needs a CUDA device (no CPU fallback)")
    out = C.c_void_p()
    bad = C.c_int(-1)
    rc = lib().pent_factor_periodic(N, *[t.data_ptr() for t in ts], dt, C.byref(out), C.byref(bad))
    if rc == 2:
        raise SingularPivot(bad.value)
    _check(rc)
    return Handle(out.value, N, ts[1].dtype)


def pent_solve_batch(h: Handle, M: int, f: torch.Tensor, x: torch.Tensor | None = None,
                     stream=None, kernel: int = KERNEL_AUTO) -> torch.Tensor:
    """Forward + backward sweeps for M systems; f, x of shape (N, M)."""
    _batch(f, "f", (h.N, M), h.dtype)
    if x is None:
        x = torch.empty_like(f)
    _batch(x, "x", (h.N, M), h.dtype)
    _check(lib().pent_solve_batch_v(h.ptr, M, f.data_ptr(), x.data_ptr(), _stream(stream), kernel))
    return x


ROWS_LDG = 1 << 24
ROWS_STG = 1 << 25
ROWS_TMA2D = 1 << 26


def pent_solve_batch_rows(h: Handle, M: int, f: torch.Tensor, x: torch.Tensor | None = None, stream=None,
                          kernel: int = KERNEL_AUTO) -> torch.Tensor:
    """Same solve on a system-major batch: f, x of shape (M, N), one system per row."""
    _batch(f, "f", (M, h.N), h.dtype)
    if x is None:
        x = torch.empty_like(f)
    _batch(x, "x", (M, h.N), h.dtype)
    _check(lib().pent_solve_batch_rows_v(h.ptr, M, f.data_ptr(), x.data_ptr(), _stream(stream), kernel))
    return x


def pent_solve_batch_host(h: Handle, M: int, f_host: torch.Tensor,
                          x_host: torch.Tensor | None = None) -> torch.Tensor:
    """Same with CPU tensors (pinned or pageable); copies are inside the call."""
    if f_host.is_cuda or not f_host.is_contiguous() or f_host.shape != (h.N, M) or f_host.dtype != h.dtype:
        raise ValueError("f_host: contiguous CPU tensor (N, M) of the handle's dtype expected")
    if x_host is None:
        x_host = torch.empty_like(f_host)
    if x_host.is_cuda or not x_host.is_contiguous() or x_host.shape != f_host.shape or x_host.dtype != h.dtype:
        raise ValueError("x_host: contiguous CPU tensor (N, M) of the handle's dtype expected")
    _check(lib().pent_solve_batch_host(h.ptr, M, f_host.data_ptr(), x_host.data_ptr()))
    return x_host


def pent_workspace_elems(N: int, M: int) -> int:
    """Elements of the optional workspace of pent_factor_solve_batch: 3*N*M', M' = M rounded up to 64."""
    return 3 * N * ((M + 63) // 64 * 64)


def pent_factor_solve_batch(N: int, M: int, e, c, d, a, b, f, x=None, info=None, stream=None,
                            workspace=None):
    """Per-system matrices, factor + solve fused.  All tensors (N, M) on CUDA.
    workspace: optional CUDA tensor of 3*N*M' elements, M' = M rounded up to a multiple of 64.  Returns (x, info) with info int32[M]:
    0 or first bad row + 1."""
    _dt(f)
    for t, n in zip((e, c, d, a, b, f), "ecdabf"):
        _batch(t, n, (N, M), f.dtype)
    if x is None:
        x = torch.empty_like(f)
    _batch(x, "x", (N, M), f.dtype)
    if info is None:
        info = torch.zeros(M, dtype=torch.int32, device=f.device)
    _vec(info, "info", M, torch.int32)
    if workspace is not None:
        _vec(workspace, "workspace", pent_workspace_elems(N, M), f.dtype)
    _check(lib().pent_factor_solve_batch_ws(N, M, e.data_ptr(), c.data_ptr(), d.data_ptr(),
                                            a.data_ptr(), b.data_ptr(), f.data_ptr(), x.data_ptr(),
                                            _dt(f), info.data_ptr(),
                                            0 if workspace is None else workspace.data_ptr(),
                                            _stream(stream)))
    return x, info


def pent_noalloc_scratch_bytes() -> int:
    """Size of the static device array behind pent_factor_solve_batch_noalloc (bytes)."""
    return int(lib().pent_noalloc_scratch_bytes())


def pent_factor_solve_batch_noalloc(N: int, M: int, e, c, d, a, b, f, x, info, stream=None):
    """pent_factor_solve_batch for callers that cannot allocate: the library allocates NOTHING in this call (its
    scratch is a static 32 MiB device array), so the caller passes x and info (int32[M]) as well.  PentError code 5 when
    3*N*ceil64(M)*itemsize exceeds pent_noalloc_scratch_bytes().  Calls that overlap on the GPU race on the array."""
    _dt(f)
    for t, n in zip((e, c, d, a, b, f, x), "ecdabfx"):
        _batch(t, n, (N, M), f.dtype)
    _vec(info, "info", M, torch.int32)
    _check(lib().pent_factor_solve_batch_noalloc(N, M, e.data_ptr(), c.data_ptr(), d.data_ptr(), a.data_ptr(),
                                                 b.data_ptr(), f.data_ptr(), x.data_ptr(), _dt(f), info.data_ptr(),
                                                 _stream(stream)))
    return x, info


def pent_factor_batch(N: int, M: int, e, c, d, a, b, info=None, stream=None):
    """Per-system factorisations kept in a handle for repeated pent_solve_batch_multi calls."""
    _dt(c)
    for t, n in zip((e, c, d, a, b), "ecdab"):
        _batch(t, n, (N, M), c.dtype)
    if info is None:
        info = torch.zeros(M, dtype=torch.int32, device=c.device)
    _vec(info, "info", M, torch.int32)
    out = C.c_void_p()
    _check(lib().pent_factor_batch(N, M, e.data_ptr(), c.data_ptr(), d.data_ptr(), a.data_ptr(),
                                   b.data_ptr(), _dt(c), C.byref(out), info.data_ptr(),
                                   _stream(stream)))
    return Handle(out.value, N, c.dtype, M), info


def pent_solve_batch_multi(h: Handle, f: torch.Tensor, x: torch.Tensor | None = None, stream=None):
    _batch(f, "f", (h.N, h.M), h.dtype)
    if x is None:
        x = torch.empty_like(f)
    _batch(x, "x", (h.N, h.M), h.dtype)
    _check(lib().pent_solve_batch_multi(h.ptr, f.data_ptr(), x.data_ptr(), _stream(stream)))
    return x


def pent_step_batch(h: Handle, M: int, c: torch.Tensor, nsteps: int, *, kind: int = 0, bc: int = 1,
                    form: int = 1, r: float = 0.0, sigma: float = 0.0,
                    scratch: torch.Tensor | None = None, stream=None,
                    kernel: int = KERNEL_AUTO, forcing=None) -> torch.Tensor:
    """nsteps fused steps (RHS + solve in one kernel) in place on c (N, M).  See include/pent.h.
    forcing = (mu1, mu2, dt, t0): the forced Cahn-Hilliard equation with per-system
    parameters mu1, mu2 (CUDA tensors of M elements of the handle's dtype); pent_step_batch_forced."""
    _batch(c, "c", (h.N, M), h.dtype)
    p = pent_step_params(kind, bc, form, r, sigma)
    if scratch is not None:
        _vec(scratch, "scratch", h.N * M, h.dtype)
    sp = 0 if scratch is None else scratch.data_ptr()
    if forcing is None:
        _check(lib().pent_step_batch_v(h.ptr, C.byref(p), M, c.data_ptr(), sp, nsteps, _stream(stream), kernel))
        return c
    mu1, mu2, dt, t0 = forcing
    _vec(mu1, "mu1", M, h.dtype)
    _vec(mu2, "mu2", M, h.dtype)
    g = pent_forcing(1, float(dt), float(t0), mu1.data_ptr(), mu2.data_ptr())
    _check(lib().pent_step_batch_forced_v(h.ptr, C.byref(p), C.byref(g), M, c.data_ptr(), sp, nsteps,
                                          _stream(stream), kernel))
    return c


def pent_adi_step_batch(hx: Handle, hy: Handle, u: torch.Tensor, nsteps: int, scratch: torch.Tensor | None = None,
                        stream=None) -> torch.Tensor:
    """nsteps Peaceman-Rachford ADI steps in place on the field u of shape (Ny, Nx) = (hy.N, hx.N)
    (include/pent.h)."""
    _batch(u, "u", (hy.N, hx.N), hx.dtype)
    if hy.dtype != hx.dtype:
        raise ValueError("hx and hy must have one dtype")
    if scratch is not None:
        _vec(scratch, "scratch", hx.N * hy.N, hx.dtype)
    _check(lib().pent_adi_step_batch(hx.ptr, hy.ptr, u.data_ptr(), 0 if scratch is None else scratch.data_ptr(),
                                     nsteps, _stream(stream)))
    return u


def handle_growth(h: Handle):
    """(max|Phi|, max|X|, max|Psi|) of pent_handle_growth: the stability figures of the chunked evaluation."""
    out = (C.c_double * 3)()
    _check(lib().pent_handle_growth(h.ptr, out))
    return tuple(out)


def launch_count(reset: bool = False) -> int:
    return int(lib().pent_launch_count(1 if reset else 0))
