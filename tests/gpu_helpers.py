"""Helpers of the GPU parity tests: guard-banded device buffers and the error measures.

compute-sanitizer is closed on this pool, so out-of-bounds stores are caught the plain way: every
batch array a test hands to the library (f, x, c, diagonals, info, workspace) lives INSIDE a larger
allocation with 1 MiB of sentinel words on each side, the array itself starts as sentinels too
(an output element the kernel never wrote stays a NaN and fails the comparison), and after the
call both bands must still hold the sentinel bit pattern.  The 1 MiB offset keeps the 16-byte
alignment the TMA path needs, so the kernels under test are the ones bench.py times.
"""
from __future__ import annotations

import numpy as np
import torch

GUARD_BYTES = 1 << 20
_SENT = {8: 0x7FF8DEADBEEF0001, 4: 0x7FC0BEEF}          # quiet NaNs with a recognisable payload
_IDT = {8: torch.int64, 4: torch.int32}


class Guarded:
    """A CUDA tensor of `shape` carved out of a sentinel-filled allocation."""

    def __init__(self, shape, dtype=torch.float64, src=None):
        esz = torch.empty((), dtype=dtype).element_size()
        self.g = GUARD_BYTES // esz
        self.n = int(np.prod(shape)) if len(shape) else 1
        self.buf = torch.empty(self.n + 2 * self.g, dtype=dtype, device="cuda")
        self.ibuf = self.buf.view(_IDT[esz])
        self.sent = _SENT[esz]
        self.ibuf.fill_(self.sent)
        self.t = self.buf[self.g:self.g + self.n].view(*shape)
        if src is not None:
            self.t.copy_(torch.as_tensor(np.ascontiguousarray(src)).to(dtype))

    def check(self, what=""):
        torch.cuda.synchronize()
        lo = self.ibuf[:self.g]
        hi = self.ibuf[self.g + self.n:]
        assert bool((lo == self.sent).all()), f"store below the array {what}"
        assert bool((hi == self.sent).all()), f"store beyond the array {what}"

    def numpy(self):
        return self.t.cpu().numpy()


def guarded(src, dtype=torch.float64) -> Guarded:
    src = np.ascontiguousarray(src)
    return Guarded(src.shape, dtype, src)


def check_all(*gs):
    for g in gs:
        if g is not None:
            g.check()


def normwise(x, ref):
    """max over systems of max_k |x - ref| / max_k |ref|   (interleaved (N, M) arrays; reading C-6)."""
    return float(np.max(np.max(np.abs(x - ref), axis=0) / np.max(np.abs(ref), axis=0)))


def pinned_tol(floor, oracle64, truth):
    """Parity tolerance tied to a measurement (reading C-15): the north_star bar `floor`, or twice
    the distance of the fp64 oracle from the long-double truth on the same inputs when that is larger."""
    return max(floor, 2.0 * normwise(oracle64, truth))
