"""Build libpent.so (sm_100a only) in-tree with nvcc.  `python -m paper_1807_07382_b200.build`."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libpent.so")
SOURCES = ["pent_factor.cu", "pent_solve_tps.cu", "pent_solve_chunked.cu", "pent_step.cu", "pent_step_chunked.cu", "pent_periodic.cu", "pent_solve_chunked_periodic.cu",
           "pent_api.cu", "pent_adi.cu", "pent_solve_chunked_rows.cu", "pent_solve_chunked_epi.cu"]


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: libpent cannot be built (there is no CPU fallback)")
    return p


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "pent.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu to an object file (in parallel) and link libpent.so."""
    if not force and not needs_build():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(PKG, "build")
    os.makedirs(objdir, exist_ok=True)
    common = [nvcc_path(), "-O3", "-std=c++17", "-lineinfo",
              "-gencode", "arch=compute_100a,code=sm_100a",
              "-Xcompiler", "-fPIC",
              "-I", os.path.join(ROOT, "include"), "-I", CSRC] + os.environ.get("PENT_NVCC_FLAGS", "").split()
    if verbose:
        common.insert(1, "-Xptxas=-v")

    def compile_one(src):
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        r = subprocess.run(common + ["-c", os.path.join(CSRC, src), "-o", obj], capture_output=True, text=True)
        return src, obj, r

    with ThreadPoolExecutor(max_workers=min(8, len(SOURCES))) as ex:
        results = list(ex.map(compile_one, SOURCES))
    failed = False
    for src, _, r in results:
        if verbose or r.returncode != 0:
            sys.stderr.write(f"---- {src}\n" + r.stdout + r.stderr)
        failed |= r.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libpent.so")
    r = subprocess.run([nvcc_path(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] +
                       [obj for _, obj, _ in results], capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed linking libpent.so")
    return LIB


def build_ubench() -> str:
    """The standalone microbenchmark of csrc/pent_ubench.cu (FP64 FMA, shared-memory load and shuffle rates)."""
    out = os.path.join(PKG, "pent_ubench")
    r = subprocess.run([nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a",
                        "-o", out, os.path.join(CSRC, "pent_ubench.cu")], capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed building pent_ubench")
    return out


if __name__ == "__main__":
    if "--ubench" in sys.argv:
        print(build_ubench())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
