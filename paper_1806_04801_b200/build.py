"""Builds libhsma_b200.so (the C-ABI of include/hsma.h) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The library links cudart statically and has no torch
dependency; `python -m paper_1806_04801_b200.build` rebuilds it."""
from __future__ import annotations

import fcntl
import os
import shutil
import subprocess

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libhsma_b200.so")
SOURCES = ["hsma_api.cu"]
HEADERS = ["common.cuh", "sum_kernels.cuh", "lattice_kernels.cuh", "fit_kernels.cuh", "fmm_kernels.cuh", "fmm_host.cuh", "geometry.h", "peak.cuh"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(ROOT, "include", "hsma.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Several ranks of a torchrun job may find the library stale at once: the build runs under an exclusive file
    lock, writes to a per-process temporary name and is moved into place atomically, so no rank can ever load a
    half-written library (a rank that waited for the lock finds it fresh and returns)."""
    if not force and not is_stale():
        return LIB
    with open(os.path.join(PKG, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            if not force and not is_stale():
                return LIB
            tmp = f"{LIB}.{os.getpid()}.tmp"
            cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                   "--extended-lambda", "-I" + os.path.join(ROOT, "include"), "-shared", "-Xcompiler", "-fPIC",
                   "-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
                print(" ".join(cmd))
            try:
                subprocess.check_call(cmd)
                os.replace(tmp, LIB)
            finally:
                if os.path.exists(tmp):
                    os.unlink(tmp)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
