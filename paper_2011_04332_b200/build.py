"""Compile the CUDA library in-tree: paper_2011_04332_b200/libnpfem_b200.so (sm_100a only).

nvcc cross-compiles without a GPU, so this also runs on the CPU build box.  The built .so is
git-ignored but travels to the GPU box with the repo snapshot.
"""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnpfem_b200.so")
SOURCES = ["npfem_plan.cpp", "npfem_kernels.cu", "npfem_api.cu", "npfem_peak.cu", "npfem_converged.cu"]
HEADERS = ["npfem_internal.h", "npfem_kernels.cuh", "npfem_device.cuh", os.path.join(ROOT, "include", "npfem.h")]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the npFEM CUDA library cannot be built")
    return exe


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [
        h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Build libnpfem_b200.so if missing or older than its sources; return its path."""
    if not force and not _stale():
        return LIB
    cmd = [_nvcc(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    extra = os.environ.get("NPFEM_NVCC_FLAGS", "")   # diagnostic builds, e.g. -DNPFEM_PHASE_CLOCKS
    if extra:
        cmd += extra.split()
    if verbose:
        cmd += ["-Xptxas", "-v"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
