"""Build the CUDA C-ABI library in-tree: paper_2507_08820_b200/csrc/librflbm.so (sm_100a only).

nvcc cross-compiles without a GPU.  `python -m paper_2507_08820_b200.build` or build() from Python.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "librflbm.so")
SOURCES = ["rflbm.cu"]
HEADERS = ["rflbm_lattice.cuh", "rflbm_fastmath.cuh", "rflbm_rng.cuh", "rflbm_collide.cuh", "rflbm_kernels.cuh", "rflbm_step_tma.cuh",
           os.path.join("..", "..", "include", "rflbm.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
    subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
