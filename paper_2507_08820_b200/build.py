"""Build the CUDA C-ABI library in-tree: paper_2507_08820_b200/csrc/librflbm.so (sm_100a only).

nvcc cross-compiles without a GPU.  `python -m paper_2507_08820_b200.build` or build() from Python.
The step kernels (~380 template instantiations) are compiled as 24 translation units, one per (precision, phase,
tile width),
in parallel with the C-ABI translation unit, then linked into one shared library.
"""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(CSRC, "librflbm.so")
SOURCES = ["rflbm.cu", "rflbm_step_inst.cu", "rflbm_static.cu"]
HEADERS = ["rflbm_lattice.cuh", "rflbm_fastmath.cuh", "rflbm_rng.cuh", "rflbm_collide.cuh", "rflbm_kernels.cuh",
           "rflbm_step_tma.cuh", "rflbm_host.cuh", os.path.join("..", "..", "include", "rflbm.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
# (object name, source, extra defines)
UNITS = [("rflbm.o", "rflbm.cu", []), ("rflbm_static.o", "rflbm_static.cu", [])] + [
    (f"step_{r}_{p}_{tx}.o", "rflbm_step_inst.cu", [f"-DRFLBM_INST_REAL={r}", f"-DRFLBM_INST_PHASE={p}", f"-DRFLBM_INST_TX={tx}"])
    for tx in (128, 0, 64, 32) for r in ("double", "float") for p in (0, 1, 2)]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []

    def compile_unit(unit):
        obj, src, defs = unit
        cmd = [nvcc] + NVCC_FLAGS + extra + defs + ["-c", "-o", os.path.join(OBJ, obj), src]
        r = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        return cmd, r

    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as pool:
        results = list(pool.map(compile_unit, UNITS))
    for cmd, r in results:
        if verbose or r.returncode != 0:
            print(" ".join(cmd))
            print(r.stdout + r.stderr)
        if r.returncode != 0:
            raise subprocess.CalledProcessError(r.returncode, cmd, r.stdout, r.stderr)
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [os.path.join(OBJ, u[0]) for u in UNITS]
    subprocess.run(link, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
