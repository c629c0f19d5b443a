"""Build step: compile csrc/*.cu into csrc/libtpcclus.so with nvcc for sm_100a (in-tree)."""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(CSRC, "libtpcclus.so")
LIB_CHECKED = os.path.join(CSRC, "libtpcclus_checked.so")   # -DTPCCLUS_CHECKED: bounds-checking device asserts
SOURCES = ["tpcclus.cu"]
DEPS = ["tpcclus.cu", "tpcclus_kernels.cuh", "tpcclus_tile.cuh", "tpcclus_select.cuh", os.path.join("..", "..", "include", "tpcclus.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC",
    "-cudart", "static",          # no libcudart / libcuda link dependency: loads on a CPU-only box
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def is_stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    lib = LIB_CHECKED if checked else LIB
    if not force and not is_stale(lib):
        return lib
    tmp = lib + ".tmp%d" % os.getpid()
    cmd = [_nvcc(), *NVCC_FLAGS, *(["-DTPCCLUS_CHECKED"] if checked else []), *(["-Xptxas", "-v"] if verbose else []),
           *[os.path.join(CSRC, s) for s in SOURCES], "-o", tmp]
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose=True))
