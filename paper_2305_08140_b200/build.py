"""Build csrc/libnepzbl.so for sm_100a with nvcc (in-tree; the .so travels to the GPU box)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libnepzbl.so")
SOURCES = ["nepzbl.cu", "no_alloc.cu"]
HEADERS = ["common.cuh", "neighbor.cuh", "descriptor.cuh", "force.cuh", "integrate.cuh", "wigner_seitz.cuh", "descriptor_split.cuh", "site_fp64.cuh", "stage.cuh", "tc05.cuh", "descriptor_tc.cuh", "descriptor_split_tc.cuh"]


# the same sources with -DNEPZBL_CHECKED: bounds checks on every gathered index (common.cuh: NZ_CHECK); selected with
# NEPZBL_LIB=checked at import of the binding (tests/test_gpu_checked.py)
LIB_CHECKED = os.path.join(CSRC, "libnepzbl_checked.so")


def nvcc_command(verbose: bool = False, checked: bool = False) -> list[str]:
    cmd = ["nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", LIB_CHECKED if checked else LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    if checked:
        cmd[1:1] = ["-DNEPZBL_CHECKED"]
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    return cmd


def is_stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(ROOT, "include", "nepzbl.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    lib = LIB_CHECKED if checked else LIB
    if force or is_stale(lib):
        subprocess.run(nvcc_command(verbose, checked), check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
