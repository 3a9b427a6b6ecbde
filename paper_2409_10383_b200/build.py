"""Builds the C-ABI library `libz4c.so` in-tree with nvcc for sm_100a (no torch extension machinery:
the boundary is plain C, include/z4c.h)."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libz4c.so")            # 3 ghosts, 4th-order stencils (BASELINE configs)
LIB_NG4 = os.path.join(HERE, "libz4c_ng4.so")    # 4 ghosts, 6th-order stencils (NEXT-1, the paper's production scheme)
LIBS = {3: LIB, 4: LIB_NG4}
SOURCES = ["z4c_lib.cu"]
HEADERS = ["z4c_math.cuh", "z4c_rhs.cuh", "z4c_pack.cuh", "z4c_kernels.cuh", "z4c_rhs_tiled.cuh",
           os.path.join("..", "..", "include", "z4c.h")]
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "--fmad=true", "-Xcompiler", "-fPIC", "--shared", "-cudart", "shared"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the Z4c library needs the CUDA toolkit to build")


def is_stale() -> bool:
    if not all(os.path.exists(l) for l in LIBS.values()):
        return True
    t = min(os.path.getmtime(l) for l in LIBS.values())
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    for ng, lib in LIBS.items():
        cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              [f"-DZ4C_NG={ng}", "-o", lib] + [os.path.join(CSRC, s) for s in SOURCES]
        res = subprocess.run(cmd, cwd=CSRC, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
        if verbose:
            print(res.stderr)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
