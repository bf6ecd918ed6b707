"""Build paper_2411_02206_b200/libtmd.so from csrc/ with nvcc for sm_100a (in-tree; the .so is git-ignored but ships
to the GPU box with the repository snapshot).

Flags that matter for bit-exactness with the encoder (DESIGN.md §3 reading 12): --fmad=false (no FMA contraction),
-prec-div=true -prec-sqrt=true -ftz=false (IEEE division / square root, denormals kept).  The kernels additionally use
the explicit __f*_rn intrinsics, which are never contracted.
"""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtmd.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
         "--fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
         "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps() -> list[str]:
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "tmd.h")]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    r = subprocess.run([NVCC, *FLAGS, "-o", tmp, *sources()], capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
