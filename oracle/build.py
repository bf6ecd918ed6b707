"""Build oracle/liborc.so from oracle/tmd_oracle.c and oracle/tmd_ans_oracle.c with gcc (TEST INFRASTRUCTURE ONLY).

-ffp-contract=off is mandatory: gcc's default (-ffp-contract=fast) may fuse a*b+c into an FMA on FMA-capable
targets, which would break the "every op is one IEEE binary32 RN operation" rule of the model.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tmd_oracle.c")
SRCS = [SRC, os.path.join(HERE, "tmd_ans_oracle.c")]
LIB = os.path.join(HERE, "liborc.so")
CFLAGS = ["-std=c11", "-O2", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math", "-fno-unsafe-math-optimizations",
          "-Wall", "-Wextra", "-Wno-unused-parameter"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(f) for f in SRCS):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run(["gcc", *CFLAGS, "-o", tmp, *SRCS, "-lm"], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
