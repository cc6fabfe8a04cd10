"""Compile the CPU oracle (test infrastructure) into oracle/libflod_oracle.so with gcc.

Flags matter: -ffp-contract=off and no -ffast-math keep every fp32 operation of
the canonical geometry sequence a single correctly rounded IEEE operation; x86-64 SSE arithmetic
has no excess precision.  -O2 + OpenMP over tiles is only there so that it finishes in seconds.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "flod_oracle.c")
LIB = os.path.join(HERE, "libflod_oracle.so")

CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
          "-fexcess-precision=standard", "-Wall", "-Wextra", "-Wno-unused-parameter"]


def build_oracle(force: bool = False) -> str:
    if (not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", *CFLAGS, SRC, "-o", tmp, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_oracle(force=True))
