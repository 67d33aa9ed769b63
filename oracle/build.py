"""Compile oracle/hyb_oracle.c -> oracle/libhyb_oracle.so (gcc, -ffp-contract=off, OpenMP)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hyb_oracle.c")
LIB = os.path.join(HERE, "libhyb_oracle.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "hyb_oracle.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wno-maybe-uninitialized", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
