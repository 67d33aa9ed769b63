"""Compile oracle/hyb_oracle.c -> oracle/libhyb_oracle.so (gcc, -ffp-contract=off, OpenMP)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hyb_oracle.c")
LIB = os.path.join(HERE, "libhyb_oracle.so")
LIB_SAN = os.path.join(HERE, "libhyb_oracle_san.so")


def build(force: bool = False, sanitize: bool = False) -> str:
    """sanitize=True: a second library built with -fsanitize=address,undefined (tests/test_oracle_sanitizers.py
    runs the oracle's own tests against it; the process must preload libasan, see sanitizer_env())."""
    lib = LIB_SAN if sanitize else LIB
    deps = [SRC, os.path.join(HERE, "hyb_oracle.h")]
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps):
        return lib
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wno-maybe-uninitialized"]
    if sanitize:
        cmd += ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"]
    subprocess.run(cmd + ["-o", lib, SRC, "-lm"], check=True)
    return lib


def sanitizer_env() -> dict:
    """environment for a python process that loads the sanitized oracle (HYB_ORACLE_SANITIZE=1)"""
    def so(name):
        return subprocess.run(["gcc", f"-print-file-name={name}"], check=True, capture_output=True, text=True).stdout.strip()
    return {"HYB_ORACLE_SANITIZE": "1", "LD_PRELOAD": so("libasan.so") + ":" + so("libubsan.so"),
            # CPython itself leaks at exit and numpy traps some signals; only the oracle's own errors matter
            "ASAN_OPTIONS": "detect_leaks=0:abort_on_error=1:handle_segv=0",
            "UBSAN_OPTIONS": "halt_on_error=1:print_stacktrace=1"}


if __name__ == "__main__":
    print(build(force=True))
