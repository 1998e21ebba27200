"""Compile the CPU oracle (oracle/wilson_clover.c) into oracle/liboracle.so with gcc.

TEST INFRASTRUCTURE.  Building the checker is not using it: only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
load the result.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "wilson_clover.c")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


def build_sanitized() -> str:
    """The same source under AddressSanitizer + UndefinedBehaviorSanitizer (no OpenMP, -O1): used by
    tests/test_oracle_sanitizers.py in a subprocess with libasan preloaded (ORACLE_LIB selects it)."""
    out = os.path.join(HERE, "liboracle_asan.so")
    if os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(SRC):
        return out
    cmd = ["gcc", "-O1", "-g", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra", "-fno-omit-frame-pointer",
           "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-Wno-unknown-pragmas",
           "-o", out, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return out


if __name__ == "__main__":
    print(build(force=True))
