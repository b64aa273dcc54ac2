"""Compile the C oracle into oracle/libhines_oracle.so with gcc.

ORACLE -- TEST INFRASTRUCTURE.  No fast-math, FP contraction off, so the arithmetic is
exactly what hines_oracle.c writes (one rounding per operation).
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["hines_oracle.c", "tables_oracle.c", "split_oracle.c", "reroot_oracle.c"]
LIB = os.path.join(HERE, "libhines_oracle.so")
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
          "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    srcs = [os.path.join(HERE, s) for s in SOURCES]
    if not force and os.path.exists(LIB):
        t = os.path.getmtime(LIB)
        if all(os.path.getmtime(s) <= t for s in srcs + [os.path.abspath(__file__)]):
            return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", *CFLAGS, *srcs, "-o", tmp, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
