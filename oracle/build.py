"""Build the CPU oracle (plain C + OpenMP) into oracle/libomerf_oracle.so.

TEST INFRASTRUCTURE: called by tests/, __graft_entry__.build()/smoke() and bench.py's
cpu_baseline / --impl reference legs only.  `-ffp-contract=off`, no fast-math: every
fp32 step of the decision path must be one correctly rounded IEEE operation.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "omerf_oracle.c")
LIB = os.path.join(HERE, "libomerf_oracle.so")

CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-std=c11",
          "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, SRC, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
