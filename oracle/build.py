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

LIB_SAN = os.path.join(HERE, "libomerf_oracle_san.so")

CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-std=c11",
          "-Wall", "-Wextra"]
# ORACLE_SANITIZE=1: the same source, same arithmetic flags, under AddressSanitizer + UndefinedBehaviorSanitizer
# (SURVEY.md sec. 5 "sanitizers for the oracle").  Any finding aborts the process.  The host is python, so the ASan
# runtime has to be preloaded and python's own leaks silenced:
#   ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
#       python -m pytest tests -q -m "not gpu"
SAN_FLAGS = ["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"]


def sanitized() -> bool:
    return os.environ.get("ORACLE_SANITIZE", "0") not in ("", "0")


def build(force: bool = False) -> str:
    lib, flags = (LIB_SAN, CFLAGS + SAN_FLAGS) if sanitized() else (LIB, CFLAGS)
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", *flags, "-o", tmp, SRC, "-lm"])
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force=True))
