"""Build the CUDA library (csrc/*.cu -> libomerf.so, in-tree) for sm_100a with nvcc.

nvcc cross-compiles without a GPU.  The library is plain C-ABI (include/omerf.h); no torch headers.
"""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libomerf.so")
LIB_CHECKED = os.path.join(HERE, "libomerf_checked.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",            # colour path may contract; the decision path uses explicit *_rn intrinsics
    "-Xcompiler", "-fPIC", "-shared",
    "-Xptxas", "-v",
]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """checked=True builds libomerf_checked.so: the same sources with -DOMERF_CHECKED (device-side range checks of every
    index of the render kernels, csrc/omerf_render.cu), used by tests/test_gpu_checked.py."""
    lib = LIB_CHECKED if checked else LIB
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "omerf.h")]
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [NVCC, *NVCC_FLAGS, *(["-DOMERF_CHECKED"] if checked else []), "-o", tmp, *sources()]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stderr[-4000:])
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose=True))
    print(build(force=True, checked=True))
