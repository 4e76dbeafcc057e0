"""Writes tests/golden/config0_oracle.txt from the CPU oracle ALONE (never from the CUDA path).

    python tests/golden/make_golden.py

The paper (arxiv 2404.09531) prints no worked numeric example for the render path (R4, R10, R13,
R19 are "parity unpinned by the paper"), so there is no paper value to store here.  This file is a drift guard: the
oracle's output on BASELINE.json configs[0] (brute loop), so that a later change to the oracle's arithmetic cannot
pass unnoticed - such a change must regenerate this file in a commit that names the passage or DESIGN.md reading
that justifies it.
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import synth  # noqa: E402


def summary():
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    r = oracle.OracleScene(sc).render(cams, W, H, mode="brute")
    ns, rgb = r["nsamples"][0], r["rgb"][0]
    lines = ["# oracle output on BASELINE.json configs[0] (128x128, brute loop); written by tests/golden/make_golden.py",
             f"total_samples {int(ns.sum())}",
             f"nsamples_sha256 {hashlib.sha256(np.ascontiguousarray(ns, dtype=np.uint32).tobytes()).hexdigest()}",
             "row_sums " + " ".join(str(int(x)) for x in ns.sum(axis=1)),
             "rgb_mean " + " ".join(f"{x:.12f}" for x in rgb.reshape(-1, 3).mean(axis=0)),
             "rgb_row64 " + " ".join(f"{x:.9f}" for x in rgb[64, ::16].reshape(-1))]
    return "\n".join(lines) + "\n"


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_oracle.txt")
    open(path, "w").write(summary())
    print("wrote", path)
