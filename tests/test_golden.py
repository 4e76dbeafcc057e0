"""Drift guard: the oracle still produces the stored configs[0] summary (tests/golden/config0_oracle.txt, written by
tests/golden/make_golden.py from the oracle alone), and on a GPU the CUDA path reproduces it through the C-ABI."""
import hashlib
import os

import numpy as np
import pytest

import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config0_oracle.txt")


def _gold():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        key, *vals = line.split()
        out[key] = vals
    return out


def test_oracle_matches_golden_file():
    import oracle
    g = _gold()
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    r = oracle.OracleScene(sc).render(cams, W, H, mode="brute")
    ns, rgb = r["nsamples"][0], r["rgb"][0]
    assert int(ns.sum()) == int(g["total_samples"][0])
    assert hashlib.sha256(np.ascontiguousarray(ns, dtype=np.uint32).tobytes()).hexdigest() == g["nsamples_sha256"][0]
    assert [int(x) for x in ns.sum(axis=1)] == [int(x) for x in g["row_sums"]]
    assert np.allclose(rgb.reshape(-1, 3).mean(axis=0), [float(x) for x in g["rgb_mean"]], atol=1e-10)
    assert np.allclose(rgb[64, ::16].reshape(-1), [float(x) for x in g["rgb_row64"]], atol=1e-8)


@pytest.mark.gpu
def test_cuda_path_matches_golden_file():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2404_09531_b200 as omerf
    g = _gold()
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    with omerf.scene_create(sc) as h:
        rgb, ns = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
    ns = ns.cpu().numpy().view(np.uint32)[0]
    rgb = rgb.cpu().numpy().astype(np.float64)[0]
    assert hashlib.sha256(np.ascontiguousarray(ns).tobytes()).hexdigest() == g["nsamples_sha256"][0]   # bit-exact counts
    assert np.abs(rgb[64, ::16].reshape(-1) - np.array([float(x) for x in g["rgb_row64"]])).max() <= 2e-3
    assert np.abs(rgb.reshape(-1, 3).mean(axis=0) - np.array([float(x) for x in g["rgb_mean"]])).max() <= 2e-3
