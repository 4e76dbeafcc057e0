"""Pins of the oracle's soft occupancy variant (Eq. 6-8), -m "not gpu".

The pins do not re-call the oracle's mask routine: Eq. 6 is typed here as the paper's four literal cases
(numpy, float64) and the compositing weights come from the closed form of a constant-density slab.
"""
import math

import numpy as np
import pytest

import oracle
import synth


def _eq6_literal(z, zmin, zmax, eps, q=2):
    """Eq. 6 exactly as printed, valid when zmax - zmin >= 2 eps."""
    if zmin + eps <= z <= zmax - eps:
        return 1.0
    if z < zmin or z > zmax:
        return 0.0
    if zmin <= z <= zmin + eps:
        return (z - zmin) ** q / eps ** q
    return (zmax - z) ** q / eps ** q


def _zero_mlp(sc):
    """G == sigmoid(0) = 1/2 for every input, so rgb - 1/2 is the accumulated diffuse colour when bg = 0."""
    for nm in ("W0", "b0", "W1", "b1", "W2", "b2"):
        getattr(sc, nm)[...] = 0.0
    return sc


@pytest.mark.parametrize("eps", [0.25, 0.6, 1.0])
def test_soft_mask_closed_form_on_constant_slab(eps):
    """Straight-down rays through a flat slab [za, zb] of constant density and colour:
    omega_k = T^k (1 - T1) with T1 = exp(-tau step); Eq. 8 gives D = sum_k M(z_k) omega_k c."""
    za, zb, step = 1.0, 3.0, 0.125
    fill = [128, 120, 110, 125, 128, 128, 128, 128]       # small density: the ray crosses the whole slab
    sc = _zero_mlp(synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=za, h_up=zb, fill=fill, step=step,
                                      bg=(0.0, 0.0, 0.0), seed=3))
    cam = np.array([4.1, 3.9, 6.03, 1, 0, 0, 0, 1, 0, 0, 0, -1, 200.0, 200.0, 1.5, 1.5], dtype=np.float32)
    soft = oracle.OracleScene(sc, soft_eps=eps).render(cam, 3, 3, mode="brute", aux=True)
    hard = oracle.OracleScene(sc).render(cam, 3, 3, mode="brute", aux=True)
    # M weights colours only: the samples, the transmittance and the termination are those of the binary mask
    assert np.array_equal(soft["nsamples"], hard["nsamples"])
    assert np.array_equal(soft["Q"], hard["Q"]) and np.array_equal(soft["T_end"], hard["T_end"])
    tau = math.exp(4.0 * (fill[0] * 28.0 / 255.0 - 14.0))
    c = 1.0 / (1.0 + np.exp(-4.0 * (np.array(fill[1:4]) * 28.0 / 255.0 - 14.0)))
    oz = float(cam[2])
    ks = [k for k in range(200) if za <= oz - (k + 0.5) * step <= zb and 0 <= oz - (k + 0.5) * step < 4.0]
    assert len(ks) == int(hard["nsamples"][0, 1, 1]) == 16
    T1 = math.exp(-tau * step)
    D = np.zeros(3)
    for i, k in enumerate(ks):
        z = np.float32(oz) - np.float32((k + 0.5) * step)          # exact in fp32: the oracle's z
        D += _eq6_literal(float(z), za, zb, eps) * (T1 ** i) * (1.0 - T1) * c
    got = soft["rgb"][0, 1, 1] - 0.5
    # od is rounded to 2^-20 in the transmittance (R8): relative 1e-6 per sample
    assert np.allclose(got, D, rtol=2e-5, atol=1e-9)
    assert np.all(soft["rgb"][0, 1, 1] < hard["rgb"][0, 1, 1])       # buffers remove weight


def test_soft_mask_function_properties():
    """0 <= M <= 1, M = 0 outside, M = 1 in the core, continuous and monotone in each buffer, symmetric, and the
    thin-interval reading R23 (min of the two ramps) agrees with Eq. 6 wherever Eq. 6 is unambiguous."""
    rng = np.random.default_rng(0)
    lo = (1.0 + rng.random((9, 9))).astype(np.float32)
    hi = (lo + 0.1 + 2.0 * rng.random((9, 9))).astype(np.float32)    # some intervals are thinner than 2 eps
    eps = 0.5
    sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=lo, h_up=hi, seed=1)
    O = oracle.OracleScene(sc, soft_eps=eps)
    for _ in range(4000):
        ix, iy = rng.integers(0, 9, 2)
        z = np.float32(rng.uniform(0.0, 4.0))
        p = np.array([ix + rng.uniform(-0.45, 0.45), iy + rng.uniform(-0.45, 0.45), z], dtype=np.float32)
        p[:2] = np.clip(p[:2], 0.0, 7.999)
        zmin, zmax = float(lo[ix, iy]), float(hi[ix, iy])
        m = O.soft_mask(p)
        assert 0.0 <= m <= 1.0
        assert (m > 0.0) == (zmin < float(z) < zmax) or float(z) in (zmin, zmax)
        if zmax - zmin >= 2 * eps:
            assert m == pytest.approx(_eq6_literal(float(z), zmin, zmax, eps), abs=1e-12)
        else:
            a, b = (float(z) - zmin) / eps, (zmax - float(z)) / eps
            if zmin <= float(z) <= zmax:
                assert m == pytest.approx(min(1.0, a * a, b * b), abs=1e-12)
    # symmetry about the interval centre and monotonicity in the lower buffer
    sc2 = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=1.0, h_up=3.0, seed=1)
    O2 = oracle.OracleScene(sc2, soft_eps=eps)
    zs = np.linspace(1.0, 1.5, 33, dtype=np.float32)
    ms = [O2.soft_mask(np.array([4.0, 4.0, z], dtype=np.float32)) for z in zs]
    assert all(a <= b for a, b in zip(ms, ms[1:])) and ms[0] == 0.0 and ms[-1] == 1.0
    for z in (1.1, 1.3, 1.7):
        lo_side = O2.soft_mask(np.array([4.0, 4.0, z], dtype=np.float32))
        hi_side = O2.soft_mask(np.array([4.0, 4.0, 4.0 - z], dtype=np.float32))
        assert lo_side == pytest.approx(hi_side, abs=1e-6)


def test_soft_mask_reduces_to_binary_and_is_monotone_in_eps():
    """eps -> 0 recovers the binary mask; growing eps can only remove weight (every M_i is non-increasing in eps)."""
    sc = _zero_mlp(synth.custom_scene(box=(16.0, 16.0, 8.0), hf_n=(17, 17), h_lo=2.0, h_up=6.0, seed=8, step=0.25,
                                      bg=(0.0, 0.0, 0.0)))
    cam = synth.look_at_camera((8.0, -6.0, 14.0), (8.0, 8.0, 4.0), 24, 16)
    hard = oracle.OracleScene(sc).render(cam, 24, 16, mode="brute")
    tiny = oracle.OracleScene(sc, soft_eps=1e-7).render(cam, 24, 16, mode="brute")
    assert np.array_equal(hard["nsamples"], tiny["nsamples"])
    assert np.abs(hard["rgb"] - tiny["rgb"]).max() < 1e-6
    prev = hard["rgb"]
    for eps in (0.25, 0.5, 1.0, 2.0):
        cur = oracle.OracleScene(sc, soft_eps=eps).render(cam, 24, 16, mode="brute")
        assert np.array_equal(cur["nsamples"], hard["nsamples"])
        assert np.all(cur["rgb"] <= prev + 1e-12)
        prev = cur["rgb"]
    assert (hard["rgb"] - prev).max() > 1e-3
