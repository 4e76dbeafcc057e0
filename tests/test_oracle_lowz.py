"""Pins of the oracle's low-z triplane bake (SURVEY 8(f).1 second half; R27), -m "not gpu".

The band rule is pinned against what it is for - the z-texel rows a bilinear lookup of a slab point can touch - by
brute force over occupied points, against a closed form for flat slabs, and for tightness at the extreme columns."""
import math

import numpy as np
import pytest

import oracle
import synth


def _scene(seed, hf=11, xz_n=(24, 40), yz_n=(20, 32), box=(10.0, 9.0, 6.0), lo_rng=(1.1, 2.0), thick=(0.05, 2.0),
           empty_frac=0.15):
    rng = np.random.default_rng(seed)
    lo = (lo_rng[0] + (lo_rng[1] - lo_rng[0]) * rng.random((hf, hf))).astype(np.float32)
    hi = (lo + thick[0] + (thick[1] - thick[0]) * rng.random((hf, hf))).astype(np.float32)
    kill = rng.random((hf, hf)) < empty_frac
    # empty columns (R17) carry values far outside the band: they must not widen it
    lo[kill], hi[kill] = 5.9, 0.1
    return synth.custom_scene(box=box, hf_n=(hf, hf), h_lo=lo, h_up=hi, xz_n=xz_n, yz_n=yz_n, seed=seed, smooth=False)


@pytest.mark.parametrize("za,zb", [(1.0, 3.0), (0.0, 6.0), (2.26, 2.27), (5.99, 6.0), (0.0, 0.01)])
def test_flat_slab_closed_form(za, zb):
    """Flat slab [za, zb]: band = [floor(za Nz/Z - 1/2 - 1/64), floor(zb Nz/Z - 1/2 + 1/64) + 1] clamped to the plane."""
    Z, Nz = 6.0, 48
    sc = synth.custom_scene(box=(8.0, 6.0, Z), hf_n=(9, 7), h_lo=za, h_up=zb, xz_n=(16, Nz), yz_n=(12, Nz), seed=1)
    O = oracle.OracleScene(sc)
    for which in ("xz", "yz"):
        Bd = oracle.LowZBand(O, which)
        k0 = max(math.floor(za * Nz / Z - 0.5 - 1 / 64), 0)
        k1 = min(math.floor(zb * Nz / Z - 0.5 + 1 / 64) + 1, Nz - 1)
        assert (Bd.b_lo, Bd.b_hi, Bd.rows) == (k0, k1, k1 - k0 + 1)
        plane = getattr(sc, "plane_" + which)
        assert np.array_equal(Bd.band, plane[:, k0:k1 + 1])


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_every_z_tap_of_an_occupied_point_is_kept_and_the_lookup_is_unchanged(seed):
    """Soundness by brute force: points that pass the per-sample predicate (Eq. 7, fp32) only touch rows inside the
    band, and the lookup through the band returns the full plane's integers."""
    sc = _scene(seed)
    O = oracle.OracleScene(sc)
    bands = {w: oracle.LowZBand(O, w) for w in ("xz", "yz")}
    assert bands["xz"].rows < sc.plane_xz.shape[1] and bands["yz"].rows < sc.plane_yz.shape[1]   # something is saved
    rng = np.random.default_rng(50 + seed)
    pts = (rng.random((20000, 3)) * np.array(sc.box)).astype(np.float32)
    pts = [p for p in pts if np.all(p < np.array(sc.box, dtype=np.float32)) and O.occupied(p)]
    # extreme samples: exactly on z_min / z_max of every non-empty column (closed interval, R2)
    Mx, My = sc.h_lo.shape
    for ix in range(Mx):
        for iy in range(My):
            if sc.h_lo[ix, iy] <= sc.h_up[ix, iy]:
                x, y = ix * sc.box[0] / (Mx - 1), iy * sc.box[1] / (My - 1)
                for z in (sc.h_lo[ix, iy], sc.h_up[ix, iy]):
                    p = np.array([min(x, sc.box[0] * 0.999), min(y, sc.box[1] * 0.999), z], dtype=np.float32)
                    if O.occupied(p):
                        pts.append(p)
    assert len(pts) > 2500
    for p in pts:
        rc, got = bands["xz"].lookup(p[0], p[2])
        assert rc == 0, p
        assert np.array_equal(got, O.plane_lookup("xz", p[0], p[2]))
        rc, got = bands["yz"].lookup(p[1], p[2])
        assert rc == 0, p
        assert np.array_equal(got, O.plane_lookup("yz", p[1], p[2]))


def test_band_is_tight_at_the_extreme_columns():
    """The first and last kept rows are touched (up to the 1/64-texel padding) by the slab's lowest / highest point:
    the true taps of z_lo and z_hi lie within one row of the band's ends, and empty columns do not widen the band."""
    sc = _scene(9)
    O = oracle.OracleScene(sc)
    ok = sc.h_lo <= sc.h_up
    z_lo, z_hi = float(sc.h_lo[ok].min()), float(sc.h_up[ok].max())
    for which, Nz in (("xz", sc.plane_xz.shape[1]), ("yz", sc.plane_yz.shape[1])):
        Bd = oracle.LowZBand(O, which, crop=False)
        t_lo = math.floor(z_lo * Nz / sc.box[2] - 0.5)             # lower tap of the lowest slab point
        t_hi = math.floor(z_hi * Nz / sc.box[2] - 0.5) + 1         # upper tap of the highest slab point
        assert t_lo - 1 <= Bd.b_lo <= t_lo and t_hi <= Bd.b_hi <= t_hi + 1
        assert Bd.rows == Bd.b_hi - Bd.b_lo + 1


def test_band_is_monotone_and_clipped_to_the_box():
    prev = 0
    for zb in (1.2, 2.0, 3.0, 4.0, 9.0):                           # 9.0 > Z: clipped to the box
        sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=1.0, h_up=zb, xz_n=(16, 32), yz_n=(16, 32), seed=1)
        Bd = oracle.LowZBand(oracle.OracleScene(sc), "xz", crop=False)
        assert Bd.rows >= prev and 0 <= Bd.b_lo <= Bd.b_hi <= 31
        prev = Bd.rows
    assert Bd.b_hi == 31
    sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=-3.0, h_up=4.0, xz_n=(16, 32), yz_n=(16, 32), seed=1)
    Bd = oracle.LowZBand(oracle.OracleScene(sc), "yz", crop=False)
    assert (Bd.b_lo, Bd.b_hi) == (0, 31)                           # the whole box: nothing to save


def test_scene_without_occupied_columns_keeps_one_row():
    sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=3.0, h_up=1.0, xz_n=(16, 32), yz_n=(16, 32), seed=1)
    Bd = oracle.LowZBand(oracle.OracleScene(sc), "xz")
    assert (Bd.b_lo, Bd.b_hi, Bd.rows) == (0, 0, 1) and Bd.band.shape == (16, 1, 8)
