"""Pins for the small pieces of the CPU oracle (run with -m "not gpu").

Each test pins one function of oracle/omerf_oracle.c to something other than itself:
libm / numpy / scipy routines, closed forms, exact special cases.
Citations: PAPER.md line numbers; R# = DESIGN.md readings.
"""
import math
from fractions import Fraction

import numpy as np
import pytest
from scipy.ndimage import map_coordinates

import oracle
import synth


# ----------------------------------------------------------------------------- exp_q (R8)
def test_exp_q_accuracy_and_monotone():
    x = np.linspace(-60.0, 60.0, 20001).astype(np.float32)
    y = oracle.exp_q(x).astype(np.float64)
    ref = np.exp(x.astype(np.float64))
    assert np.max(np.abs(y - ref) / ref) < 4e-7
    assert np.all(np.diff(y) >= 0.0)
    assert oracle.exp_q([0.0])[0] == np.float32(1.0)


def test_q_stop_value():
    # ceil(ln(1000) * 2^20): the integer the early-stop test compares against (R7/R8)
    assert oracle.q_stop(1e-3) == math.ceil(-math.log(float(np.float32(1e-3))) * 2 ** 20)
    assert oracle.q_stop(1e-3) == 7243307


# ----------------------------------------------------------------------------- ray generation (R19)
def test_ray_matches_float64_pinhole():
    cams = synth.make_cameras(2)
    sc = synth.custom_scene()
    O = oracle.OracleScene(sc)
    W, H = synth.config_resolution(2)
    rng = np.random.default_rng(5)
    for cam in cams[:4]:
        c = cam.astype(np.float64)
        o, r, up, f = c[0:3], c[3:6], c[6:9], c[9:12]
        fx, fy, cx, cy = c[12:16]
        for _ in range(20):
            u, v = int(rng.integers(W)), int(rng.integers(H))
            g = f + ((u + 0.5 - cx) / fx) * r - ((v + 0.5 - cy) / fy) * up
            g /= np.linalg.norm(g)
            d = O.ray(cam, u, v)
            assert np.allclose(d, g, atol=3e-7)
            assert abs(float(np.linalg.norm(d.astype(np.float64))) - 1.0) < 2e-7
    # centre pixel (between the four central pixels) looks along fwd; row 0 is the TOP row
    cam = cams[0]
    d_top = O.ray(cam, W // 2, 0)
    d_bot = O.ray(cam, W // 2, H - 1)
    up = cam[6:9]
    assert np.dot(d_top, up) > 0 > np.dot(d_bot, up)
    d_left = O.ray(cam, 0, H // 2)
    assert np.dot(d_left, cam[3:6]) < 0


# ----------------------------------------------------------------------------- interpolation (Eq. 2, R9, R10)
def _scipy_plane(tex, box_a, box_b, pa, pb):
    na, nb = tex.shape[:2]
    qa = pa * na / box_a - 0.5
    qb = pb * nb / box_b - 0.5
    return np.array([map_coordinates(tex[..., c].astype(np.float64), [[qa], [qb]], order=1, mode="nearest")[0]
                     for c in range(8)])


def test_plane_lookup_vs_scipy_and_texel_centres():
    sc = synth.custom_scene(box=(8.0, 6.0, 4.0), xy_n=(16, 12), xz_n=(20, 8), yz_n=(10, 6), seed=3,
                            smooth=False)
    O = oracle.OracleScene(sc)
    rng = np.random.default_rng(0)
    specs = {"xy": (sc.plane_xy, 0, 1), "xz": (sc.plane_xz, 0, 2), "yz": (sc.plane_yz, 1, 2)}
    for which, (tex, a, b) in specs.items():
        na, nb = tex.shape[:2]
        # texel centres: exact texel value (weights 0/256)
        for _ in range(20):
            i, j = int(rng.integers(na)), int(rng.integers(nb))
            pa = (i + 0.5) * sc.box[a] / na
            pb = (j + 0.5) * sc.box[b] / nb
            B = O.plane_lookup(which, pa, pb)
            assert np.array_equal(B, tex[i, j].astype(np.uint32) * 65536)
        # random points incl. the clamp-to-edge border: within the 8-bit weight quantisation
        for _ in range(300):
            pa = float(rng.uniform(0, sc.box[a]))
            pb = float(rng.uniform(0, sc.box[b]))
            B = O.plane_lookup(which, pa, pb).astype(np.float64) / 65536.0
            ref = _scipy_plane(tex, sc.box[a], sc.box[b], pa, pb)
            # |w - w_exact| <= 1/512 per axis, texel range 255
            assert np.max(np.abs(B - ref)) <= 255.0 * (2.0 / 512.0) + 1e-3
        # and tight on a smooth texture: quantisation error scales with adjacent differences
    smooth = synth.custom_scene(box=(8.0, 6.0, 4.0), xy_n=(64, 48), seed=4, smooth=True)
    Os = oracle.OracleScene(smooth)
    tex = smooth.plane_xy
    dmax = max(np.abs(np.diff(tex.astype(np.int32), axis=0)).max(),
               np.abs(np.diff(tex.astype(np.int32), axis=1)).max())
    for _ in range(300):
        pa, pb = float(rng.uniform(0, 8.0)), float(rng.uniform(0, 6.0))
        B = Os.plane_lookup("xy", pa, pb).astype(np.float64) / 65536.0
        ref = _scipy_plane(tex, 8.0, 6.0, pa, pb)
        assert np.max(np.abs(B - ref)) <= dmax * (2.0 / 512.0) * 1.01 + 2e-3


def test_grid_lookup_vs_scipy():
    sc = synth.custom_scene(box=(8.0, 6.0, 4.0), grid_n=(7, 5, 3), seed=9, smooth=False)
    O = oracle.OracleScene(sc)
    g = sc.grid
    rng = np.random.default_rng(1)
    for _ in range(20):
        i, j, k = (int(rng.integers(n)) for n in g.shape[:3])
        p = [(i + 0.5) * 8.0 / 7, (j + 0.5) * 6.0 / 5, (k + 0.5) * 4.0 / 3]
        assert np.array_equal(O.grid_lookup(p), g[i, j, k].astype(np.uint32) * 65536)
    for _ in range(300):
        p = rng.uniform(0, 1, 3) * np.array(sc.box)
        q = [[p[0] * 7 / 8.0 - 0.5], [p[1] * 5 / 6.0 - 0.5], [p[2] * 3 / 4.0 - 0.5]]
        ref = np.array([map_coordinates(g[..., c].astype(np.float64), q, order=1, mode="nearest")[0]
                        for c in range(8)])
        V = O.grid_lookup(p).astype(np.float64) / 65536.0
        assert np.max(np.abs(V - ref)) <= 255.0 * (3.0 / 512.0) + 1e-2


def test_constant_textures_reproduced_exactly():
    fill = [10, 20, 30, 40, 50, 60, 70, 255]
    sc = synth.custom_scene(fill=fill)
    O = oracle.OracleScene(sc)
    rng = np.random.default_rng(2)
    for _ in range(50):
        p = rng.uniform(0, 1, 3) * np.array(sc.box)
        I, t = O.features(p)
        assert np.array_equal(I, 4 * 65536 * np.array(fill))          # V + Pxy + Pxz + Pyz (Eq. 2)
        ref = 4.0 * (np.array(fill) * 28.0 / 255.0 - 14.0)            # R12, four sources summed
        assert np.allclose(t, ref, atol=2e-5)


def test_features_is_sum_of_four_sources_with_right_axes():
    # planes of pairwise different shapes and an anisotropic box: a transposed operand or a
    # wrong axis pairing (xz sampled with (y,z), ...) cannot reproduce scipy's answer
    sc = synth.custom_scene(box=(8.0, 6.0, 4.0), grid_n=(6, 5, 4), xy_n=(32, 24), xz_n=(28, 12),
                            yz_n=(20, 10), seed=11, smooth=True)
    O = oracle.OracleScene(sc)
    rng = np.random.default_rng(3)
    for _ in range(200):
        p = rng.uniform(0.02, 0.98, 3) * np.array(sc.box)
        I, t = O.features(p)
        q = [[p[0] * 6 / 8.0 - 0.5], [p[1] * 5 / 6.0 - 0.5], [p[2] * 4 / 4.0 - 0.5]]
        ref = np.array([map_coordinates(sc.grid[..., c].astype(np.float64), q, order=1, mode="nearest")[0]
                        for c in range(8)])
        ref += _scipy_plane(sc.plane_xy, 8.0, 6.0, p[0], p[1])
        ref += _scipy_plane(sc.plane_xz, 8.0, 4.0, p[0], p[2])
        ref += _scipy_plane(sc.plane_yz, 6.0, 4.0, p[1], p[2])
        assert np.max(np.abs(I / 65536.0 - ref)) < 1.5            # u8 units; smooth textures
        assert np.allclose(t, ref * 28.0 / 255.0 - 56.0, atol=1.5 * 28 / 255)


# ----------------------------------------------------------------------------- occupancy predicate (Eq. 7, R1, R2)
def test_occupied_nearest_grid_point_closed_interval():
    m = 5
    lo = np.arange(m * m, dtype=np.float32).reshape(m, m) * 0.01 + 1.0
    hi = lo + 1.0
    sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(m, m), h_lo=lo, h_up=hi)
    O = oracle.OracleScene(sc)
    h = 8.0 / (m - 1)
    rng = np.random.default_rng(4)
    for _ in range(500):
        x, y = rng.uniform(0, 8.0, 2)
        ix, iy = int(math.floor(x / h + 0.5)), int(math.floor(y / h + 0.5))
        if abs(x / h + 0.5 - round(x / h + 0.5)) < 1e-4 or abs(y / h + 0.5 - round(y / h + 0.5)) < 1e-4:
            continue
        zlo, zhi = float(lo[ix, iy]), float(hi[ix, iy])
        assert O.occupied([x, y, zlo])            # closed at both ends (R2)
        assert O.occupied([x, y, zhi])
        assert O.occupied([x, y, 0.5 * (zlo + zhi)])
        assert not O.occupied([x, y, np.nextafter(np.float32(zlo), np.float32(-1))])
        assert not O.occupied([x, y, np.nextafter(np.float32(zhi), np.float32(9))])
    # empty cell: h_up < h_lo (R17)
    sc2 = synth.custom_scene(h_lo=3.0, h_up=1.0)
    O2 = oracle.OracleScene(sc2)
    assert not O2.occupied([4.0, 4.0, 2.0])


# ----------------------------------------------------------------------------- MLP (Eq. 4, R13)
def test_mlp_vs_numpy_and_encoding():
    sc = synth.custom_scene(seed=7, bias_amp=0.5)
    O = oracle.OracleScene(sc)
    rng = np.random.default_rng(6)
    W0, b0, W1, b1, W2, b2 = (np.asarray(a, dtype=np.float64) for a in (sc.W0, sc.b0, sc.W1, sc.b1, sc.W2, sc.b2))
    for _ in range(50):
        x = rng.uniform(-1, 1, 34)
        h1 = np.maximum(W0 @ x + b0, 0)
        h2 = np.maximum(W1 @ h1 + b1, 0)
        ref = 1.0 / (1.0 + np.exp(-(W2 @ h2 + b2)))
        assert np.allclose(O.mlp(x), ref, atol=1e-12)
    d = np.array([0.3, -0.5, 0.81], dtype=np.float32)
    enc = O.encode_dir(d)
    dd = d.astype(np.float64)
    ref = list(dd)
    for j in range(4):
        for c in range(3):
            ref += [math.sin(2 ** j * dd[c]), math.cos(2 ** j * dd[c])]
    assert np.allclose(enc, ref, atol=1e-15)


# ----------------------------------------------------------------------------- bitfield (R18)
def _brute_bitfield(sc):
    """Exact-rational restatement on a tiny scene (pure Python loops)."""
    Nx, Ny, Nz = sc.occ_n
    Mx, My = sc.h_lo.shape
    X, Y, Z = (Fraction(float(b)) for b in sc.box)
    out = np.zeros((Nx, Ny, Nz), dtype=bool)
    for jx in range(Nx):
        for jy in range(Ny):
            for ix in range(Mx):
                a0, a1 = (Fraction(2 * ix - 1, 2)) * X / (Mx - 1), (Fraction(2 * ix + 1, 2)) * X / (Mx - 1)
                if min(a1, Fraction(jx + 1) * X / Nx) - max(a0, Fraction(jx) * X / Nx) <= 0:
                    continue
                for iy in range(My):
                    c0, c1 = (Fraction(2 * iy - 1, 2)) * Y / (My - 1), (Fraction(2 * iy + 1, 2)) * Y / (My - 1)
                    if min(c1, Fraction(jy + 1) * Y / Ny) - max(c0, Fraction(jy) * Y / Ny) <= 0:
                        continue
                    lo, hi = Fraction(float(sc.h_lo[ix, iy])), Fraction(float(sc.h_up[ix, iy]))
                    if lo > hi:
                        continue
                    for jz in range(Nz):
                        if Fraction(jz) * Z / Nz <= hi and Fraction(jz + 1) * Z / Nz >= lo:
                            out[jx, jy, jz] = True
    return out


@pytest.mark.parametrize("hf_n,occ_n", [((5, 5), (8, 8, 8)), ((5, 4), (6, 7, 5)), ((3, 3), (9, 5, 16))])
def test_bitfield_vs_exact_rational_brute_force(hf_n, occ_n):
    rng = np.random.default_rng(8)
    lo = rng.uniform(0.2, 1.5, hf_n).astype(np.float32)
    hi = (lo + rng.uniform(-0.3, 2.0, hf_n)).astype(np.float32)       # some cells empty
    sc = synth.custom_scene(box=(8.0, 6.0, 4.0), hf_n=hf_n, h_lo=lo, h_up=hi, occ_n=occ_n)
    O = oracle.OracleScene(sc, sampler=1)
    n = int(np.prod(occ_n))
    bits = np.unpackbits(O.bits.view(np.uint8), bitorder="little")[:n].reshape(occ_n).astype(bool)
    assert np.array_equal(bits, _brute_bitfield(sc))


def test_occupied_grid_lookup_reads_the_voxel_that_contains_the_point():
    """The config-4 predicate (sampler 1) pinned directly: for random points away from voxel faces
    the voxel (jx,jy,jz) is recomputed in float64 and the answer is read from the exact-rational brute-force bitfield.
    Non-cubic occ_n with Ny != Nz != Nx: an index swap, a transposed stride or an enlarged set fails."""
    rng = np.random.default_rng(12)
    hf_n, occ_n, box = (5, 4), (6, 7, 5), (8.0, 6.0, 4.0)
    lo = rng.uniform(0.2, 1.5, hf_n).astype(np.float32)
    hi = (lo + rng.uniform(-0.3, 2.0, hf_n)).astype(np.float32)
    sc = synth.custom_scene(box=box, hf_n=hf_n, h_lo=lo, h_up=hi, occ_n=occ_n)
    O = oracle.OracleScene(sc, sampler=1)
    want = _brute_bitfield(sc)
    assert 0 < want.sum() < want.size                              # both answers occur
    seen = {False: 0, True: 0}
    for p in rng.uniform(0.0, 1.0, (6000, 3)) * np.array(box):
        q = p * np.array(occ_n) / np.array(box)                   # voxel coordinates, float64
        if np.any(np.abs(q - np.rint(q)) < 1e-3):                 # too close to a voxel face for fp32 to agree
            continue
        j = np.floor(q).astype(int)
        got = O.occupied(p.astype(np.float32))
        assert got == bool(want[j[0], j[1], j[2]]), (p, j)
        seen[got] += 1
    assert seen[False] > 500 and seen[True] > 500
    # clamp at the far faces: a point on the box face belongs to the last voxel
    for p, j in (((8.0, 3.0, 2.0), (5, 3, 2)), ((4.0, 6.0, 2.0), (3, 6, 2)), ((4.0, 3.0, 4.0), (3, 3, 4))):
        assert O.occupied(np.array(p, dtype=np.float32)) == bool(want[j])


def test_distinct_sector_count_matches_numpy_recount():
    """SURVEY 8(d) compulsory-byte figure: distinct 32-byte sectors per source touched by a render, recounted in numpy
    from the kept sample positions (thin density: no ray terminates, so every kept lattice point is a sample)."""
    fill = [100, 128, 128, 128, 128, 128, 128, 128]
    sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=1.0, h_up=3.0, grid_n=(12, 10, 8), xy_n=(40, 36),
                            xz_n=(40, 16), yz_n=(36, 16), fill=fill, seed=2, step=0.2)
    O = oracle.OracleScene(sc)
    cam = synth.look_at_camera((4.0, -3.0, 7.0), (4.0, 4.0, 2.0), 20, 14)
    with oracle.SectorMaps(O) as M:
        r = O.render(cam, 20, 14, mode="brute")
    want = {"grid": set(), "xy": set(), "xz": set(), "yz": set()}
    total = 0
    for v in range(14):
        for u in range(20):
            n, ks, pos = O.pixel_samples(cam, u, v)
            assert n == r["nsamples"][0, v, u]
            total += n
            for p in pos.astype(np.float64):
                def taps(x, N, X):
                    i = int(np.floor(x * N / X - 0.5))
                    return {min(max(i, 0), N - 1), min(max(i + 1, 0), N - 1)}
                gx, gy, gz = taps(p[0], 12, 8.0), taps(p[1], 10, 8.0), taps(p[2], 8, 4.0)
                want["grid"] |= {((x * 10 + y) * 8 + z) // 4 for x in gx for y in gy for z in gz}
                want["xy"] |= {(a * 36 + b) // 4 for a in taps(p[0], 40, 8.0) for b in taps(p[1], 36, 8.0)}
                want["xz"] |= {(a * 16 + b) // 4 for a in taps(p[0], 40, 8.0) for b in taps(p[2], 16, 4.0)}
                want["yz"] |= {(a * 16 + b) // 4 for a in taps(p[1], 36, 8.0) for b in taps(p[2], 16, 4.0)}
    got = M.sectors()
    assert total > 1000
    for k in want:      # float64 vs the oracle's fp32 taps may disagree on a point within an ulp of a texel boundary
        assert abs(got[k] - len(want[k])) <= 2, (k, got[k], len(want[k]))
    assert M.compulsory_bytes() == 32 * sum(got.values())
    # nothing is recorded outside the with-block
    before = M.sectors()
    O.render(cam, 20, 14, mode="brute")
    assert M.sectors() == before


def test_heatmap_ramp_pins():
    """R26: blue at 0 samples, green at the middle, red at and above n_max; red channel monotone, blue its mirror."""
    hm = oracle.heatmap(np.arange(0, 40), 32)
    assert hm.dtype == np.uint8 and hm.shape == (40, 3)
    assert tuple(hm[0]) == (0, 0, 255) and tuple(hm[32]) == (255, 0, 0) and tuple(hm[39]) == (255, 0, 0)
    assert tuple(hm[16]) == (127, 254, 128)                       # v = 16 * 255 // 32 = 127
    assert np.all(np.diff(hm[:, 0].astype(int)) >= 0) and np.array_equal(hm[:, 2], 255 - hm[:, 0])
    assert hm[:, 1].max() == 254 and hm[:, 1].argmax() == 16
    assert tuple(oracle.heatmap(np.array([1]), 1)[0]) == (255, 0, 0)
