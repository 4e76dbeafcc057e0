"""Render-level pins of the CPU oracle (run with -m "not gpu").

Closed forms, invariants, an independent float64 'textbook' renderer built from
scipy/numpy library routines, brute force vs the clipped loop, symmetry.
Citations: PAPER.md line numbers; R# = DESIGN.md readings.
"""
import math

import numpy as np
import pytest
from scipy.ndimage import map_coordinates

import oracle
import synth


def _np_mlp(sc, x):
    W0, b0, W1, b1, W2, b2 = (np.asarray(a, dtype=np.float64) for a in (sc.W0, sc.b0, sc.W1, sc.b1, sc.W2, sc.b2))
    h1 = np.maximum(W0 @ x + b0, 0)
    h2 = np.maximum(W1 @ h1 + b1, 0)
    return 1.0 / (1.0 + np.exp(-(W2 @ h2 + b2)))


def _np_ray(cam, u, v):
    c = cam.astype(np.float64)
    g = c[9:12] + ((u + 0.5 - c[14]) / c[12]) * c[3:6] - ((v + 0.5 - c[15]) / c[13]) * c[6:9]
    return c[0:3], g / np.linalg.norm(g)


def _np_enc(d):
    e = list(d)
    for j in range(4):
        for c in range(3):
            e += [math.sin(2 ** j * d[c]), math.cos(2 ** j * d[c])]
    return np.array(e)


# ----------------------------------------------------------------------------- closed form: constant slab
@pytest.mark.parametrize("byte,step", [(150, 0.25), (140, 0.25), (150, 0.125), (150, 0.0625), (128, 0.5)])
def test_constant_slab_closed_form(byte, step):
    """Flat height fields z_a, z_b and constant texels: tau = exp(4(u 28/255 - 14)),
    n = #{k : z_a <= o_z + t_k d_z <= z_b}, T = exp(-tau n step) -> exp(-tau L) as step -> 0
    (BASELINE.json north_star; Eq. 1), colour = (1-T) sigmoid(.) + S + T bg (Eq. 4)."""
    za, zb = 1.0, 3.0
    fill = [byte, 100, 128, 180, 90, 128, 200, 60]
    sc = synth.custom_scene(box=(32.0, 32.0, 4.0), hf_n=(9, 9), h_lo=za, h_up=zb, fill=fill, step=step,
                            bias_amp=0.3, seed=1)
    O = oracle.OracleScene(sc)
    W = H = 24
    cam = synth.look_at_camera((16.0, 4.0, 14.0), (16.0, 16.0, 2.0), W, H, vfov_deg=40.0)
    r = O.render(cam, W, H, mode="brute", aux=True)
    tau = math.exp(4.0 * (byte * 28.0 / 255.0 - 14.0))
    pre = 4.0 * (np.array(fill[1:]) * 28.0 / 255.0 - 14.0)
    sig = 1.0 / (1.0 + np.exp(-pre))
    qs = oracle.q_stop(1e-3)
    checked = 0
    for v in range(H):
        for u in range(W):
            o, d = _np_ray(cam, u, v)
            assert d[2] < 0
            K = O.lattice_K(cam)
            t = (np.arange(K) + 0.5) * step
            p = o[None, :] + t[:, None] * d[None, :]
            inb = np.all((p >= 0) & (p < np.array(sc.box)), axis=1)
            z = p[:, 2]
            # skip rays with a sample within 1e-4 of a decision boundary (fp32 vs fp64 positions)
            margin = np.min(np.abs(np.concatenate([z - za, z - zb])))
            edge = min(np.min(np.abs(p[:, 0])), np.min(np.abs(p[:, 0] - 32.0)), np.min(np.abs(p[:, 1])),
                       np.min(np.abs(p[:, 1] - 32.0)))
            if margin < 1e-4 or edge < 1e-4:
                continue
            n_all = int(np.sum(inb & (z >= za) & (z <= zb)))
            # early stop: samples are taken while accumulated optical depth < ln(1000) (R7)
            per = tau * step
            n_stop = n_all if per * n_all * 2 ** 20 < qs else int(math.ceil(qs / round(min(per * 2 ** 20, qs))))
            n = min(n_all, n_stop)
            assert r["nsamples"][0, v, u] == n
            # continuum limit: n step -> L = (z_b - z_a)/|d_z| when the ray crosses the whole slab in the box
            L = (zb - za) / abs(d[2])
            if n == n_all and inb[(z >= za) & (z <= zb)].all() and n_all > 0:
                assert abs(n_all * step - L) <= step * 1.0001
            T = math.exp(-tau * n * step) if n < n_stop or per * 2 ** 20 < qs else r["T_end"][0, v, u]
            if n > 0:
                assert abs(r["T_end"][0, v, u] - T) <= max(n * 2.0 ** -20, 1e-9) * max(T, 1e-3) + 1e-12
                Tn = r["T_end"][0, v, u]
                D = (1.0 - math.exp(-tau * n * step)) * sig[:3]
                Fs = (1.0 - math.exp(-tau * n * step)) * sig[3:]
                S = _np_mlp(sc, np.concatenate([D, Fs, _np_enc(d)]))
                rgb = np.clip(D + S + Tn * np.array(sc.bg), 0, 1)
                assert np.allclose(r["rgb"][0, v, u], rgb, atol=2e-5)
            else:
                assert np.array_equal(r["rgb"][0, v, u], np.array(sc.bg, dtype=np.float64))
            checked += 1
    assert checked > W * H // 2


def test_step_refinement_converges_first_order():
    """Piecewise-constant density: -log T_end -> tau L at first order in step."""
    za, zb, byte = 1.0, 3.0, 127
    tau = math.exp(4.0 * (byte * 28.0 / 255.0 - 14.0))
    cam = synth.look_at_camera((16.0, 4.0, 14.0), (16.0, 16.0, 2.0), 8, 8, vfov_deg=20.0)
    errs = []
    for step in (0.5, 0.25, 0.125, 0.0625):
        sc = synth.custom_scene(box=(32.0, 32.0, 4.0), h_lo=za, h_up=zb, fill=byte, step=step)
        r = oracle.OracleScene(sc).render(cam, 8, 8, mode="brute", aux=True)
        e = 0.0
        for v in range(8):
            for u in range(8):
                _, d = _np_ray(cam, u, v)
                L = (zb - za) / abs(d[2])
                e = max(e, abs(-math.log(r["T_end"][0, v, u]) - tau * L))
                assert abs(-math.log(r["T_end"][0, v, u]) - tau * L) <= tau * step * 1.001 + 1e-5
        errs.append(e)
    assert errs[-1] < errs[0] / 3.0


# ----------------------------------------------------------------------------- empty scene == background
def test_empty_slab_and_looking_away_return_background_exactly():
    cam = synth.look_at_camera((4.0, -6.0, 9.0), (4.0, 4.0, 2.0), 16, 16)
    sc = synth.custom_scene(h_lo=3.0, h_up=1.0, bg=(0.25, 0.5, 0.75))       # h_up < h_lo everywhere (R17)
    for mode in ("brute", "clipped"):
        r = oracle.OracleScene(sc).render(cam, 16, 16, mode=mode)
        assert r["nsamples"].sum() == 0
        assert np.array_equal(r["rgb"], np.broadcast_to(np.array(sc.bg, dtype=np.float32).astype(np.float64),
                                                        r["rgb"].shape))
    sc2 = synth.custom_scene(bg=(0.25, 0.5, 0.75))
    away = synth.look_at_camera((4.0, -6.0, 9.0), (4.0, -20.0, 12.0), 16, 16)
    r = oracle.OracleScene(sc2).render(away, 16, 16, mode="brute")
    assert r["nsamples"].sum() == 0
    assert np.all(r["rgb"] == np.array(sc2.bg, dtype=np.float32).astype(np.float64))


# ----------------------------------------------------------------------------- weights
def test_weights_sum_le_one_and_telescope(cfg0):
    sc, cams, (W, H) = cfg0
    r = oracle.OracleScene(sc).render(cams, W, H, mode="clipped", aux=True)
    # sum of weights <= 1 up to the 2^-20 quantisation of the optical depth that T is formed from (R8):
    # each sample can push T up by at most 2^-21 relative
    assert np.all(r["sum_w"] <= 1.0 + r["nsamples"] * 2.0 ** -21 + 1e-12)
    qs = oracle.q_stop(sc.t_stop)
    open_ = r["Q"] < qs                     # not terminated: no capped sample, exact telescoping
    assert np.max(np.abs(r["sum_w"][open_] - (1.0 - r["T_end"][open_]))) < 1e-5
    # terminated rays: q_k is capped at Q_STOP, so T_end >= true T by at most t_stop
    assert np.max(np.abs(r["sum_w"] - (1.0 - r["T_end"]))) <= 1e-3 + 1e-5
    assert np.all((r["rgb"] >= 0) & (r["rgb"] <= 1))


# ----------------------------------------------------------------------------- brute == clipped
def test_brute_equals_clipped_config0(cfg0):
    sc, cams, (W, H) = cfg0
    O = oracle.OracleScene(sc)
    a = O.render(cams, W, H, mode="brute")
    b = O.render(cams, W, H, mode="clipped")
    assert np.array_equal(a["nsamples"], b["nsamples"])
    assert np.array_equal(a["rgb"], b["rgb"])
    assert a["nsamples"].sum() > W * H          # the test is not vacuous


@pytest.mark.parametrize("origin,target", [
    ((4.0, 4.0, 2.0), (7.0, 5.0, 2.1)),         # inside the box, near-horizontal
    ((4.0, -3.0, 1.5), (4.0, 4.0, 1.5)),        # horizontal, entering through a side
    ((4.0, 4.0, 30.0), (4.0, 4.0001, 0.0)),     # straight down
    ((-5.0, -5.0, 0.5), (8.0, 8.0, 3.5)),       # upward from below the slab
    ((4.0, 4.0, 2.0), (4.0, 4.0, 9.0)),         # inside looking up
])
def test_brute_equals_clipped_edge_cameras(origin, target):
    rng = np.random.default_rng(12)
    lo = rng.uniform(0.5, 1.5, (9, 9)).astype(np.float32)
    hi = (lo + rng.uniform(0.2, 2.0, (9, 9))).astype(np.float32)
    sc = synth.custom_scene(h_lo=lo, h_up=hi, seed=5)
    O = oracle.OracleScene(sc)
    cam = synth.look_at_camera(origin, target, 24, 24, vfov_deg=70.0)
    a = O.render(cam, 24, 24, mode="brute")
    b = O.render(cam, 24, 24, mode="clipped")
    assert np.array_equal(a["nsamples"], b["nsamples"])
    assert np.array_equal(a["rgb"], b["rgb"])


# ----------------------------------------------------------------------------- textbook renderer from library routines
def _textbook_pixel(sc, cam, u, v, K):
    """Eq. 1-4 and 7-8 written with numpy/scipy in float64, T_i as the literal product
    prod_{j<i}(1 - alpha_j) (R6), exact (unquantised) interpolation weights."""
    o, d = _np_ray(cam, u, v)
    box = np.array(sc.box)
    t = (np.arange(K) + 0.5) * sc.step
    p = o[None, :] + t[:, None] * d[None, :]
    inb = np.all((p >= 0) & (p < box), axis=1)
    Mx, My = sc.h_lo.shape
    ix = np.clip(np.floor(p[:, 0] * (Mx - 1) / box[0] + 0.5).astype(int), 0, Mx - 1)
    iy = np.clip(np.floor(p[:, 1] * (My - 1) / box[1] + 0.5).astype(int), 0, My - 1)
    keep = inb & (sc.h_lo[ix, iy] <= p[:, 2]) & (p[:, 2] <= sc.h_up[ix, iy])
    p = p[keep]
    if len(p) == 0:
        return 0, np.array(sc.bg, dtype=np.float64), p
    feats = np.zeros((len(p), 8))
    for tex, axes in ((sc.grid, (0, 1, 2)), (sc.plane_xy, (0, 1)), (sc.plane_xz, (0, 2)), (sc.plane_yz, (1, 2))):
        q = [p[:, a] * tex.shape[i] / box[a] - 0.5 for i, a in enumerate(axes)]
        for c in range(8):
            feats[:, c] += map_coordinates(tex[..., c].astype(np.float64), q, order=1, mode="nearest")
    pre = feats * sc.deq_scale + 4 * sc.deq_bias
    tau = np.exp(pre[:, 0])
    alpha = 1.0 - np.exp(-tau * sc.step)
    T = np.concatenate([[1.0], np.cumprod(1.0 - alpha)[:-1]])
    od_before = np.concatenate([[0.0], np.cumsum(tau * sc.step)[:-1]])
    live = od_before < -math.log(sc.t_stop)                       # early stop tested before the sample (R7)
    n = int(live.sum())
    w = (T * alpha)[live]
    sig = 1.0 / (1.0 + np.exp(-pre[live, 1:]))
    D = (w[:, None] * sig[:, :3]).sum(0)
    Fs = (w[:, None] * sig[:, 3:]).sum(0)
    T_end = max(float(np.prod(1.0 - alpha[live])), 0.0)
    S = _np_mlp(sc, np.concatenate([D, Fs, _np_enc(d)]))
    return n, np.clip(D + S + T_end * np.array(sc.bg), 0, 1), p


def test_oracle_vs_textbook_renderer(cfg0):
    sc, cams, (W, H) = cfg0
    O = oracle.OracleScene(sc)
    r = O.render(cams, W, H, mode="brute")
    K = O.lattice_K(cams[0])
    rng = np.random.default_rng(21)
    same, tot = 0, 0
    for _ in range(250):
        u, v = int(rng.integers(W)), int(rng.integers(H))
        n, rgb, _ = _textbook_pixel(sc, cams[0], u, v, K)
        tot += 1
        if n == r["nsamples"][0, v, u]:
            same += 1
            # weight quantisation (1/512 per axis) and the Q_STOP cap on T_end (<= 1e-3) are the only differences
            assert np.max(np.abs(rgb - r["rgb"][0, v, u])) < 6e-3
    assert same >= 0.97 * tot
    assert r["nsamples"].max() > 10


def test_positions_of_kept_samples(cfg0):
    """The kept samples are lattice points o + (k+1/2) step d inside box and slab (R4, Eq. 7)."""
    sc, cams, (W, H) = cfg0
    O = oracle.OracleScene(sc)
    for (u, v) in [(64, 64), (10, 100), (120, 30)]:
        n, ks, pos = O.pixel_samples(cams[0], u, v)
        o, d = _np_ray(cams[0], u, v)
        ref = o[None, :] + ((ks + 0.5) * sc.step)[:, None] * d[None, :]
        assert np.allclose(pos, ref, atol=2e-5)
        _, _, p = _textbook_pixel(sc, cams[0], u, v, O.lattice_K(cams[0]))
        assert abs(len(p) - n) <= 1


# ----------------------------------------------------------------------------- x <-> y transpose symmetry
def test_transpose_symmetry(cfg0):
    sc, cams, (W, H) = cfg0
    import copy
    st = copy.copy(sc)
    st.box = (sc.box[1], sc.box[0], sc.box[2])
    st.h_lo = np.ascontiguousarray(sc.h_lo.T)
    st.h_up = np.ascontiguousarray(sc.h_up.T)
    st.grid = np.ascontiguousarray(sc.grid.transpose(1, 0, 2, 3))
    st.plane_xy = np.ascontiguousarray(sc.plane_xy.transpose(1, 0, 2))
    st.plane_xz, st.plane_yz = sc.plane_yz, sc.plane_xz
    # the deferred MLP sees enc(d): swap the x and y columns of its first layer as well
    perm = list(range(34))
    perm[7], perm[8] = 8, 7
    for j in range(4):
        bx, by = 10 + (3 * j + 0) * 2, 10 + (3 * j + 1) * 2
        perm[bx], perm[bx + 1], perm[by], perm[by + 1] = by, by + 1, bx, bx + 1
    st.W0 = np.ascontiguousarray(sc.W0[:, perm])
    camt = cams.copy()
    for b in (0, 3, 6, 9):
        camt[:, [b, b + 1]] = cams[:, [b + 1, b]]
    # a camera off the symmetry axes, so the test is not trivially symmetric
    cam = synth.look_at_camera((10.0, -20.0, 35.0), (30.0, 34.0, 8.0), W, H)
    camt = cam.copy()
    for b in (0, 3, 6, 9):
        camt[[b, b + 1]] = cam[[b + 1, b]]
    a = oracle.OracleScene(sc).render(cam, W, H, mode="clipped")
    b_ = oracle.OracleScene(st).render(camt, W, H, mode="clipped")
    # identical up to the rounding order of |g|^2 (x and y swap inside one fma chain)
    assert np.mean(a["nsamples"] == b_["nsamples"]) > 0.995
    same = a["nsamples"] == b_["nsamples"]
    # (a one-ulp change of d can swap one boundary sample for another at equal count: allow a few pixels)
    err = np.max(np.abs(a["rgb"][same] - b_["rgb"][same]), axis=-1)
    assert np.mean(err < 1e-4) > 0.995
    assert a["nsamples"].sum() > W * H


# ----------------------------------------------------------------------------- config-4 comparator (R18)
def test_grid_sampler_superset_and_occupancy_ratio():
    rng = np.random.default_rng(31)
    m = 17
    lo = (1.0 + 0.5 * rng.random((m, m))).astype(np.float32)
    hi = (lo + 0.3 + 1.5 * rng.random((m, m))).astype(np.float32)
    # low density everywhere (byte 100 -> tau ~ 1e-5): no ray terminates early
    sc = synth.custom_scene(box=(16.0, 16.0, 4.0), hf_n=(m, m), h_lo=lo, h_up=hi, fill=100, step=0.125,
                            occ_n=(32, 32, 32))
    cam = synth.look_at_camera((8.0, -10.0, 14.0), (8.0, 8.0, 2.0), 48, 48)
    Op = oracle.OracleScene(sc, sampler=0)
    Og = oracle.OracleScene(sc, sampler=1)
    a = Op.render(cam, 48, 48, mode="brute")
    for mode in ("brute", "clipped"):
        b = Og.render(cam, 48, 48, mode=mode)
        assert np.all(b["nsamples"] >= a["nsamples"])
    assert b["nsamples"].sum() > a["nsamples"].sum() > 0
    # occupancy ratio vs the analytic slab volume fraction: each column adds at most two partial voxels
    n = 32 ** 3
    ratio = np.unpackbits(Og.bits.view(np.uint8), bitorder="little")[:n].sum() / n
    w = np.ones(m)
    w[0] = w[-1] = 0.5                                         # half cells at the border (R1)
    area = np.outer(w, w)
    frac = float(((hi - lo) * area).sum() / area.sum() / 4.0)
    dz = 4.0 / 32
    assert frac <= ratio <= frac + 2 * dz / 4.0 + 1e-9


def test_render_pixels_equals_render_on_random_pixels_of_a_batch():
    """orc_render_pixels (the oracle's entry for scattered (view, u, v) triples, used by the full-size GPU tests where a
    whole batch would take minutes) is the same per-pixel routine as orc_render: on random pixels of a 3-view batch -
    cameras of different pose, a non-square image, repeated and border pixels - counts, colours and the auxiliary
    outputs are bit-identical to the whole-image render, in both the brute-force and the clipped loop.  A wrong view
    stride, swapped (u, v) or a camera taken from the wrong row fails it (W != H, three different poses)."""
    sc = synth.make_scene(0)
    W, H = 45, 31
    cams = np.stack([synth.look_at_camera((10.0, -14.0, 30.0), (32.0, 32.0, 8.0), W, H),
                     synth.look_at_camera((70.0, 70.0, 25.0), (32.0, 32.0, 6.0), W, H),
                     synth.look_at_camera((32.0, 32.0, 60.0), (32.0, 32.5, 0.0), W, H)])
    O = oracle.OracleScene(sc)
    rng = np.random.default_rng(11)
    m = 400
    vuv = np.stack([rng.integers(0, 3, m), rng.integers(0, W, m), rng.integers(0, H, m)], axis=1).astype(np.int32)
    vuv[:6] = [[0, 0, 0], [2, W - 1, H - 1], [1, 0, H - 1], [1, W - 1, 0], [2, 5, 7], [2, 5, 7]]
    for mode in ("clipped", "brute"):
        full = O.render(cams, W, H, mode=mode, aux=True)
        got = O.render_pixels(cams, W, H, vuv, mode=mode, aux=True)
        idx = (vuv[:, 0], vuv[:, 2], vuv[:, 1])             # images are indexed [view][row v][column u]
        assert full["nsamples"].sum() > 10000 and len({int(x) for x in got["nsamples"]}) > 5
        assert np.array_equal(got["nsamples"], full["nsamples"][idx])
        assert np.array_equal(got["rgb"], full["rgb"][idx])
        for key in ("T_end", "sum_w", "Q"):
            assert np.array_equal(got[key], full[key][idx]), key
    # the three views really differ at the sampled pixels (else a wrong camera row would go unnoticed)
    assert not np.array_equal(full["nsamples"][0], full["nsamples"][1])
    with pytest.raises(ValueError):
        O.render_pixels(cams, W, H, [[3, 0, 0]])            # view out of range
    with pytest.raises(ValueError):
        O.render_pixels(cams, W, H, [[0, 0, H]])            # row out of range (u = 0 .. W-1, v = 0 .. H-1)
