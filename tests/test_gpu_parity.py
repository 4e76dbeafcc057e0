"""Parity of the CUDA path against the CPU oracle, through the C-ABI (run on the B200 box: -m gpu).

Bar (BASELINE.json north_star): per-pixel sample counts bit-exact; max |dRGB| <= 2e-3 per channel.
"""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu

RGB_TOL = 2e-3   # north_star: "max |dRGB| <= 2e-3 per channel on [0,1] for the fp32 colour path"


@pytest.fixture(scope="module")
def omerf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2404_09531_b200 as m
    m.load_library()
    return m


@pytest.fixture(scope="module")
def oracle():
    import oracle as o
    return o


def _gpu_render(omerf, scene, cams, W, H, sampler=0, host=False):
    import torch
    with omerf.scene_create(scene, sampler=sampler) as h:
        if host:
            rgb, ns = omerf.render_host(h, cams, W, H)
            launches = omerf.last_launch_count(h)
            return rgb.astype(np.float64), ns, launches
        rgb, ns = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        launches = omerf.last_launch_count(h)
        return rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), launches


def _assert_parity(got_rgb, got_n, ref, what=""):
    bad = got_n != ref["nsamples"]
    assert not bad.any(), f"{what}: {int(bad.sum())} pixels with wrong sample counts, first at {np.argwhere(bad)[:5].tolist()}"
    err = np.abs(got_rgb - ref["rgb"]).max()
    assert err <= RGB_TOL, f"{what}: max |dRGB| = {err}"


# ----------------------------------------------------------------------------- config 0 (whole image, brute oracle)
def test_config0_full_image(omerf, oracle):
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    rgb, ns, launches = _gpu_render(omerf, sc, cams, W, H)
    ref = oracle.OracleScene(sc).render(cams, W, H, mode="brute")
    assert launches >= 1
    assert ref["nsamples"].sum() > 50000
    _assert_parity(rgb, ns, ref, "config 0")


def test_config0_host_buffers_and_ragged_sizes(omerf, oracle):
    sc = synth.make_scene(0)
    O = oracle.OracleScene(sc)
    for (W, H) in [(37, 29), (1, 1), (16, 8), (17, 9), (130, 3)]:
        cam = synth.look_at_camera((10.0, -14.0, 30.0), (32.0, 32.0, 8.0), W, H)
        rgb, ns, _ = _gpu_render(omerf, sc, cam, W, H, host=True)
        _assert_parity(rgb, ns, O.render(cam, W, H, mode="clipped"), f"{W}x{H}")


# ----------------------------------------------------------------------------- edge cameras, degenerate scenes
EDGE_CAMS = [
    ((4.0, 4.0, 2.0), (7.0, 5.0, 2.1)),         # inside the box, near-horizontal
    ((4.0, -3.0, 1.5), (4.0, 4.0, 1.5)),        # horizontal, entering through a side
    ((4.0, 4.0, 30.0), (4.0, 4.0001, 0.0)),     # straight down
    ((-5.0, -5.0, 0.5), (8.0, 8.0, 3.5)),       # upward from below the slab
    ((4.0, 4.0, 2.0), (4.0, 4.0, 9.0)),         # inside looking up
    ((4.0, -6.0, 9.0), (4.0, -20.0, 12.0)),     # looking away: pure background
    ((4.0, 4.0, 2.0), (9.0, 4.0, 2.0)),         # axis-parallel centre ray (d_y = d_z = 0 at the centre)
]


@pytest.mark.parametrize("origin,target", EDGE_CAMS)
def test_edge_cameras(omerf, oracle, origin, target):
    rng = np.random.default_rng(12)
    lo = rng.uniform(0.5, 1.5, (9, 9)).astype(np.float32)
    hi = (lo + rng.uniform(-0.2, 2.0, (9, 9))).astype(np.float32)      # a few empty columns (h_up < h_lo)
    sc = synth.custom_scene(h_lo=lo, h_up=hi, seed=5, bias_amp=0.2, bg=(0.2, 0.5, 0.9))
    cam = synth.look_at_camera(origin, target, 48, 40, vfov_deg=70.0)
    rgb, ns, _ = _gpu_render(omerf, sc, cam, 48, 40)
    _assert_parity(rgb, ns, oracle.OracleScene(sc).render(cam, 48, 40, mode="brute"), "edge camera")


def test_empty_scene_is_background_exactly(omerf):
    sc = synth.custom_scene(h_lo=3.0, h_up=1.0, bg=(0.25, 0.5, 0.75))
    cam = synth.look_at_camera((4.0, -6.0, 9.0), (4.0, 4.0, 2.0), 32, 32)
    rgb, ns, _ = _gpu_render(omerf, sc, cam, 32, 32)
    assert ns.sum() == 0
    assert np.array_equal(rgb.astype(np.float32), np.broadcast_to(np.array(sc.bg, dtype=np.float32), rgb.shape))


def test_zero_views_and_batches(omerf, oracle):
    import torch
    sc = synth.make_scene(0)
    W, H = 40, 24
    cams = np.stack([synth.look_at_camera((32.0 + 30 * np.cos(a), 32.0 + 30 * np.sin(a), 25.0 + 3 * i), (32.0, 32.0, 8.0), W, H)
                     for i, a in enumerate(np.linspace(0, 5, 7))])
    with omerf.scene_create(sc) as h:
        L = omerf.load_library()
        dummy = torch.zeros(4, device="cuda")
        assert L.omerf_render(h.ptr, cams.ctypes.data, 0, W, H, dummy.data_ptr(), dummy.data_ptr(), None) == 0
        assert omerf.last_launch_count(h) == 0
        rgb, ns = omerf.render(h, cams, W, H)
        # a second call right behind the first (camera staging ring) on a side stream
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            rgb2, ns2 = omerf.render(h, cams[::-1].copy(), W, H, stream=st)
        torch.cuda.synchronize()
    ref = oracle.OracleScene(sc).render(cams, W, H, mode="clipped")
    _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, "batch")
    assert np.array_equal(ns2.cpu().numpy()[::-1], ns.cpu().numpy())
    assert np.array_equal(rgb2.cpu().numpy()[::-1], rgb.cpu().numpy())


def test_constant_slab_closed_form_on_gpu(omerf):
    """The GPU path against the closed form directly (not via the oracle): T = exp(-tau n step)."""
    import math
    za, zb, byte, step = 1.0, 3.0, 127, 0.125
    sc = synth.custom_scene(box=(32.0, 32.0, 4.0), h_lo=za, h_up=zb, fill=byte, step=step)
    # zero the MLP's last layer: S = sigmoid(0) = 0.5, so rgb = (1-T) sigmoid(pre) + 0.5 + T bg, clamped
    sc.W2[:] = 0
    cam = synth.look_at_camera((16.0, 4.0, 14.0), (16.0, 16.0, 2.0), 16, 16, vfov_deg=20.0)
    rgb, ns, _ = _gpu_render(omerf, sc, cam, 16, 16)
    pre = 4.0 * (byte * 28.0 / 255.0 - 14.0)
    tau = math.exp(pre)
    sig = 1.0 / (1.0 + math.exp(-pre))
    T = np.exp(-tau * ns * step)
    expect = np.clip((1 - T) * sig + 0.5 + T * 1.0, 0, 1)
    assert np.all(ns > 0)
    c = cam.astype(np.float64)
    for v in range(16):
        for u in range(16):
            g = c[9:12] + ((u + 0.5 - c[14]) / c[12]) * c[3:6] - ((v + 0.5 - c[15]) / c[13]) * c[6:9]
            L = (zb - za) / abs(g[2] / np.linalg.norm(g))
            assert abs(ns[0, v, u] * step - L) <= step * 1.001
    sc.bg = (0.0, 0.0, 0.0)
    rgb0, _, _ = _gpu_render(omerf, sc, cam, 16, 16)
    assert np.max(np.abs(rgb0[..., 0] - np.clip((1 - T) * sig + 0.5, 0, 1))) < 1e-4
    assert np.max(np.abs(rgb[..., 0] - expect)) < 1e-4 or np.all(expect == 1.0)


# ----------------------------------------------------------------------------- S1 pyramid
def test_pyramid_levels(omerf):
    sc = synth.make_scene(0)
    with omerf.scene_create(sc) as h:
        info = omerf.scene_info(h)
        assert info["pyramid_levels"] == 8                 # 65 -> 33 -> 17 -> 9 -> 5 -> 3 -> 2 -> 1
        mn, mx = omerf.pyramid_level(h, 0)
        assert np.array_equal(mn, sc.h_lo) and np.array_equal(mx, sc.h_up)
        for l in range(1, info["pyramid_levels"]):
            cmn, cmx = omerf.pyramid_level(h, l)
            assert cmn.shape == ((mn.shape[0] + 1) // 2, (mn.shape[1] + 1) // 2)
            pmn = np.pad(mn, ((0, mn.shape[0] % 2), (0, mn.shape[1] % 2)), constant_values=np.inf)
            pmx = np.pad(mx, ((0, mx.shape[0] % 2), (0, mx.shape[1] % 2)), constant_values=-np.inf)
            ref_mn = pmn.reshape(cmn.shape[0], 2, cmn.shape[1], 2).min(axis=(1, 3))
            ref_mx = pmx.reshape(cmx.shape[0], 2, cmx.shape[1], 2).max(axis=(1, 3))
            assert np.array_equal(cmn, ref_mn) and np.array_equal(cmx, ref_mx)
            mn, mx = cmn, cmx
        assert mn.shape == (1, 1) and mn[0, 0] == sc.h_lo.min() and mx[0, 0] == sc.h_up.max()
        assert info["device_bytes"] >= sc.grid.nbytes + sc.plane_xy.nbytes + sc.plane_xz.nbytes + sc.plane_yz.nbytes


# ----------------------------------------------------------------------------- S10 comparator (config 4 at small size)
@pytest.mark.parametrize("hf_n,occ_n", [((17, 17), (32, 32, 32)), ((9, 12), (20, 23, 7)), ((33, 33), (64, 64, 16))])
def test_bitfield_matches_oracle(omerf, oracle, hf_n, occ_n):
    rng = np.random.default_rng(31)
    lo = (1.0 + 0.5 * rng.random(hf_n)).astype(np.float32)
    hi = (lo - 0.2 + 1.7 * rng.random(hf_n)).astype(np.float32)
    sc = synth.custom_scene(box=(16.0, 12.0, 4.0), hf_n=hf_n, h_lo=lo, h_up=hi, occ_n=occ_n)
    O = oracle.OracleScene(sc, sampler=1)
    with omerf.scene_create(sc, sampler=1) as h:
        bits = omerf.bitfield(h, occ_n)
        info = omerf.scene_info(h)
    assert np.array_equal(bits, O.bits)
    assert info["occ_bits_set"] == int(np.unpackbits(O.bits.view(np.uint8)).sum())


def test_grid_sampler_parity_and_superset(omerf, oracle):
    rng = np.random.default_rng(33)
    m = 33
    lo = (1.0 + 0.5 * rng.random((m, m))).astype(np.float32)
    hi = (lo + 0.3 + 1.5 * rng.random((m, m))).astype(np.float32)
    sc = synth.custom_scene(box=(16.0, 16.0, 4.0), hf_n=(m, m), h_lo=lo, h_up=hi, step=0.125, occ_n=(64, 64, 32), seed=2)
    cams = np.stack([synth.look_at_camera((8.0, -10.0, 14.0), (8.0, 8.0, 2.0), 64, 48),
                     synth.look_at_camera((2.0, 3.0, 2.5), (14.0, 12.0, 1.0), 64, 48)])
    rgb_g, ns_g, _ = _gpu_render(omerf, sc, cams, 64, 48, sampler=1)
    _assert_parity(rgb_g, ns_g, oracle.OracleScene(sc, sampler=1).render(cams, 64, 48, mode="brute"), "grid sampler")
    rgb_p, ns_p, _ = _gpu_render(omerf, sc, cams, 64, 48, sampler=0)
    _assert_parity(rgb_p, ns_p, oracle.OracleScene(sc, sampler=0).render(cams, 64, 48, mode="brute"), "plane sampler")
    assert ns_g.sum() >= ns_p.sum()


# ----------------------------------------------------------------------------- interpolation-weight corner cases
def test_texel_centre_and_weight_256_taps(omerf, oracle):
    """Samples exactly on texel centres (all four bilinear weights collapse to w00 = 2^16) and a hair below a
    centre (fractional weight rounds to 256): the packed-u16 dot-product path of the gather must stay exact (R9)."""
    sc = synth.custom_scene(box=(16.0, 16.0, 8.0), hf_n=(17, 17), h_lo=1.0, h_up=6.0, grid_n=(16, 16, 8),
                            xy_n=(64, 64), xz_n=(64, 32), yz_n=(64, 32), seed=5, step=0.25, smooth=False)
    cams = []
    for dx, dy in ((0.0, 0.0), (-0.25 / 1024, 0.0), (0.0, -0.25 / 1024), (-0.25 / 1024, -0.25 / 1024), (0.125, 0.0)):
        # principal ray straight down through a texel centre of the 0.25-spaced planes (and the shifted variants);
        # z samples fall on texel centres of the xz / yz planes as well: 12 - (k + 1/2)/4 = (j + 1/2)/4
        row = np.array([5.125 + dx, 7.375 + dy, 12.0, 1, 0, 0, 0, 1, 0, 0, 0, -1, 40.0, 40.0, 1.5, 1.5], dtype=np.float32)
        cams.append(row)
    cams = np.stack(cams)
    rgb, ns, _ = _gpu_render(omerf, sc, cams, 3, 3)
    ref = oracle.OracleScene(sc).render(cams, 3, 3, mode="brute")
    assert ref["nsamples"][:, 1, 1].min() >= 1
    _assert_parity(rgb, ns, ref, "texel-centre taps")


def test_gather_probe_replays_every_sample(omerf):
    import torch
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    with omerf.scene_create(sc) as h:
        _, ns = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        res = omerf.gather_probe(h, cams[0], W, H, repeats=2, flush_l2=False)
        assert res["samples"] == int(ns.sum().item())
        assert res["ms_frame_order"] > 0 and res["ms_scattered"] > 0
        # the probe must leave the scene usable
        _, ns2 = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        assert torch.equal(ns, ns2)


def test_planes_with_unrelated_resolutions(omerf, oracle):
    """Plane resolutions that differ per world axis: the gather may not share taps between planes."""
    rng = np.random.default_rng(9)
    m = 21
    lo = (1.0 + rng.random((m, m))).astype(np.float32)
    hi = (lo + 0.5 + 2.0 * rng.random((m, m))).astype(np.float32)
    sc = synth.custom_scene(box=(10.0, 12.0, 5.0), hf_n=(m, m), h_lo=lo, h_up=hi, grid_n=(7, 9, 5), xy_n=(20, 24),
                            xz_n=(28, 12), yz_n=(36, 10), seed=4, step=0.2, bias_amp=0.3)
    cams = np.stack([synth.look_at_camera((5.0, -7.0, 11.0), (5.0, 6.0, 2.0), 48, 40),
                     synth.look_at_camera((1.0, 2.0, 2.2), (9.0, 10.0, 1.5), 48, 40)])
    rgb, ns, _ = _gpu_render(omerf, sc, cams, 48, 40)
    ref = oracle.OracleScene(sc).render(cams, 48, 40, mode="brute")
    assert ref["nsamples"].sum() > 2000
    _assert_parity(rgb, ns, ref, "unrelated plane resolutions")


# ----------------------------------------------------------------------------- soft occupancy (Eq. 6-8)
@pytest.mark.parametrize("eps", [0.3, 1.0, 4.0])
def test_soft_mask_variant(omerf, oracle, eps):
    import torch
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    with omerf.scene_create(sc, soft_eps=eps) as h:
        rgb, ns = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        rgb, ns = rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32)
    ref = oracle.OracleScene(sc, soft_eps=eps).render(cams, W, H, mode="clipped")
    _assert_parity(rgb, ns, ref, f"soft mask eps={eps}")
    hard = oracle.OracleScene(sc).render(cams, W, H, mode="clipped")
    assert np.array_equal(ns, hard["nsamples"])                 # M weights colours, it does not change the samples
    assert np.abs(ref["rgb"] - hard["rgb"]).max() > 1e-2        # and the test would notice a missing M


def test_soft_mask_thin_intervals_and_rejections(omerf, oracle):
    rng = np.random.default_rng(12)
    m = 25
    lo = (1.0 + rng.random((m, m))).astype(np.float32)
    hi = (lo + 0.05 + 1.5 * rng.random((m, m))).astype(np.float32)   # many intervals thinner than 2 eps (R23)
    sc = synth.custom_scene(box=(12.0, 12.0, 4.0), hf_n=(m, m), h_lo=lo, h_up=hi, seed=6, step=0.1, bias_amp=0.2)
    cams = np.stack([synth.look_at_camera((6.0, -5.0, 9.0), (6.0, 6.0, 1.5), 56, 40)])
    import torch
    with omerf.scene_create(sc, soft_eps=0.5) as h:
        rgb, ns = omerf.render(h, cams, 56, 40)
        torch.cuda.synchronize()
    ref = oracle.OracleScene(sc, soft_eps=0.5).render(cams, 56, 40, mode="brute")
    _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, "thin intervals")
    with pytest.raises(omerf.OmerfError):
        omerf.scene_create(sc, soft_eps=-1.0)
    sc_g = synth.custom_scene(box=(12.0, 12.0, 4.0), hf_n=(m, m), h_lo=lo, h_up=hi, seed=6, occ_n=(24, 24, 8))
    with pytest.raises(omerf.OmerfError):
        omerf.scene_create(sc_g, sampler=1, soft_eps=0.5)


# ----------------------------------------------------------------------------- sparse-block grid
@pytest.mark.parametrize("B", [2, 4, 8, 16])
def test_sparse_block_grid_matches_oracle_bake_and_dense_render(omerf, oracle, B):
    """The device bake allocates exactly the oracle's blocks with the oracle's ids (bit-exact table), and rendering
    through the table gives the dense oracle's image: the same texels are fetched."""
    import torch
    rng = np.random.default_rng(21)
    m = 29
    lo = (0.5 + 2.0 * rng.random((m, m))).astype(np.float32)
    hi = (lo + 0.05 + 3.0 * rng.random((m, m))).astype(np.float32)
    kill = rng.random((m, m)) < 0.2
    hi[kill] = lo[kill] - 1.0
    sc = synth.custom_scene(box=(14.0, 13.0, 8.0), hf_n=(m, m), h_lo=lo, h_up=hi, grid_n=(37, 30, 21), xy_n=(64, 64),
                            xz_n=(64, 32), yz_n=(64, 32), seed=11, step=0.15, smooth=False, bias_amp=0.2)
    cams = np.stack([synth.look_at_camera((7.0, -8.0, 15.0), (7.0, 6.5, 2.0), 72, 56),
                     synth.look_at_camera((1.0, 1.5, 3.0), (13.0, 12.0, 2.0), 72, 56)])
    O = oracle.OracleScene(sc)
    S = oracle.SparseBlocks(O, B, atlas=False)
    with omerf.scene_create(sc, grid_block=B) as h:
        info = omerf.scene_info(h)
        assert info["grid_blocks_total"] == S.table.size and info["grid_blocks_allocated"] == S.n_alloc
        assert info["grid_bytes"] == S.n_alloc * B ** 3 * 16 + S.table.size * 4     # 16-byte entries (texel pairs along y)
        assert np.array_equal(omerf.block_table(h), S.table.ravel())
        rgb, ns = omerf.render(h, cams, 72, 56)
        torch.cuda.synchronize()
        res = omerf.gather_probe(h, cams[0], 72, 56, repeats=1, flush_l2=False)
    ref = O.render(cams, 72, 56, mode="brute")
    assert ref["nsamples"].sum() > 5000 and 0 < S.n_alloc < S.table.size
    _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, f"sparse blocks B={B}")
    assert res["samples"] == int(ref["nsamples"][0].sum())


def test_sparse_block_grid_config0_and_rejections(omerf, oracle):
    import torch
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    with omerf.scene_create(sc, grid_block=8) as h:
        rgb, ns = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
    ref = oracle.OracleScene(sc).render(cams, W, H, mode="clipped")
    _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, "config 0, sparse blocks")
    with pytest.raises(omerf.OmerfError):
        omerf.scene_create(sc, grid_block=3)
    with omerf.scene_create(sc) as h:
        with pytest.raises(omerf.OmerfError):
            omerf.block_table(h)


def test_gather_probe_on_grid_sampler_and_sparse_soft_combination(omerf, oracle):
    """The calibration probe follows whatever sampler / layout the scene uses; soft mask + sparse blocks combine."""
    import torch
    rng = np.random.default_rng(33)
    m = 33
    lo = (1.0 + 0.5 * rng.random((m, m))).astype(np.float32)
    hi = (lo + 0.3 + 1.5 * rng.random((m, m))).astype(np.float32)
    sc = synth.custom_scene(box=(16.0, 16.0, 4.0), hf_n=(m, m), h_lo=lo, h_up=hi, grid_n=(16, 16, 8), step=0.125,
                            occ_n=(64, 64, 32), seed=2)
    cams = np.stack([synth.look_at_camera((8.0, -10.0, 14.0), (8.0, 8.0, 2.0), 64, 48)])
    with omerf.scene_create(sc, sampler=1) as h:
        _, ns = omerf.render(h, cams, 64, 48)
        torch.cuda.synchronize()
        assert omerf.gather_probe(h, cams[0], 64, 48, repeats=1, flush_l2=False)["samples"] == int(ns.sum().item())
    with omerf.scene_create(sc, soft_eps=0.4, grid_block=4) as h:
        rgb, ns = omerf.render(h, cams, 64, 48)
        torch.cuda.synchronize()
    ref = oracle.OracleScene(sc, soft_eps=0.4).render(cams, 64, 48, mode="brute")
    _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, "soft mask + sparse blocks")


def test_more_views_than_the_initial_camera_ring_and_repeated_calls(omerf, oracle):
    """40 views (the camera staging ring starts at 16 per slot and must grow), then 20 calls back to back (more calls
    than ring slots), then fewer views again."""
    import torch
    sc = synth.make_scene(0)
    W, H = 24, 16
    cams = np.stack([synth.look_at_camera((32.0 + 28 * np.cos(a), 32.0 + 28 * np.sin(a), 20.0 + 0.5 * i), (32.0, 32.0, 8.0), W, H)
                     for i, a in enumerate(np.linspace(0, 6, 40))])
    ref = oracle.OracleScene(sc).render(cams, W, H, mode="clipped")
    with omerf.scene_create(sc) as h:
        rgb, ns = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, "40 views")
        outs = [omerf.render(h, cams[i:i + 2], W, H) for i in range(20)]
        torch.cuda.synchronize()
        for i, (r2, n2) in enumerate(outs):
            assert np.array_equal(n2.cpu().numpy().view(np.uint32), ref["nsamples"][i:i + 2])
        h_rgb, h_ns = omerf.render_host(h, cams[:3], W, H)
        assert np.array_equal(h_ns, ref["nsamples"][:3])


def test_heatmap_is_bit_exact(omerf, oracle):
    import torch
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    with omerf.scene_create(sc) as h:
        _, ns = omerf.render(h, cams, W, H)
        for n_max in (1, 7, 16, 255):
            hm = omerf.heatmap(ns, n_max)
            torch.cuda.synchronize()
            assert np.array_equal(hm.cpu().numpy(), oracle.heatmap(ns.cpu().numpy().view(np.uint32), n_max))
    with pytest.raises(omerf.OmerfError):
        omerf.heatmap(ns, 0)


def test_device_block_table_against_the_plain_definition(omerf, oracle):
    """The DEVICE bake judged against the plain definition, not against the oracle's formula: on a tiny scene the voxels
    that a dense sampling of the slab really touches (brute force over points that pass Eq. 7) must all lie in blocks
    the device allocated (soundness), and every allocated block must hold a voxel within one voxel of a touched one
    (tightness: the rule may over-mark by its stated padding only)."""
    import math
    from scipy.ndimage import binary_dilation
    rng = np.random.default_rng(7)
    hf, G, box, B = 9, (10, 9, 8), (8.0, 8.0, 4.0), 2
    lo = (0.5 + 2.0 * rng.random((hf, hf))).astype(np.float32)
    hi = (lo + 0.05 + 1.0 * rng.random((hf, hf))).astype(np.float32)
    kill = rng.random((hf, hf)) < 0.2
    hi[kill] = lo[kill] - 1.0
    sc = synth.custom_scene(box=box, hf_n=(hf, hf), h_lo=lo, h_up=hi, grid_n=G, seed=7, smooth=False)
    O = oracle.OracleScene(sc)
    touched = np.zeros(G, dtype=bool)
    xs = np.linspace(0.0, 8.0, 161, dtype=np.float32)[:-1] + np.float32(0.013)
    zs = np.linspace(0.0, 4.0, 201, dtype=np.float32)[:-1] + np.float32(0.007)
    for x in xs:
        for y in xs:
            ix, iy = int(math.floor(x + 0.5)), int(math.floor(y + 0.5))
            for z in zs[(zs >= sc.h_lo[ix, iy]) & (zs <= sc.h_up[ix, iy])]:
                c = oracle.grid_corners(O, np.array([x, y, z], dtype=np.float32))
                touched[c[0]:c[1] + 1, c[2]:c[3] + 1, c[4]:c[5] + 1] = True
    assert touched.sum() > 50
    with omerf.scene_create(sc, grid_block=B) as h:
        nb = tuple((g + B - 1) // B for g in G)
        alloc = omerf.block_table(h).reshape(nb) >= 0
    vox_alloc = np.repeat(np.repeat(np.repeat(alloc, B, 0), B, 1), B, 2)[:G[0], :G[1], :G[2]]
    assert not (touched & ~vox_alloc).any()                                    # soundness
    near = binary_dilation(touched, structure=np.ones((3, 3, 3), bool))
    pad = np.zeros(tuple(n * B for n in nb), dtype=bool)
    pad[:G[0], :G[1], :G[2]] = near
    blocks_near = pad.reshape(nb[0], B, nb[1], B, nb[2], B).any(axis=(1, 3, 5))
    assert not (alloc & ~blocks_near).any()                                    # tightness
    assert 0 < alloc.sum() < alloc.size


# ----------------------------------------------------------------------------- SURVEY 8(f).1, second half: low-z triplane bake
def _lowz_scene(seed, m=21, lo_rng=(2.2, 3.0), thick=(0.05, 1.5), empty=0.2, **kw):
    rng = np.random.default_rng(seed)
    lo = (lo_rng[0] + (lo_rng[1] - lo_rng[0]) * rng.random((m, m))).astype(np.float32)
    hi = (lo + thick[0] + (thick[1] - thick[0]) * rng.random((m, m))).astype(np.float32)
    kill = rng.random((m, m)) < empty
    lo[kill], hi[kill] = 7.5, 0.2                                  # empty columns must not widen the band
    return synth.custom_scene(box=(14.0, 13.0, 8.0), hf_n=(m, m), h_lo=lo, h_up=hi, grid_n=(20, 18, 12), xy_n=(64, 60),
                              xz_n=(64, 48), yz_n=(60, 40), seed=seed, step=0.15, smooth=False, bias_amp=0.2, **kw)


@pytest.mark.parametrize("seed", [1, 2])
def test_lowz_bake_band_is_the_oracles_and_the_image_is_unchanged(omerf, oracle, seed):
    """PAPER.md:186 / DESIGN.md R27: the device keeps exactly the oracle's band of z rows (bit-exact integers), stores
    fewer plane bytes, and renders the UNCROPPED oracle's image (same texels fetched), alone and with sparse blocks + soft mask."""
    import torch
    sc = _lowz_scene(seed)
    cams = np.stack([synth.look_at_camera((7.0, -8.0, 15.0), (7.0, 6.5, 2.0), 72, 56),
                     synth.look_at_camera((1.0, 1.5, 3.0), (13.0, 12.0, 2.6), 72, 56)])
    O = oracle.OracleScene(sc)
    bands = {w: oracle.LowZBand(O, w, crop=False) for w in ("xz", "yz")}
    with omerf.scene_create(sc) as h:
        full = omerf.scene_info(h)
    assert full["xz_band"] == (0, 47) and full["yz_band"] == (0, 39)
    with omerf.scene_create(sc, lowz_bake=True) as h:
        info = omerf.scene_info(h)
        rgb, ns = omerf.render(h, cams, 72, 56)
        torch.cuda.synchronize()
        probe = omerf.gather_probe(h, cams[0], 72, 56, repeats=1, flush_l2=False)
    assert info["xz_band"] == (bands["xz"].b_lo, bands["xz"].b_hi) and info["yz_band"] == (bands["yz"].b_lo, bands["yz"].b_hi)
    assert bands["xz"].rows < 48 and bands["yz"].rows < 40
    assert full["plane_bytes"] - info["plane_bytes"] == 16 * (64 * (48 - bands["xz"].rows) + 60 * (40 - bands["yz"].rows))
    ref = O.render(cams, 72, 56, mode="brute")
    assert ref["nsamples"].sum() > 3000
    _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, "low-z bake")
    assert probe["samples"] == int(ref["nsamples"][0].sum())
    with omerf.scene_create(sc, lowz_bake=True, grid_block=4, soft_eps=0.3) as h:
        rgb, ns = omerf.render(h, cams, 72, 56)
        torch.cuda.synchronize()
    ref = oracle.OracleScene(sc, soft_eps=0.3).render(cams, 72, 56, mode="brute")
    _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32), ref, "low-z + sparse + soft")


def test_lowz_bake_degenerate_scenes_and_rejections(omerf, oracle):
    import torch
    cam = synth.look_at_camera((4.0, -6.0, 9.0), (4.0, 4.0, 2.0), 40, 30)
    for lo, hi, want in ((3.0, 1.0, (0, 0)),        # no occupied column: one row is kept, nothing is ever fetched
                         (-2.0, 9.0, (0, 31)),      # slab larger than the box: the whole plane
                         (1.0, 1.0, None)):         # zero-thickness slab
        sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=lo, h_up=hi, xz_n=(16, 32), yz_n=(16, 32), seed=3)
        O = oracle.OracleScene(sc)
        Bd = oracle.LowZBand(O, "xz", crop=False)
        with omerf.scene_create(sc, lowz_bake=True) as h:
            info = omerf.scene_info(h)
            rgb, ns = omerf.render(h, cam, 40, 30)
            torch.cuda.synchronize()
        assert info["xz_band"] == (Bd.b_lo, Bd.b_hi) == info["yz_band"]
        if want is not None:
            assert info["xz_band"] == want
        _assert_parity(rgb.cpu().numpy().astype(np.float64), ns.cpu().numpy().view(np.uint32),
                       O.render(cam, 40, 30, mode="brute"), f"low-z, slab [{lo}, {hi}]")
    sc = synth.custom_scene(occ_n=(8, 8, 8))
    with pytest.raises(omerf.OmerfError):
        omerf.scene_create(sc, sampler=1, lowz_bake=True)     # the grid sampler's voxels are a superset of the slab


# ----------------------------------------------------------------------------- the exact in-box index range (setup_ray)
def _axis_camera(origin, fwd, up, W, H, f=20.0):
    """camera row with an exactly axis-aligned frame (so rays through the principal point have zero components)"""
    fwd = np.asarray(fwd, dtype=np.float64)
    up = np.asarray(up, dtype=np.float64)
    right = np.cross(fwd, up)
    return np.concatenate([origin, right, up, fwd, [f, f, W / 2.0, H / 2.0]]).astype(np.float32)


FACE_CAMS = [
    ((0.0, 4.0, 2.0), (1, 0, 0), (0, 0, 1)),     # origin ON the face x = 0, looking in: first lattice points just inside
    ((8.0, 4.0, 2.0), (-1, 0, 0), (0, 0, 1)),    # origin ON the far face x = X (p < X fails at t = 0), looking in
    ((4.0, 4.0, 4.0), (0, 0, -1), (0, 1, 0)),    # origin ON the top face z = Z, straight down
    ((4.0, 0.0, 0.0), (0, 1, 0), (0, 0, 1)),     # origin ON the edge y = 0, z = 0: rays along the bottom face
    ((0.0, 0.0, 0.0), (1, 0, 0), (0, 0, 1)),     # origin ON a corner, along an edge of the box
    ((-3.0, 8.0, 2.0), (1, 0, 0), (0, 0, 1)),    # in the plane y = Y (never inside: p.y < Y fails), grazing
    ((-3.0, 7.999999, 3.9999998), (1, 0, 0), (0, 0, 1)),   # one ulp inside two faces, parallel to both
    ((4.0, 4.0, 2.0), (1, 0, 0), (0, 0, 1)),     # inside, axis-parallel
]


@pytest.mark.parametrize("sampler", [0, 1])
@pytest.mark.parametrize("origin,fwd,up", FACE_CAMS)
def test_cameras_on_faces_edges_and_grazing_rays(omerf, oracle, origin, fwd, up, sampler):
    """setup_ray searches the exact range of lattice indices inside the box and the march then drops every box test and
    clamp: rays that start on a face, run inside a face plane, or are parallel to an axis (zero direction components,
    odd image sizes put a pixel centre on the principal point) must still give the brute-force oracle's counts."""
    rng = np.random.default_rng(3)
    lo = rng.uniform(0.0, 1.5, (9, 9)).astype(np.float32)
    hi = (lo + rng.uniform(-0.2, 2.6, (9, 9))).astype(np.float32)      # some empty columns, some reaching the top face
    hi[2:4, 2:4] = 4.0
    lo[5:7, 5:7] = 0.0
    sc = synth.custom_scene(h_lo=lo, h_up=hi, seed=8, bias_amp=0.1, occ_n=(16, 16, 8) if sampler else (0, 0, 0))
    W, H = 33, 21
    cam = _axis_camera(origin, fwd, up, W, H)
    rgb, ns, _ = _gpu_render(omerf, sc, cam, W, H, sampler=sampler)
    _assert_parity(rgb, ns, oracle.OracleScene(sc, sampler=sampler).render(cam, W, H, mode="brute"), f"face camera {origin}")
