"""The range-checked build of the CUDA library (libomerf_checked.so, -DOMERF_CHECKED) on the small workloads (-m gpu).

compute-sanitizer is closed on the GPU pool (profiles/r02_checked_build.md), so the memcheck role is taken by the
library's own device-side range checks: every global-memory index (pyramid, V, the three planes, block table, bitfield,
cameras, output pixels) and every ray-pool slot the render kernels use is compared with its bound; a violation is
recorded in a device word (omerf_check_errors) instead of faulting.  The checked library must report no violation and
produce the shipped library's images bit for bit."""
import ctypes as C

import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def libs():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2404_09531_b200 import binding, build
    build.build()
    checked = build.build(checked=True)

    class Swap:
        """binding.* routed through the checked library inside the `with` block"""

        def __enter__(self):
            self.saved = (binding._lib, binding.LIB_PATH)
            binding._lib, binding.LIB_PATH = None, checked
            self.lib = binding.load_library()
            assert self.lib.omerf_check_errors() == 0
            return self.lib

        def __exit__(self, *exc):
            binding._lib, binding.LIB_PATH = self.saved

    return Swap


def _render(scene, cams, W, H, **kw):
    import torch
    import paper_2404_09531_b200 as omerf
    with omerf.scene_create(scene, **kw) as h:
        rgb, ns = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        return rgb.cpu().numpy(), ns.cpu().numpy()


CASES = [
    ("config0 plain", dict()),
    ("sparse blocks + soft mask", dict(soft_eps=1.0, grid_block=4)),
    ("low-z bake", dict(lowz_bake=True)),
    ("grid sampler", dict(sampler=1)),
]


@pytest.mark.parametrize("name,kw", CASES, ids=[c[0] for c in CASES])
def test_checked_build_reports_nothing_and_matches_the_shipped_library(libs, name, kw):
    scene = synth.make_scene(0)
    if kw.get("sampler") == 1:
        scene.occ_n = (64, 64, 16)
    cams = synth.make_cameras(0)
    W, H = synth.config_resolution(0)
    ref_rgb, ref_n = _render(scene, cams, W, H, **kw)
    with libs() as L:
        rgb, ns = _render(scene, cams, W, H, **kw)
        assert L.omerf_check_errors() == 0, "a device index left its array"
    assert np.array_equal(ns, ref_n) and np.array_equal(rgb, ref_rgb)


def test_checked_build_edge_cameras_ragged_sizes_and_probe(libs):
    """cameras inside the box, looking away, axis-parallel; image sizes that are not multiples of the 8x4 tile; a batch;
    the gather probe's replay"""
    import torch
    import paper_2404_09531_b200 as omerf
    rng = np.random.default_rng(12)
    lo = rng.uniform(0.5, 1.5, (9, 9)).astype(np.float32)
    hi = (lo + rng.uniform(-0.2, 2.0, (9, 9))).astype(np.float32)      # a few empty columns (h_up < h_lo)
    scene = synth.custom_scene(h_lo=lo, h_up=hi, seed=5, bias_amp=0.2)
    cams = np.stack([synth.look_at_camera(o, t, 37, 23, vfov_deg=70.0) for o, t in
                     [((4.0, 4.0, 2.0), (7.0, 5.0, 2.1)), ((4.0, -3.0, 1.5), (4.0, 4.0, 1.5)), ((4.0, 4.0, 30.0), (4.0, 4.0001, 0.0)),
                      ((-5.0, -5.0, 0.5), (8.0, 8.0, 3.5)), ((4.0, 4.0, 2.0), (4.0, 4.0, 9.0)), ((4.0, -6.0, 9.0), (4.0, -20.0, 12.0)),
                      ((4.0, 4.0, 2.0), (9.0, 4.0, 2.0))]])
    with libs() as L:
        with omerf.scene_create(scene) as h:
            rgb, ns = omerf.render(h, cams, 37, 23)
            torch.cuda.synchronize()
            omerf.gather_probe(h, cams[0], 37, 23, repeats=1, flush_l2=False)
        assert L.omerf_check_errors() == 0
    ref_rgb, ref_n = _render(scene, cams, 37, 23)
    assert np.array_equal(ns.cpu().numpy(), ref_n) and np.array_equal(rgb.cpu().numpy(), ref_rgb)


def test_checked_build_at_the_timed_size(libs):
    """configs[1] (1920x1080, 8.3 M samples) and configs[5]'s in-box cameras through the checked library: plain path,
    sparse blocks + soft mask, low-z bake; no violation, counts equal to the shipped library's"""
    import torch
    import paper_2404_09531_b200 as omerf
    scene = synth.make_scene(1)
    runs = [(1, {}), (1, dict(grid_block=4, soft_eps=2.0)), (1, dict(lowz_bake=True)), (5, {})]
    ref = []
    for cfg, kw in runs:
        cams = synth.make_cameras(cfg)
        W, H = synth.config_resolution(cfg)
        with omerf.scene_create(scene, **kw) as h:
            _, ns = omerf.render(h, cams, W, H)
            torch.cuda.synchronize()
            ref.append(ns.cpu())
    with libs() as L:
        for (cfg, kw), want in zip(runs, ref):
            cams = synth.make_cameras(cfg)
            W, H = synth.config_resolution(cfg)
            with omerf.scene_create(scene, **kw) as h:
                _, ns = omerf.render(h, cams, W, H)
                torch.cuda.synchronize()
                omerf.gather_probe(h, cams[0], W, H, repeats=1, flush_l2=False)
            assert L.omerf_check_errors() == 0, f"config {cfg} {kw}: a device index left its array"
            assert torch.equal(ns.cpu(), want)
