"""SURVEY 8(e) on the GPU (-m gpu): every rank's share of a partitioned batch, rendered through omerf_render_tiles /
omerf_render on one device, stitches to the single-rank render bit for bit.  (The N-rank plumbing itself - process
group, gather onto rank 0 - is covered on CPU with gloo in tests/test_bench_host.py.)"""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def omerf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2404_09531_b200 as m
    m.load_library()
    return m


@pytest.mark.parametrize("world", [2, 3, 8])
def test_shares_stitch_to_the_single_rank_render(omerf, world):
    import torch

    from paper_2404_09531_b200 import partition
    sc = synth.make_scene(0)
    for cams, W, H in ((synth.make_cameras(0), 130, 99),               # one view: bands of tile rows, ragged sizes
                       (synth.orbit_cameras(0, 16), 64, 48)):          # 16 views: whole views, longest first
        n_views = cams.shape[0]
        with omerf.scene_create(sc) as h:
            rgb, ns = omerf.render(h, cams, W, H)
            torch.cuda.synchronize()
            full_rgb, full_n = rgb.cpu().numpy(), ns.cpu().numpy()
            plans = partition.make_plans(full_n.view(np.uint32), world)          # previous frame's counts
            parts = []
            for plan in plans:
                if plan.mode == "views":
                    r, n = omerf.render(h, cams[plan.views], W, H)
                    torch.cuda.synchronize()
                    parts.append((r.cpu().numpy(), n.cpu().numpy()))
                else:
                    r = torch.full((n_views, H, W, 3), -7.0, dtype=torch.float32, device="cuda")
                    n = torch.full((n_views, H, W), -7, dtype=torch.int32, device="cuda")
                    omerf.render_tiles(h, cams, W, H, r, n, plan.tile_first, plan.tile_end)
                    torch.cuda.synchronize()
                    r0, r1 = partition.pixel_row_range(plan, H)
                    rr, nn = r.cpu().numpy().reshape(n_views * H, W, 3), n.cpu().numpy().reshape(n_views * H, W)
                    assert np.all(nn[:r0] == -7) and np.all(nn[r1:] == -7) and np.all(rr[:r0] == -7.0)   # nothing else is written
                    parts.append((rr[r0:r1], nn[r0:r1]))
        got_rgb, got_n = partition.stitch(plans, parts, n_views, H, W)
        assert np.array_equal(got_n, full_n) and np.array_equal(got_rgb, full_rgb)
        assert sum(p.samples for p in plans) == int(full_n.view(np.uint32).sum())


def test_render_tiles_argument_checks(omerf):
    import torch
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = 64, 48
    tiles = 8 * 12
    with omerf.scene_create(sc) as h:
        r = torch.zeros((1, H, W, 3), dtype=torch.float32, device="cuda")
        n = torch.zeros((1, H, W), dtype=torch.int32, device="cuda")
        omerf.render_tiles(h, cams, W, H, r, n, 5, 5)                  # empty range: no-op
        torch.cuda.synchronize()
        assert omerf.last_launch_count(h) == 0 and int(n.abs().sum().item()) == 0
        for first, end in ((3, 2), (0, tiles + 1)):
            with pytest.raises(omerf.OmerfError):
                omerf.render_tiles(h, cams, W, H, r, n, first, end)
        omerf.render_tiles(h, cams, W, H, r, n, 0, tiles)
        ref_r, ref_n = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        assert torch.equal(n, ref_n) and torch.equal(r, ref_r)
