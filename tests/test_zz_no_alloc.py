"""omerf_render_static, the render call that allocates nothing, against omerf_render (run on the B200 box: -m gpu).

Why the entry point exists: omerf_render grows its camera ring with cudaMalloc / cudaMallocHost behind a
cudaDeviceSynchronize whenever a call brings more views than any call before it.  A frame loop with a deadline cannot take
that device-wide stall at a moment it did not choose, and a plug-in inside a host program that owns all GPU memory (or
forbids driver allocations after start-up) cannot allocate at all.  omerf_render_static runs the same march kernel with
its scratch - device cameras and work-queue head - in one fixed 2304-byte array inside the library, so it takes at most
32 views per call, and every call on a GPU shares that array and finds the previous call's contents in it.

What is checked: two calls in a row on one stream, with different view counts, cameras and image sizes, each give the
image omerf_render gives (sample counts identical, colours within the suite's 2e-3 bar): nothing stale from the first
call (queue head past the end, cameras of other views) reaches the second.  Then the limit: 33 views are refused with a
message that names it, and the call after a refusal still renders correctly.

This file sorts last on purpose: the suite runs with pytest -x, and a failure here must not hide any other test.  It holds
no state of its own, so it passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu

RGB_TOL = 2e-3   # the parity bar of the other GPU tests (tests/test_gpu_parity.py)


@pytest.fixture(scope="module")
def omerf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2404_09531_b200 as m
    m.load_library()
    return m


def _outputs(n, W, H, fill):
    """The caller's output buffers, pre-filled so that a pixel the call did not write shows up."""
    import torch
    rgb = torch.full((n, H, W, 3), float(fill), dtype=torch.float32, device="cuda")
    ns = torch.full((n, H, W), 0x7fffffff, dtype=torch.int32, device="cuda")
    return rgb, ns


def _same_image(got, ref, what):
    import torch
    torch.cuda.synchronize()
    (g_rgb, g_n), (r_rgb, r_n) = got, ref
    bad = int((g_n != r_n).sum())
    assert bad == 0, f"{what}: {bad} pixels with other sample counts than omerf_render"
    assert int(r_n.sum()) > 0, f"{what}: the view sees nothing, the comparison would be empty"
    err = float((g_rgb.double() - r_rgb.double()).abs().max())
    assert err <= RGB_TOL, f"{what}: max |dRGB| against omerf_render = {err}"


def test_two_calls_in_a_row_match_the_allocating_path(omerf):
    sc = synth.make_scene(0)
    W1, H1 = 96, 64
    cams1 = np.stack([synth.look_at_camera((10.0, -14.0, 30.0), (32.0, 32.0, 8.0), W1, H1),
                      synth.look_at_camera((70.0, 70.0, 25.0), (32.0, 32.0, 6.0), W1, H1),
                      synth.look_at_camera((32.0, 32.0, 60.0), (32.0, 32.5, 0.0), W1, H1)])
    W2, H2 = 61, 45                                             # ragged tiles, one view, another pose
    cams2 = synth.look_at_camera((-20.0, 30.0, 18.0), (32.0, 32.0, 8.0), W2, H2)
    with omerf.scene_create(sc) as h:
        ref1 = omerf.render(h, cams1, W1, H1)
        ref2 = omerf.render(h, cams2, W2, H2)
        got1 = omerf.render_static(h, cams1, W1, H1, *_outputs(3, W1, H1, -1.0))
        assert omerf.last_launch_count(h) == 2                  # camera staging kernel + march kernel
        got2 = omerf.render_static(h, cams2, W2, H2, *_outputs(1, W2, H2, -2.0))   # straight after, same stream
        _same_image(got1, ref1, "first call (3 views)")
        _same_image(got2, ref2, "second call (1 view)")
        # and once more with the first batch: the array now holds the second call's leftovers
        got3 = omerf.render_static(h, cams1, W1, H1, *_outputs(3, W1, H1, -3.0))
        _same_image(got3, ref1, "third call (3 views again)")


def test_more_views_than_the_array_holds_are_refused(omerf):
    sc = synth.make_scene(0)
    W, H = 16, 8
    one = synth.look_at_camera((10.0, -14.0, 30.0), (32.0, 32.0, 8.0), W, H)
    too_many = np.tile(one, (omerf.STATIC_MAX_VIEWS + 1, 1))
    full = np.tile(one, (omerf.STATIC_MAX_VIEWS, 1))
    with omerf.scene_create(sc) as h:
        with pytest.raises(omerf.OmerfError, match=f"at most {omerf.STATIC_MAX_VIEWS} views"):
            omerf.render_static(h, too_many, W, H, *_outputs(omerf.STATIC_MAX_VIEWS + 1, W, H, -1.0))
        ref = omerf.render(h, full, W, H)
        got = omerf.render_static(h, full, W, H, *_outputs(omerf.STATIC_MAX_VIEWS, W, H, -1.0))   # exactly the limit
        _same_image(got, ref, f"{omerf.STATIC_MAX_VIEWS} views")
