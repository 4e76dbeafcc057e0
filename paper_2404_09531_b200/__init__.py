"""B200-native Oblique-MERF renderer (arxiv 2404.09531): Python face of the C-ABI in include/omerf.h.

    import paper_2404_09531_b200 as omerf
    h = omerf.scene_create(scene)                      # omerf_scene_create
    rgb, ns = omerf.render(h, cameras, W, H)           # omerf_render (device tensors, async)
    omerf.scene_destroy(h)                             # omerf_scene_destroy

All arithmetic runs in hand-written CUDA kernels (csrc/*.cu, sm_100a).  No CPU fallback.
"""
from .binding import (  # noqa: F401
    SAMPLER_GRID,
    SAMPLER_PLANE,
    STATIC_MAX_VIEWS,
    EXPORTS,
    LIB_PATH,
    OmerfError,
    SceneHandle,
    bitfield,
    block_table,
    gather_probe,
    heatmap,
    last_launch_count,
    load_library,
    mlp_smoothness,
    pyramid_level,
    render,
    render_host,
    render_host_async,
    render_static,
    render_tiles,
    scene_create,
    scene_destroy,
    scene_info,
    wait,
)
