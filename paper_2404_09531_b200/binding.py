"""Thin ctypes binding of include/omerf.h — argument marshalling only.

Every step of the path runs in the CUDA kernels of libomerf.so; PyTorch is used for device
memory and streams.  There is no CPU fallback: a missing library or a missing GPU raises.
Function names mirror the C-ABI: scene_create / render / render_host / scene_destroy.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libomerf.so")

_f32p = C.POINTER(C.c_float)
_u8p = C.POINTER(C.c_uint8)
_u32p = C.POINTER(C.c_uint32)

SAMPLER_PLANE = 0
SAMPLER_GRID = 1
STATIC_MAX_VIEWS = 32           # OMERF_STATIC_MAX_VIEWS of include/omerf.h

EXPORTS = (
    "omerf_scene_create", "omerf_render", "omerf_render_tiles", "omerf_render_host", "omerf_render_host_async", "omerf_wait", "omerf_render_static", "omerf_gather_probe", "omerf_mlp_smoothness", "omerf_heatmap",
    "omerf_last_launch_count",
    "omerf_scene_get_info", "omerf_scene_get_pyramid_level", "omerf_scene_get_bitfield", "omerf_scene_get_block_table",
    "omerf_scene_destroy", "omerf_last_error", "omerf_version", "omerf_check_errors",
)


class SceneDesc(C.Structure):
    _fields_ = [
        ("box", C.c_float * 3),
        ("hf_n", C.c_int32 * 2), ("h_lo", _f32p), ("h_up", _f32p),
        ("grid_n", C.c_int32 * 3), ("grid", _u8p),
        ("xy_n", C.c_int32 * 2), ("xz_n", C.c_int32 * 2), ("yz_n", C.c_int32 * 2),
        ("plane_xy", _u8p), ("plane_xz", _u8p), ("plane_yz", _u8p),
        ("deq_scale", C.c_float), ("deq_bias", C.c_float),
        ("mlp_in", C.c_int32), ("mlp_hidden", C.c_int32),
        ("W0", _f32p), ("b0", _f32p), ("W1", _f32p), ("b1", _f32p), ("W2", _f32p), ("b2", _f32p),
        ("step", C.c_float), ("t_stop", C.c_float), ("bg", C.c_float * 3),
        ("sampler", C.c_int32), ("occ_n", C.c_int32 * 3),
        ("soft_eps", C.c_float), ("grid_block", C.c_int32), ("lowz_bake", C.c_int32),
    ]


class SceneInfo(C.Structure):
    _fields_ = [("device_bytes", C.c_uint64), ("pyramid_levels", C.c_int32), ("sampler", C.c_int32),
                ("occ_bits_set", C.c_uint64), ("grid_bytes", C.c_uint64), ("grid_blocks_total", C.c_uint64),
                ("grid_blocks_allocated", C.c_uint64), ("plane_bytes", C.c_uint64),
                ("xz_band", C.c_int32 * 2), ("yz_band", C.c_int32 * 2)]


class GatherProbeResult(C.Structure):
    _fields_ = [("samples", C.c_uint64), ("ms_frame_order", C.c_double), ("ms_scattered", C.c_double)]


class OmerfError(RuntimeError):
    pass


_lib = None


def load_library() -> C.CDLL:
    """dlopen libomerf.so (built in-tree by paper_2404_09531_b200.build).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise OmerfError(f"{LIB_PATH} not found: build it with `python -m paper_2404_09531_b200.build` "
                         "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.omerf_last_error.restype = C.c_char_p
    L.omerf_version.restype = C.c_char_p
    L.omerf_check_errors.restype = C.c_uint32
    L.omerf_scene_create.argtypes = [C.POINTER(SceneDesc), C.POINTER(C.c_void_p)]
    L.omerf_render.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    L.omerf_render_host.argtypes = L.omerf_render.argtypes
    L.omerf_render_static.argtypes = L.omerf_render.argtypes
    L.omerf_render_host_async.argtypes = L.omerf_render.argtypes
    L.omerf_wait.argtypes = [C.c_void_p]
    L.omerf_render_tiles.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_uint32,
                                     C.c_uint32, C.c_void_p]
    L.omerf_gather_probe.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int,
                                     C.POINTER(GatherProbeResult)]
    L.omerf_mlp_smoothness.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p]
    L.omerf_heatmap.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]
    L.omerf_last_launch_count.argtypes = [C.c_void_p]
    L.omerf_scene_get_info.argtypes = [C.c_void_p, C.POINTER(SceneInfo)]
    L.omerf_scene_get_pyramid_level.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                                C.c_void_p, C.c_void_p]
    L.omerf_scene_get_bitfield.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
    L.omerf_scene_get_block_table.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64]
    L.omerf_scene_destroy.argtypes = [C.c_void_p]
    L.omerf_scene_destroy.restype = None
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != 0:
        raise OmerfError(f"{what} failed ({rc}): {load_library().omerf_last_error().decode()}")


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def make_desc(scene, sampler: int = SAMPLER_PLANE, soft_eps: float = 0.0, grid_block: int = 0, lowz_bake: bool = False):
    """Fill an omerf_scene_desc from an object with synth.Scene's attributes. Returns (desc, keepalive)."""
    d = SceneDesc()
    keep = []

    def arr(a, dt, pt):
        a = _np(a, dt)
        keep.append(a)
        return a, a.ctypes.data_as(pt)

    d.box[:] = scene.box
    lo, d.h_lo = arr(scene.h_lo, np.float32, _f32p)
    _, d.h_up = arr(scene.h_up, np.float32, _f32p)
    d.hf_n[:] = lo.shape
    g, d.grid = arr(scene.grid, np.uint8, _u8p)
    assert g.ndim == 4 and g.shape[3] == 8, "grid must be [Gx][Gy][Gz][8] uint8"
    d.grid_n[:] = g.shape[:3]
    assert lo.ndim == 2 and np.shape(scene.h_up) == lo.shape, "h_lo / h_up must be [Mx][My]"
    for nm in ("xy", "xz", "yz"):
        p, ptr = arr(getattr(scene, "plane_" + nm), np.uint8, _u8p)
        assert p.ndim == 3 and p.shape[2] == 8, f"plane_{nm} must be [A][B][8] uint8"
        getattr(d, nm + "_n")[:] = p.shape[:2]
        setattr(d, "plane_" + nm, ptr)
    d.deq_scale, d.deq_bias = scene.deq_scale, scene.deq_bias
    W0 = _np(scene.W0, np.float32)
    d.mlp_in, d.mlp_hidden = W0.shape[1], W0.shape[0]
    for nm in ("W0", "b0", "W1", "b1", "W2", "b2"):
        _, ptr = arr(getattr(scene, nm), np.float32, _f32p)
        setattr(d, nm, ptr)
    d.step, d.t_stop = scene.step, scene.t_stop
    d.bg[:] = scene.bg
    d.sampler = sampler
    d.soft_eps = soft_eps
    d.grid_block = grid_block
    d.lowz_bake = int(lowz_bake)
    d.occ_n[:] = scene.occ_n
    return d, keep


class SceneHandle:
    """Owns one omerf_scene*.  Use scene_create(); free with scene_destroy() or as a context manager."""

    def __init__(self, ptr):
        self.ptr = ptr

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        scene_destroy(self)

    def __del__(self):
        try:
            scene_destroy(self)
        except Exception:
            pass


def scene_create(scene, sampler: int = SAMPLER_PLANE, soft_eps: float = 0.0, grid_block: int = 0,
                 lowz_bake: bool = False) -> SceneHandle:
    """omerf_scene_create: upload + re-layout + pyramid (+ bitfield) on the current CUDA device."""
    import torch
    if not torch.cuda.is_available():
        raise OmerfError("no CUDA device: the renderer has no CPU fallback")
    torch.cuda.init()
    torch.cuda.current_stream()          # make sure torch's primary context is current
    L = load_library()
    d, keep = make_desc(scene, sampler, soft_eps, grid_block, lowz_bake)
    out = C.c_void_p()
    _check(L.omerf_scene_create(C.byref(d), C.byref(out)), "omerf_scene_create")
    del keep
    return SceneHandle(out)


def scene_destroy(h: SceneHandle):
    if h is not None and h.ptr:
        load_library().omerf_scene_destroy(h.ptr)
        h.ptr = None


def _cams(cameras):
    cams = _np(np.atleast_2d(cameras), np.float32)
    assert cams.shape[1] == 16, "camera rows are origin,right,up,fwd,fx,fy,cx,cy (16 floats)"
    return cams


def render(h: SceneHandle, cameras, W: int, H: int, out_rgb=None, out_nsamples=None, stream=None):
    """omerf_render: enqueue on `stream` (default: torch's current stream); DEVICE outputs (torch tensors).
    Returns (out_rgb float32 [n][H][W][3], out_nsamples int32-viewed uint32 [n][H][W]); asynchronous."""
    import torch
    cams = _cams(cameras)
    n = cams.shape[0]
    if out_rgb is None:
        out_rgb = torch.empty((n, H, W, 3), dtype=torch.float32, device="cuda")
    if out_nsamples is None:
        out_nsamples = torch.empty((n, H, W), dtype=torch.int32, device="cuda")
    assert out_rgb.is_cuda and out_rgb.is_contiguous() and out_rgb.dtype == torch.float32 and out_rgb.numel() == n * H * W * 3
    assert out_nsamples.is_cuda and out_nsamples.is_contiguous() and out_nsamples.element_size() == 4 \
        and out_nsamples.numel() == n * H * W
    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().omerf_render(h.ptr, cams.ctypes.data, n, W, H, out_rgb.data_ptr(), out_nsamples.data_ptr(),
                                       st.cuda_stream), "omerf_render")
    return out_rgb, out_nsamples


def render_tiles(h: SceneHandle, cameras, W: int, H: int, out_rgb, out_nsamples, tile_first: int, tile_end: int, stream=None):
    """omerf_render_tiles: only the 8x4 tiles [tile_first, tile_end) of the batch are rendered into the FULL batch
    buffers (DEVICE torch tensors); asynchronous."""
    import torch
    cams = _cams(cameras)
    n = cams.shape[0]
    assert out_rgb.is_cuda and out_rgb.is_contiguous() and out_rgb.dtype == torch.float32 and out_rgb.numel() == n * H * W * 3
    assert out_nsamples.is_cuda and out_nsamples.is_contiguous() and out_nsamples.element_size() == 4 \
        and out_nsamples.numel() == n * H * W
    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().omerf_render_tiles(h.ptr, cams.ctypes.data, n, W, H, out_rgb.data_ptr(), out_nsamples.data_ptr(),
                                             int(tile_first), int(tile_end), st.cuda_stream), "omerf_render_tiles")
    return out_rgb, out_nsamples


def render_static(h: SceneHandle, cameras, W: int, H: int, out_rgb, out_nsamples, stream=None):
    """omerf_render_static: omerf_render for callers that must not allocate device memory - a frame loop that cannot
    afford the device-wide stall of a cudaMalloc, or a plug-in whose host program owns all GPU memory.  The march
    kernel's scratch (device cameras, work-queue head) is a fixed 2304-byte array inside the library instead of a
    ring the call may have to grow, so at most STATIC_MAX_VIEWS (32) views per call; more raises OmerfError.  Both
    outputs are the caller's DEVICE tensors (this wrapper does not create them either).  Every call on a GPU shares
    the one array: back-to-back calls on one stream are fine, calls on unordered streams race.  The first call on a
    device looks up the array's address; make it before any stream capture.  Asynchronous on `stream`."""
    import torch
    cams = _cams(cameras)
    n = cams.shape[0]
    assert out_rgb.is_cuda and out_rgb.is_contiguous() and out_rgb.dtype == torch.float32 and out_rgb.numel() == n * H * W * 3
    assert out_nsamples.is_cuda and out_nsamples.is_contiguous() and out_nsamples.element_size() == 4 \
        and out_nsamples.numel() == n * H * W
    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().omerf_render_static(h.ptr, cams.ctypes.data, n, W, H, out_rgb.data_ptr(), out_nsamples.data_ptr(),
                                              st.cuda_stream), "omerf_render_static")
    return out_rgb, out_nsamples


def render_host(h: SceneHandle, cameras, W: int, H: int, out_rgb=None, out_nsamples=None, stream=None):
    """omerf_render_host: HOST outputs (numpy arrays or pinned CPU torch tensors); synchronous."""
    import torch
    cams = _cams(cameras)
    n = cams.shape[0]
    if out_rgb is None:
        out_rgb = np.empty((n, H, W, 3), dtype=np.float32)
    if out_nsamples is None:
        out_nsamples = np.empty((n, H, W), dtype=np.uint32)

    def hptr(a, nbytes):
        if isinstance(a, np.ndarray):
            assert a.flags["C_CONTIGUOUS"] and a.nbytes == nbytes
            return a.ctypes.data
        assert (not a.is_cuda) and a.is_contiguous() and a.numel() * a.element_size() == nbytes
        return a.data_ptr()

    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().omerf_render_host(h.ptr, cams.ctypes.data, n, W, H, hptr(out_rgb, n * H * W * 12),
                                            hptr(out_nsamples, n * H * W * 4), st.cuda_stream), "omerf_render_host")
    return out_rgb, out_nsamples


def render_host_async(h: SceneHandle, cameras, W: int, H: int, out_rgb, out_nsamples, stream=None):
    """omerf_render_host_async: enqueue a render whose HOST outputs (pinned CPU torch tensors, or numpy arrays over
    pinned memory) are delivered in the background; they belong to the library until wait(h) returns."""
    import torch
    cams = _cams(cameras)
    n = cams.shape[0]

    def hptr(a, nbytes):
        if isinstance(a, np.ndarray):
            assert a.flags["C_CONTIGUOUS"] and a.nbytes == nbytes
            return a.ctypes.data
        assert (not a.is_cuda) and a.is_contiguous() and a.numel() * a.element_size() == nbytes
        return a.data_ptr()

    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().omerf_render_host_async(h.ptr, cams.ctypes.data, n, W, H, hptr(out_rgb, n * H * W * 12),
                                                  hptr(out_nsamples, n * H * W * 4), st.cuda_stream), "omerf_render_host_async")


def wait(h: SceneHandle):
    """omerf_wait: block until every render_host_async call on this scene has delivered its host buffers."""
    _check(load_library().omerf_wait(h.ptr), "omerf_wait")


def gather_probe(h: SceneHandle, camera, W: int, H: int, repeats: int = 10, flush_l2: bool = True) -> dict:
    """omerf_gather_probe: gather-only replay of one frame's samples (calibration of the gather ceiling)."""
    cams = _cams(camera)
    res = GatherProbeResult()
    _check(load_library().omerf_gather_probe(h.ptr, cams.ctypes.data, W, H, repeats, int(flush_l2), C.byref(res)),
           "omerf_gather_probe")
    return {"samples": int(res.samples), "ms_frame_order": float(res.ms_frame_order),
            "ms_scattered": float(res.ms_scattered)}


def mlp_smoothness(h: SceneHandle, F, dirs, delta, out_loss=None, out_G=None, want_G: bool = False, stream=None):
    """omerf_mlp_smoothness (Eq. 9-10 forward): DEVICE float32 tensors F [n][7], dirs [n][3], delta [n][S][3].
    Returns out_loss [n] (and out_G [n][S+1][3] if want_G); asynchronous on `stream`."""
    import torch
    n, S = int(delta.shape[0]), int(delta.shape[1])
    for a, shp in ((F, (n, 7)), (dirs, (n, 3)), (delta, (n, S, 3))):
        assert a.is_cuda and a.dtype == torch.float32 and a.is_contiguous() and tuple(a.shape) == shp
    if out_loss is None:
        out_loss = torch.empty(n, dtype=torch.float32, device="cuda")
    if want_G and out_G is None:
        out_G = torch.empty((n, S + 1, 3), dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().omerf_mlp_smoothness(h.ptr, n, S, F.data_ptr(), dirs.data_ptr(), delta.data_ptr(),
                                               out_loss.data_ptr(), out_G.data_ptr() if out_G is not None else None,
                                               st.cuda_stream), "omerf_mlp_smoothness")
    return (out_loss, out_G) if want_G else out_loss


def heatmap(nsamples, n_max: int, out=None, stream=None):
    """omerf_heatmap: DEVICE sample counts (int32-viewed uint32 tensor) -> uint8 [..., 3] colour ramp; asynchronous."""
    import torch
    assert nsamples.is_cuda and nsamples.is_contiguous() and nsamples.element_size() == 4
    if out is None:
        out = torch.empty((*nsamples.shape, 3), dtype=torch.uint8, device="cuda")
    assert out.is_cuda and out.is_contiguous() and out.dtype == torch.uint8 and out.numel() == nsamples.numel() * 3
    st = torch.cuda.current_stream() if stream is None else stream
    _check(load_library().omerf_heatmap(nsamples.data_ptr(), nsamples.numel(), n_max, out.data_ptr(), st.cuda_stream),
           "omerf_heatmap")
    return out


def last_launch_count(h: SceneHandle) -> int:
    return int(load_library().omerf_last_launch_count(h.ptr))


def scene_info(h: SceneHandle) -> dict:
    info = SceneInfo()
    _check(load_library().omerf_scene_get_info(h.ptr, C.byref(info)), "omerf_scene_get_info")
    return {"device_bytes": int(info.device_bytes), "pyramid_levels": int(info.pyramid_levels),
            "sampler": int(info.sampler), "occ_bits_set": int(info.occ_bits_set), "grid_bytes": int(info.grid_bytes),
            "grid_blocks_total": int(info.grid_blocks_total), "grid_blocks_allocated": int(info.grid_blocks_allocated),
            "plane_bytes": int(info.plane_bytes), "xz_band": tuple(info.xz_band), "yz_band": tuple(info.yz_band)}


def pyramid_level(h: SceneHandle, level: int):
    L = load_library()
    nx, ny = C.c_int32(), C.c_int32()
    _check(L.omerf_scene_get_pyramid_level(h.ptr, level, C.byref(nx), C.byref(ny), None, None), "get_pyramid_level")
    mn = np.empty((nx.value, ny.value), dtype=np.float32)
    mx = np.empty_like(mn)
    _check(L.omerf_scene_get_pyramid_level(h.ptr, level, C.byref(nx), C.byref(ny), mn.ctypes.data, mx.ctypes.data),
           "get_pyramid_level")
    return mn, mx


def block_table(h: SceneHandle) -> np.ndarray:
    """omerf_scene_get_block_table: flat int32 block table of the sparse-block grid (C order of bx,by,bz)."""
    n = scene_info(h)["grid_blocks_total"]
    out = np.empty(n, dtype=np.int32)
    _check(load_library().omerf_scene_get_block_table(h.ptr, out.ctypes.data, n), "get_block_table")
    return out


def bitfield(h: SceneHandle, occ_n) -> np.ndarray:
    n = (int(np.prod(occ_n)) + 31) // 32
    out = np.empty(n, dtype=np.uint32)
    _check(load_library().omerf_scene_get_bitfield(h.ptr, out.ctypes.data, n), "get_bitfield")
    return out
