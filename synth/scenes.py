"""Seeded scene and camera generators (numpy only; no method arithmetic).

Shapes, sizes and value distributions follow BASELINE.json `configs[0..4]` and
SURVEY.md §8(d) "Synthetic inputs".  They stand in for the paper's baked
Campus-Oblique / Matrix City assets, which are not available.

Array conventions (C-contiguous, first axis slowest, channel last):
  h_lo, h_up : float32 [Mx][My]          occupancy plane P_o, vertex-centred
  grid       : uint8   [Gx][Gy][Gz][8]   low-res voxel grid V
  plane_xy   : uint8   [Ax][Ay][8]       triplane, sampled with (x, y)
  plane_xz   : uint8   [Ax][Az][8]       triplane, sampled with (x, z)
  plane_yz   : uint8   [Ay][Az][8]       triplane, sampled with (y, z)
  channel 0 = density, 1..3 = diffuse RGB, 4..7 = specular features
  W0 [16][34], W1 [16][16], W2 [3][16] float32 row-major [out][in]; biases float32
Cameras are float32 rows of CAMERA_FLOATS = 16 values:
  origin[3], right[3], up[3], fwd[3], fx, fy, cx, cy
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

CAMERA_FLOATS = 16

_CONFIG_RES = {0: (128, 128), 1: (1920, 1080), 2: (1920, 1080), 3: (3840, 2160), 4: (1920, 1080), 5: (1920, 1080)}


def config_resolution(config: int) -> tuple[int, int]:
    """(W, H) of the cameras of BASELINE.json configs[config]."""
    return _CONFIG_RES[config]


@dataclass
class Scene:
    box: tuple[float, float, float]
    h_lo: np.ndarray
    h_up: np.ndarray
    grid: np.ndarray
    plane_xy: np.ndarray
    plane_xz: np.ndarray
    plane_yz: np.ndarray
    W0: np.ndarray
    b0: np.ndarray
    W1: np.ndarray
    b1: np.ndarray
    W2: np.ndarray
    b2: np.ndarray
    step: float
    deq_scale: float = 28.0 / 255.0
    deq_bias: float = -14.0
    t_stop: float = 1e-3
    bg: tuple[float, float, float] = (1.0, 1.0, 1.0)
    occ_n: tuple[int, int, int] = (0, 0, 0)   # bitfield resolution for the config-4 comparator
    name: str = "custom"
    meta: dict = field(default_factory=dict)

    def nbytes(self) -> int:
        arrs = (self.h_lo, self.h_up, self.grid, self.plane_xy, self.plane_xz, self.plane_yz,
                self.W0, self.b0, self.W1, self.b1, self.W2, self.b2)
        return int(sum(a.nbytes for a in arrs))


# --------------------------------------------------------------------------------------
# random byte volumes: rint(box-filter(U{0..255})) over the spatial axes, edge-replicated
# --------------------------------------------------------------------------------------
def _box3_sum(a: np.ndarray, axis: int) -> np.ndarray:
    """a[i-1] + a[i] + a[i+1] along `axis` with edge replication (uint16 in, uint16 out)."""
    n = a.shape[axis]
    out = a.copy()
    sl = [slice(None)] * a.ndim

    def S(s):
        t = list(sl)
        t[axis] = s
        return tuple(t)

    out[S(slice(1, n))] += a[S(slice(0, n - 1))]
    out[S(slice(0, 1))] += a[S(slice(0, 1))]
    out[S(slice(0, n - 1))] += a[S(slice(1, n))]
    out[S(slice(n - 1, n))] += a[S(slice(n - 1, n))]
    return out


def smoothed_bytes(rng: np.random.Generator, shape: tuple[int, ...], n_spatial: int) -> np.ndarray:
    """uint8 array `shape` = rint(box3^n_spatial(U{0..255})), filter over the first
    `n_spatial` axes only (never over the channel axis), edges replicated."""
    # generate slab by slab along axis 0 to bound peak memory for the 1 GiB grid
    a = rng.integers(0, 256, size=shape, dtype=np.uint8).astype(np.uint16)
    for ax in range(n_spatial):
        a = _box3_sum(a, ax)
    div = 3 ** n_spatial
    # round-to-nearest of a/div; 2a+div is odd*... no ties occur since div is odd
    a = (2 * a.astype(np.uint32) + div) // (2 * div)
    return a.astype(np.uint8)


# --------------------------------------------------------------------------------------
# height fields
# --------------------------------------------------------------------------------------
def _value_noise(rng: np.random.Generator, m: int, base: int = 8, octaves: int = 5,
                 persistence: float = 0.5) -> np.ndarray:
    """Fractal value noise on an m x m vertex grid over the unit square, float64."""
    u = np.arange(m, dtype=np.float64) / (m - 1)
    out = np.zeros((m, m), dtype=np.float64)
    amp = 1.0
    for o in range(octaves):
        cells = base * (1 << o)
        lat = rng.random((cells + 1, cells + 1))
        x = u * cells
        i0 = np.minimum(np.floor(x).astype(np.int64), cells - 1)
        f = x - i0
        s = f * f * (3.0 - 2.0 * f)                       # smoothstep
        a = lat[i0][:, i0]
        b = lat[i0 + 1][:, i0]
        c = lat[i0][:, i0 + 1]
        d = lat[i0 + 1][:, i0 + 1]
        sx = s[:, None]
        sy = s[None, :]
        out += amp * ((a * (1 - sx) + b * sx) * (1 - sy) + (c * (1 - sx) + d * sx) * sy)
        amp *= persistence
    return out


def _terrain_and_blocks(rng, m: int, box, terrain_max: float, n_blocks: int):
    """h_lo = value noise scaled to [0, terrain_max]; h_up = h_lo + max(5, tallest covering
    block), blocks axis-aligned with sides U(10,60) m and heights U(5,60) m, clamped to Z."""
    X, Y, Z = box
    n = _value_noise(rng, m)
    n = (n - n.min()) / (n.max() - n.min())
    h_lo = n * terrain_max
    bh = np.full((m, m), 5.0, dtype=np.float64)
    cx = rng.uniform(0.0, X, n_blocks)
    cy = rng.uniform(0.0, Y, n_blocks)
    sx = rng.uniform(10.0, 60.0, n_blocks)
    sy = rng.uniform(10.0, 60.0, n_blocks)
    hh = rng.uniform(5.0, 60.0, n_blocks)
    hx = X / (m - 1)
    hy = Y / (m - 1)
    for b in range(n_blocks):
        i0 = max(int(math.ceil((cx[b] - sx[b] / 2) / hx)), 0)
        i1 = min(int(math.floor((cx[b] + sx[b] / 2) / hx)), m - 1)
        j0 = max(int(math.ceil((cy[b] - sy[b] / 2) / hy)), 0)
        j1 = min(int(math.floor((cy[b] + sy[b] / 2) / hy)), m - 1)
        if i1 >= i0 and j1 >= j0:
            np.maximum(bh[i0:i1 + 1, j0:j1 + 1], hh[b], out=bh[i0:i1 + 1, j0:j1 + 1])
    h_up = np.minimum(h_lo + bh, Z)
    return h_lo.astype(np.float32), h_up.astype(np.float32)


def _xavier_mlp(rng, n_in: int = 34, n_hidden: int = 16, n_out: int = 3, bias_amp: float = 0.0):
    def xav(o, i):
        lim = math.sqrt(6.0 / (i + o))
        return rng.uniform(-lim, lim, size=(o, i)).astype(np.float32)

    def bias(o):
        if bias_amp == 0.0:
            return np.zeros(o, dtype=np.float32)
        return rng.uniform(-bias_amp, bias_amp, size=o).astype(np.float32)

    W0 = xav(n_hidden, n_in)
    b0 = bias(n_hidden)
    W1 = xav(n_hidden, n_hidden)
    b1 = bias(n_hidden)
    W2 = xav(n_out, n_hidden)
    b2 = bias(n_out)
    return W0, b0, W1, b1, W2, b2


# --------------------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------------------
def _scene_tiny(seed: int) -> Scene:
    rng = np.random.default_rng(seed)
    box = (64.0, 64.0, 16.0)
    m = 65
    xs = np.arange(m, dtype=np.float64) * (box[0] / (m - 1))
    ys = np.arange(m, dtype=np.float64) * (box[1] / (m - 1))
    h_lo = 4.0 + 2.0 * np.sin(xs[:, None] / 8.0) * np.cos(ys[None, :] / 8.0)
    raw = h_lo + 6.0 + 2.0 * rng.random((m, m))
    p = np.pad(raw, 1, mode="edge")
    h_up = sum(p[1 + di:1 + di + m, 1 + dj:1 + dj + m] for di in (-1, 0, 1) for dj in (-1, 0, 1)) / 9.0
    grid = smoothed_bytes(rng, (64, 64, 16, 8), 3)
    pxy = smoothed_bytes(rng, (256, 256, 8), 2)
    pxz = smoothed_bytes(rng, (256, 64, 8), 2)
    pyz = smoothed_bytes(rng, (256, 64, 8), 2)
    mlp = _xavier_mlp(rng)
    return Scene(box, h_lo.astype(np.float32), h_up.astype(np.float32), grid, pxy, pxz, pyz, *mlp,
                 step=0.25, name="cfg0_tiny")


def _scene_city(seed: int, box, m, terrain_max, n_blocks, grid_n, axy, az, name, occ_n=(0, 0, 0)) -> Scene:
    rng = np.random.default_rng(seed)
    h_lo, h_up = _terrain_and_blocks(rng, m, box, terrain_max, n_blocks)
    grid = smoothed_bytes(rng, (*grid_n, 8), 3)
    pxy = smoothed_bytes(rng, (axy, axy, 8), 2)
    pxz = smoothed_bytes(rng, (axy, az, 8), 2)
    pyz = smoothed_bytes(rng, (axy, az, 8), 2)
    mlp = _xavier_mlp(rng)
    return Scene(box, h_lo, h_up, grid, pxy, pxz, pyz, *mlp, step=0.5, name=name, occ_n=occ_n)


def make_scene(config: int) -> Scene:
    """Scene of BASELINE.json configs[config]; seed = scene index (configs 2 and 4 reuse config 1's)."""
    if config == 0:
        return _scene_tiny(0)
    if config in (1, 2, 4, 5):   # 5 = SURVEY 8(f) item 4: low-altitude cameras in the config-1 scene
        return _scene_city(1, (1000.0, 1000.0, 100.0), 1025, 30.0, 2000, (512, 512, 64), 4096, 512,
                           "cfg1_1080p", occ_n=(2048, 2048, 256))
    if config == 3:
        return _scene_city(3, (4000.0, 4000.0, 200.0), 4097, 60.0, 32000, (1024, 1024, 128), 8192, 1024,
                           "cfg3_large")
    raise ValueError(f"unknown config {config}")


# --------------------------------------------------------------------------------------
# cameras (placement only: where the pinhole sits and where it looks)
# --------------------------------------------------------------------------------------
def look_at_camera(origin, target, width: int, height: int, vfov_deg: float = 60.0) -> np.ndarray:
    """One camera row: z-up look-at frame computed in float64, stored as float32.
    Square pixels, principal point at the image centre."""
    o = np.asarray(origin, dtype=np.float64)
    t = np.asarray(target, dtype=np.float64)
    fwd = t - o
    fwd /= np.linalg.norm(fwd)
    zup = np.array([0.0, 0.0, 1.0])
    right = np.cross(fwd, zup)
    nr = np.linalg.norm(right)
    if nr < 1e-12:                      # looking straight down/up: pick +x as right
        right = np.array([1.0, 0.0, 0.0])
    else:
        right /= nr
    up = np.cross(right, fwd)
    fy = (height / 2.0) / math.tan(math.radians(vfov_deg) / 2.0)
    row = np.concatenate([o, right, up, fwd, [fy, fy, width / 2.0, height / 2.0]])
    return row.astype(np.float32)


def _orbit_camera(target, pitch_deg, yaw_deg, z, width, height):
    """Camera at height z on the ray leaving `target` at elevation `pitch`; yaw 0 looks along +y."""
    tz = target[2]
    dist = (z - tz) / math.tan(math.radians(pitch_deg))
    yaw = math.radians(yaw_deg)
    look = np.array([math.sin(yaw), math.cos(yaw)])        # horizontal look direction
    o = np.array([target[0] - dist * look[0], target[1] - dist * look[1], z])
    return look_at_camera(o, target, width, height)


def make_cameras(config: int) -> np.ndarray:
    """float32 [n_views][16] cameras of configs[config]; seed = 1000 + config."""
    rng = np.random.default_rng(1000 + config)
    W, H = config_resolution(config)
    if config == 0:
        return _orbit_camera((32.0, 32.0, 8.0), 45.0, 0.0, 40.0, W, H)[None, :]
    if config in (1, 4):
        return _orbit_camera((500.0, 500.0, 50.0), 45.0, 0.0, 300.0, W, H)[None, :]
    if config == 2:
        yaw = rng.uniform(0.0, 360.0, 16)
        z = rng.uniform(150.0, 500.0, 16)
        return np.stack([_orbit_camera((500.0, 500.0, 50.0), 20.0 + 4.0 * i, yaw[i], z[i], W, H)
                         for i in range(16)])
    if config == 3:
        yaw = rng.uniform(0.0, 360.0, 8)
        z = rng.uniform(400.0, 800.0, 8)
        pitch = np.linspace(30.0, 60.0, 8)
        return np.stack([_orbit_camera((2000.0, 2000.0, 100.0), pitch[i], yaw[i], z[i], W, H)
                         for i in range(8)])
    if config == 5:
        return low_altitude_cameras(make_scene(1), 4, rng, W, H)
    raise ValueError(f"unknown config {config}")


def low_altitude_cameras(scene: Scene, n: int, rng, W: int, H: int) -> np.ndarray:
    """SURVEY 8(f) item 4 / PAPER.md:226-234 (Table 3, low-altitude column): cameras INSIDE the box.
    Even views stand in a street (a column without a block, 8 m above the upper height field) and look
    10 degrees below the horizon; odd views sit inside the slab itself (mid-height of a column with a
    block), so the first lattice samples of most rays are already occupied."""
    X, Y, _ = scene.box
    mx, my = scene.h_lo.shape
    thick = (scene.h_up - scene.h_lo).astype(np.float64)
    cams = []
    for i in range(n):
        want_block = bool(i & 1)
        while True:
            ix, iy = int(rng.integers(mx // 5, 4 * mx // 5)), int(rng.integers(my // 5, 4 * my // 5))
            if (thick[ix, iy] > 15.0) == want_block:
                break
        x, y = ix * X / (mx - 1), iy * Y / (my - 1)
        z = (0.5 * (float(scene.h_lo[ix, iy]) + float(scene.h_up[ix, iy])) if want_block
             else float(scene.h_up[ix, iy]) + 8.0)
        yaw = float(rng.uniform(0.0, 2.0 * math.pi))
        pitch = math.radians(10.0)
        tgt = (x + 100.0 * math.sin(yaw) * math.cos(pitch), y + 100.0 * math.cos(yaw) * math.cos(pitch),
               z - 100.0 * math.sin(pitch))
        cams.append(look_at_camera((x, y, z), tgt, W, H))
    return np.stack(cams)


def orbit_cameras(config: int, n: int) -> np.ndarray:
    """n cameras of config 1's kind on a yaw orbit (bench regime 'orbit': a new view every frame)."""
    W, H = config_resolution(config)
    if config == 3:
        tgt, pitch, z = (2000.0, 2000.0, 100.0), 45.0, 600.0
    elif config == 0:
        tgt, pitch, z = (32.0, 32.0, 8.0), 45.0, 40.0
    else:
        tgt, pitch, z = (500.0, 500.0, 50.0), 45.0, 300.0
    return np.stack([_orbit_camera(tgt, pitch, 360.0 * i / n, z, W, H) for i in range(n)])


# --------------------------------------------------------------------------------------
# small hand-built scenes for unit tests (closed forms, edge cases)
# --------------------------------------------------------------------------------------
def custom_scene(*, box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=1.0, h_up=3.0, grid_n=(4, 4, 2),
                 xy_n=(16, 16), xz_n=(16, 8), yz_n=(16, 8), fill=None, seed=0, step=0.25,
                 bias_amp=0.0, t_stop=1e-3, bg=(1.0, 1.0, 1.0), smooth=True, occ_n=(0, 0, 0)) -> Scene:
    """Scene with chosen shapes.  h_lo / h_up: scalar (flat field) or an array.
    fill: None -> seeded random bytes (box-filtered if `smooth`), int -> every texel byte = fill,
    or a length-8 sequence -> per-channel constant byte."""
    rng = np.random.default_rng(seed)

    def hf(v):
        if np.isscalar(v):
            return np.full(hf_n, v, dtype=np.float32)
        v = np.asarray(v, dtype=np.float32)
        assert v.shape == tuple(hf_n)
        return np.ascontiguousarray(v)

    def tex(shape, nsp):
        if fill is None:
            if smooth:
                return smoothed_bytes(rng, (*shape, 8), nsp)
            return rng.integers(0, 256, size=(*shape, 8), dtype=np.uint8)
        a = np.empty((*shape, 8), dtype=np.uint8)
        a[...] = np.asarray(fill, dtype=np.uint8)
        return a

    mlp = _xavier_mlp(rng, bias_amp=bias_amp)
    return Scene(tuple(float(b) for b in box), hf(h_lo), hf(h_up), tex(grid_n, 3), tex(xy_n, 2),
                 tex(xz_n, 2), tex(yz_n, 2), *mlp, step=step, t_stop=t_stop, bg=tuple(bg),
                 occ_n=tuple(occ_n), name="custom")


# --------------------------------------------------------------------------------------
# inputs of the view-direction smoothness workload (Eq. 9-10) - random draws only
# --------------------------------------------------------------------------------------
def smoothness_batch(seed: int, n: int, S: int, sigma: float = 0.05):
    """F float32 [n][7] ~ U(0,1) (accumulated colour / feature sums of Eq. 4 lie in [0,1]), unit directions d [n][3]
    on the lower hemisphere (cameras look down), and the Gaussian perturbations delta [n][S][3] ~ N(0, sigma^2 I)
    of Eq. 9.  The method's arithmetic (encoding, MLP, cosine, loss) is NOT here."""
    rng = np.random.default_rng(seed)
    F = rng.random((n, 7), dtype=np.float32)
    g = rng.standard_normal((n, 3))
    g[:, 2] = -np.abs(g[:, 2])
    d = (g / np.linalg.norm(g, axis=1, keepdims=True)).astype(np.float32)
    delta = (sigma * rng.standard_normal((n, S, 3))).astype(np.float32)
    return F, d, delta
