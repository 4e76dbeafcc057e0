"""ctypes binding of the CPU oracle (oracle/omerf_oracle.c).

TEST INFRASTRUCTURE — only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package.  The product package
(paper_2404_09531_b200) never imports it and it never imports the product.
Inputs come from `synth` (seeded generators, no method arithmetic).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_f32p = C.POINTER(C.c_float)
_u8p = C.POINTER(C.c_uint8)
_u32p = C.POINTER(C.c_uint32)


class _Scene(C.Structure):
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
        ("sampler", C.c_int32), ("occ_n", C.c_int32 * 3), ("occ_bits", _u32p),
        ("soft_eps", C.c_float),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        L.orc_soft_mask.restype = C.c_double
        L.orc_exp_q.restype = C.c_float
        L.orc_exp_q.argtypes = [C.c_float]
        L.orc_q_stop.restype = C.c_uint32
        L.orc_q_stop.argtypes = [C.c_float]
        L.orc_lattice_K.restype = C.c_int64
        L.orc_pixel_samples.restype = C.c_int64
        L.orc_render.restype = C.c_int
        L.orc_render_pixels.restype = C.c_int
        _lib = L
    return _lib


def _ptr(a, t):
    return a.ctypes.data_as(t)


def exp_q(x) -> np.ndarray:
    x = np.atleast_1d(np.asarray(x, dtype=np.float32))
    L = lib()
    return np.array([L.orc_exp_q(C.c_float(float(v))) for v in x], dtype=np.float32)


def q_stop(t_stop: float) -> int:
    return int(lib().orc_q_stop(C.c_float(t_stop)))


class OracleScene:
    """Holds a synth.Scene (keeps the numpy arrays alive) and its C view."""

    def __init__(self, scene, sampler: int = 0, soft_eps: float = 0.0):
        self.scene = scene
        s = _Scene()
        self._keep = []

        def arr(a, dt):
            a = np.ascontiguousarray(a, dtype=dt)
            self._keep.append(a)
            return a

        s.box[:] = scene.box
        h_lo, h_up = arr(scene.h_lo, np.float32), arr(scene.h_up, np.float32)
        s.hf_n[:] = h_lo.shape
        s.h_lo, s.h_up = _ptr(h_lo, _f32p), _ptr(h_up, _f32p)
        g = arr(scene.grid, np.uint8)
        s.grid_n[:] = g.shape[:3]
        s.grid = _ptr(g, _u8p)
        for nm in ("xy", "xz", "yz"):
            p = arr(getattr(scene, "plane_" + nm), np.uint8)
            getattr(s, nm + "_n")[:] = p.shape[:2]
            setattr(s, "plane_" + nm, _ptr(p, _u8p))
        s.deq_scale, s.deq_bias = scene.deq_scale, scene.deq_bias
        W0 = arr(scene.W0, np.float32)
        s.mlp_in, s.mlp_hidden = W0.shape[1], W0.shape[0]
        for nm in ("W0", "b0", "W1", "b1", "W2", "b2"):
            setattr(s, nm, _ptr(arr(getattr(scene, nm), np.float32), _f32p))
        s.step, s.t_stop = scene.step, scene.t_stop
        s.bg[:] = scene.bg
        s.sampler = sampler
        s.soft_eps = soft_eps
        s.occ_n[:] = scene.occ_n
        self.c = s
        self.bits = None
        if sampler == 1:
            n = int(np.prod(scene.occ_n))
            assert n > 0, "sampler 1 needs occ_n"
            self.bits = np.zeros((n + 31) // 32, dtype=np.uint32)
            lib().orc_build_bitfield(C.byref(s), _ptr(self.bits, _u32p))
            s.occ_bits = _ptr(self.bits, _u32p)

    # ---- small pieces, for the pins -------------------------------------------------
    def ray(self, cam_row, u, v):
        cam = np.ascontiguousarray(cam_row, dtype=np.float32)
        d = np.zeros(3, dtype=np.float32)
        lib().orc_ray(_ptr(cam, _f32p), C.c_int(u), C.c_int(v), _ptr(d, _f32p))
        return d

    def features(self, p):
        p = np.ascontiguousarray(p, dtype=np.float32)
        I = np.zeros(8, dtype=np.int32)
        t = np.zeros(8, dtype=np.float32)
        lib().orc_features(C.byref(self.c), _ptr(p, _f32p), _ptr(I, C.POINTER(C.c_int32)), _ptr(t, _f32p))
        return I, t

    def grid_lookup(self, p):
        p = np.ascontiguousarray(p, dtype=np.float32)
        out = np.zeros(8, dtype=np.uint32)
        lib().orc_grid_lookup(self.c.grid, self.c.grid_n, self.c.box, _ptr(p, _f32p), _ptr(out, _u32p))
        return out

    def plane_lookup(self, which, pa, pb):
        s = self.c
        tex = getattr(s, "plane_" + which)
        n = getattr(s, which + "_n")
        ax = {"xy": (0, 1), "xz": (0, 2), "yz": (1, 2)}[which]
        out = np.zeros(8, dtype=np.uint32)
        lib().orc_plane_lookup(tex, C.c_int(n[0]), C.c_int(n[1]), C.c_float(s.box[ax[0]]),
                               C.c_float(s.box[ax[1]]), C.c_float(pa), C.c_float(pb), _ptr(out, _u32p))
        return out

    def occupied(self, p) -> bool:
        p = np.ascontiguousarray(p, dtype=np.float32)
        f = lib().orc_occupied_plane if self.c.sampler == 0 else lib().orc_occupied_grid
        return bool(f(C.byref(self.c), _ptr(p, _f32p)))

    def soft_mask(self, p) -> float:
        p = np.ascontiguousarray(p, dtype=np.float32)
        return float(lib().orc_soft_mask(C.byref(self.c), _ptr(p, _f32p)))

    def mlp(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        out = np.zeros(3, dtype=np.float64)
        lib().orc_mlp(C.byref(self.c), _ptr(x, C.POINTER(C.c_double)), _ptr(out, C.POINTER(C.c_double)))
        return out

    def encode_dir(self, d):
        d = np.ascontiguousarray(d, dtype=np.float32)
        out = np.zeros(27, dtype=np.float64)
        lib().orc_encode_dir(_ptr(d, _f32p), _ptr(out, C.POINTER(C.c_double)))
        return out

    def lattice_K(self, cam_row) -> int:
        cam = np.ascontiguousarray(cam_row, dtype=np.float32)
        return int(lib().orc_lattice_K(C.byref(self.c), _ptr(cam, _f32p)))

    def pixel_samples(self, cam_row, u, v, cap=4096):
        cam = np.ascontiguousarray(cam_row, dtype=np.float32)
        ks = np.zeros(cap, dtype=np.int64)
        pos = np.zeros((cap, 3), dtype=np.float32)
        n = int(lib().orc_pixel_samples(C.byref(self.c), _ptr(cam, _f32p), C.c_int(u), C.c_int(v),
                                        C.c_int64(cap), _ptr(ks, C.POINTER(C.c_int64)), _ptr(pos, _f32p)))
        m = min(n, cap)
        return n, ks[:m], pos[:m]

    # ---- rendering ------------------------------------------------------------------
    def render(self, cams, W, H, mode="clipped", rows=None, aux=False, stats=False):
        """Returns dict(rgb float64 [n][H][W][3], nsamples uint32 [n][H][W], threads, ...)."""
        cams = np.ascontiguousarray(np.atleast_2d(cams), dtype=np.float32)
        n = cams.shape[0]
        v0, v1 = (0, H) if rows is None else rows
        rgb = np.zeros((n, H, W, 3), dtype=np.float64)
        ns = np.zeros((n, H, W), dtype=np.uint32)
        ax = np.zeros((n, H, W, 3), dtype=np.float64) if aux else None
        tot = np.zeros(n, dtype=np.uint64)
        hist = np.zeros(64, dtype=np.uint64)
        thr = lib().orc_render(C.byref(self.c), _ptr(cams, _f32p), C.c_int(n), C.c_int(W), C.c_int(H),
                               C.c_int(v0), C.c_int(v1), C.c_int({"brute": 0, "clipped": 1}[mode]),
                               _ptr(rgb, C.POINTER(C.c_double)), _ptr(ns, _u32p),
                               _ptr(ax, C.POINTER(C.c_double)) if aux else None,
                               _ptr(tot, C.POINTER(C.c_uint64)), _ptr(hist, C.POINTER(C.c_uint64)))
        out = {"rgb": rgb, "nsamples": ns, "threads": int(thr), "view_total": tot, "hist": hist}
        if aux:
            out["T_end"], out["sum_w"], out["Q"] = ax[..., 0], ax[..., 1], ax[..., 2]
        return out

    def render_pixels(self, cams, W, H, vuv, mode="clipped", aux=False):
        cams = np.ascontiguousarray(np.atleast_2d(cams), dtype=np.float32)
        vuv = np.ascontiguousarray(vuv, dtype=np.int32).reshape(-1, 3)
        m = vuv.shape[0]
        rgb = np.zeros((m, 3), dtype=np.float64)
        ns = np.zeros(m, dtype=np.uint32)
        ax = np.zeros((m, 3), dtype=np.float64) if aux else None
        rc = lib().orc_render_pixels(C.byref(self.c), _ptr(cams, _f32p), C.c_int(cams.shape[0]),
                                     C.c_int(W), C.c_int(H), C.c_int({"brute": 0, "clipped": 1}[mode]),
                                     C.c_int64(m), _ptr(vuv, C.POINTER(C.c_int32)),
                                     _ptr(rgb, C.POINTER(C.c_double)), _ptr(ns, _u32p),
                                     _ptr(ax, C.POINTER(C.c_double)) if aux else None)
        if rc != 0:
            raise ValueError("pixel outside the image")
        out = {"rgb": rgb, "nsamples": ns}
        if aux:
            out["T_end"], out["sum_w"], out["Q"] = ax[:, 0], ax[:, 1], ax[:, 2]
        return out


# ---- sparse-block grid ----------------------------------------------------
class SparseBlocks:
    """Oracle-side bake of the sparse-block grid from the occupancy plane (omerf_oracle.c, R24)."""

    def __init__(self, O: OracleScene, B: int = 8, atlas: bool = True):
        L = lib()
        L.orc_sparse_mark_blocks.restype = C.c_int64
        L.orc_sparse_grid_lookup.restype = C.c_int
        self.O, self.B = O, B
        G = tuple(int(x) for x in O.c.grid_n)
        self.nb = tuple((g + B - 1) // B for g in G)
        self.mark = np.zeros(self.nb, dtype=np.uint8)
        self.n_alloc = int(L.orc_sparse_mark_blocks(C.byref(O.c), C.c_int(B), _ptr(self.mark, _u8p)))
        self.table = np.zeros(self.nb, dtype=np.int32)
        self.atlas = np.zeros((self.n_alloc, B, B, B, 8), dtype=np.uint8) if atlas else None
        L.orc_sparse_build(C.byref(O.c), C.c_int(B), _ptr(self.mark, _u8p), _ptr(self.table, C.POINTER(C.c_int32)),
                           _ptr(self.atlas, _u8p) if atlas else None)

    def need_mask(self) -> np.ndarray:
        G = tuple(int(x) for x in self.O.c.grid_n)
        need = np.zeros(G, dtype=np.uint8)
        lib().orc_sparse_need_mask(C.byref(self.O.c), _ptr(need, _u8p))
        return need

    def lookup(self, p):
        p = np.ascontiguousarray(p, dtype=np.float32)
        out = np.zeros(8, dtype=np.uint32)
        rc = lib().orc_sparse_grid_lookup(_ptr(self.table, C.POINTER(C.c_int32)), _ptr(self.atlas, _u8p), C.c_int(self.B),
                                          self.O.c.grid_n, self.O.c.box, _ptr(p, _f32p), _ptr(out, _u32p))
        return rc, out


def grid_corners(O: OracleScene, p) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float32)
    c = np.zeros(6, dtype=np.int32)
    lib().orc_grid_corners(O.c.grid_n, O.c.box, _ptr(p, _f32p), _ptr(c, C.POINTER(C.c_int32)))
    return c


def mlp_smoothness(O: OracleScene, F, d, delta, want_G: bool = False):
    """Eq. 9-10 forward: per-direction loss terms, and optionally G for every (direction, perturbation)."""
    F = np.ascontiguousarray(F, dtype=np.float32)
    d = np.ascontiguousarray(d, dtype=np.float32)
    delta = np.ascontiguousarray(delta, dtype=np.float32)
    n, S = delta.shape[0], delta.shape[1]
    assert F.shape == (n, 7) and d.shape == (n, 3) and delta.shape == (n, S, 3)
    loss = np.zeros(n, dtype=np.float64)
    G = np.zeros((n, S + 1, 3), dtype=np.float64) if want_G else None
    lib().orc_mlp_smoothness(C.byref(O.c), C.c_int64(n), C.c_int(S), _ptr(F, _f32p), _ptr(d, _f32p), _ptr(delta, _f32p),
                             _ptr(loss, C.POINTER(C.c_double)), _ptr(G, C.POINTER(C.c_double)) if want_G else None)
    return (loss, G) if want_G else loss


class SectorMaps:
    """Distinct 32-byte sectors touched per feature source by the renders run inside the `with` block (SURVEY 8(d):
    the compulsory-byte figure of the HBM roofline)."""

    def __init__(self, O: OracleScene):
        sc = O.scene
        self.texels = [int(np.prod(a.shape[:-1])) for a in (sc.grid, sc.plane_xy, sc.plane_xz, sc.plane_yz)]
        self.maps = [np.zeros(((t + 3) // 4 + 7) // 8, dtype=np.uint8) for t in self.texels]

    def __enter__(self):
        lib().orc_set_sector_maps(*[_ptr(m, _u8p) for m in self.maps])
        return self

    def __exit__(self, *exc):
        lib().orc_set_sector_maps(None, None, None, None)

    def sectors(self):
        return dict(zip(("grid", "xy", "xz", "yz"), (int(np.unpackbits(m).sum()) for m in self.maps)))

    def compulsory_bytes(self) -> int:
        return 32 * sum(self.sectors().values())


def heatmap(nsamples, n_max: int) -> np.ndarray:
    """Sample-count visualisation (Fig. 1; R26), exact integers:
    v = min(n, n_max) * 255 // n_max, rgb = (v, 255 - |2 v - 255|, 255 - v)."""
    n = np.minimum(np.asarray(nsamples, dtype=np.int64), n_max)
    v = n * 255 // n_max
    return np.stack([v, 255 - np.abs(2 * v - 255), 255 - v], axis=-1).astype(np.uint8)


class LowZBand:
    """Oracle-side low-z bake of the xz / yz planes from the occupancy plane (omerf_oracle.c, R27;
    PAPER.md:186).  which in {"xz", "yz"}."""

    def __init__(self, O: OracleScene, which: str, crop: bool = True):
        assert which in ("xz", "yz")
        self.O, self.which = O, which
        n = getattr(O.c, which + "_n")
        self.Na, self.Nb = int(n[0]), int(n[1])
        lo, hi = C.c_int(), C.c_int()
        self.rows = int(lib().orc_lowz_band(C.byref(O.c), C.c_int(self.Nb), C.byref(lo), C.byref(hi)))
        self.b_lo, self.b_hi = lo.value, hi.value
        self.band = None
        if crop:
            self.band = np.zeros((self.Na, self.rows, 8), dtype=np.uint8)
            lib().orc_lowz_crop(getattr(O.c, "plane_" + which), C.c_int(self.Na), C.c_int(self.Nb), lo, hi,
                                _ptr(self.band, _u8p))

    def lookup(self, pa: float, pz: float):
        Xa = self.O.c.box[0 if self.which == "xz" else 1]
        out = np.zeros(8, dtype=np.uint32)
        rc = lib().orc_plane_lookup_band(_ptr(self.band, _u8p), C.c_int(self.Na), C.c_int(self.Nb), C.c_int(self.b_lo),
                                         C.c_int(self.b_hi), C.c_float(Xa), C.c_float(self.O.c.box[2]), C.c_float(pa),
                                         C.c_float(pz), _ptr(out, _u32p))
        return int(rc), out
