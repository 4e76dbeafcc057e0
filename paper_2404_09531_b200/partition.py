"""Host-side partition of one batch of views across GPUs (PAPER.md:273 names divide-and-conquer as the
scaling route, "consistent rendering speeds across scales").

Pixels and views are independent and the scene is read-only, so the scene is REPLICATED on every GPU and the batch is
split with no exchange on the data path: by whole views (greedy longest-first) when there are at least as many views
as ranks, else by contiguous bands of 8x4-pixel tile rows (what `omerf_render_tiles` takes).  Work is balanced by
SAMPLES, not pixels (sky rows are nearly free): the cost of a tile row or a view is its sample count of the previous
frame (or of a counts-only pre-pass) plus a fixed cost per pixel.  Only index arithmetic lives here; all rendering is
`omerf_render_tiles` / `omerf_render`.
"""
from __future__ import annotations

import numpy as np

TILE_W, TILE_H = 8, 4            # the march kernel's tile (csrc/omerf_render.cu)
PIXEL_COST = 7.0                 # fixed work per pixel (ray setup, traversal, MLP) in units of one sample's work


def tile_grid(W: int, H: int) -> tuple[int, int]:
    return (W + TILE_W - 1) // TILE_W, (H + TILE_H - 1) // TILE_H


def tile_row_costs(nsamples: np.ndarray, pixel_cost: float = PIXEL_COST) -> np.ndarray:
    """Cost of every flattened tile row (view-major, n_views * tiles_y entries) from per-pixel sample counts
    [n_views][H][W] of the previous frame."""
    n = np.asarray(nsamples)
    n_views, H, W = n.shape
    _, tiles_y = tile_grid(W, H)
    per_row = n.reshape(n_views, H, W).sum(axis=2, dtype=np.int64).astype(np.float64) + pixel_cost * W
    pad = tiles_y * TILE_H - H
    if pad:
        per_row = np.concatenate([per_row, np.zeros((n_views, pad))], axis=1)
    return per_row.reshape(n_views, tiles_y, TILE_H).sum(axis=2).reshape(-1)


def view_costs(nsamples: np.ndarray, pixel_cost: float = PIXEL_COST) -> np.ndarray:
    n = np.asarray(nsamples)
    return n.reshape(n.shape[0], -1).sum(axis=1, dtype=np.int64).astype(np.float64) + pixel_cost * n.shape[1] * n.shape[2]


def split_rows(costs: np.ndarray, world: int) -> np.ndarray:
    """Boundaries b[0..world] (b[0] = 0, b[world] = len(costs)) of `world` contiguous bands of tile rows whose largest
    cost is minimal (binary search over the bottleneck, greedy feasibility check: exact for contiguous partitions)."""
    c = np.asarray(costs, dtype=np.float64)
    n = len(c)
    assert world >= 1 and np.all(c >= 0)
    pre = np.concatenate([[0.0], np.cumsum(c)])

    def cuts(limit):
        b, at = [0], 0
        for _ in range(world):
            # the furthest end with cost(at .. end) <= limit; limit >= max(c), so a band takes at least one row
            end = int(np.searchsorted(pre, pre[at] + limit * (1 + 1e-12), side="right")) - 1
            at = min(max(end, at), n)
            b.append(at)
        return b

    lo, hi = float(c.max()) if n else 0.0, float(pre[-1])
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if cuts(mid)[-1] >= n:
            hi = mid
        else:
            lo = mid
    b = cuts(hi)
    b[-1] = n
    return np.asarray(b, dtype=np.int64)


def assign_views(costs: np.ndarray, world: int) -> list[list[int]]:
    """Greedy longest-first: views in decreasing cost, each to the least loaded rank.  Every view goes to exactly one rank."""
    c = np.asarray(costs, dtype=np.float64)
    load = np.zeros(world)
    out: list[list[int]] = [[] for _ in range(world)]
    for v in np.argsort(-c, kind="stable"):
        r = int(np.argmin(load))
        out[r].append(int(v))
        load[r] += c[v]
    return [sorted(x) for x in out]


def imbalance(loads) -> float:
    """max / mean - 1 of the per-rank loads (0 = perfectly balanced)."""
    l = np.asarray(loads, dtype=np.float64)
    return float(l.max() / l.mean() - 1.0) if l.sum() > 0 else 0.0


class Plan:
    """What one rank renders.  mode "views": `views` (indices into the batch, rendered as a smaller batch);
    mode "rows": tiles [tile_first, tile_end) of the full batch = flattened tile rows [row_first, row_end)."""

    def __init__(self, mode, rank, world, **kw):
        self.mode, self.rank, self.world = mode, rank, world
        self.__dict__.update(kw)


def make_plans(nsamples_prev: np.ndarray, world: int, pixel_cost: float = PIXEL_COST) -> list[Plan]:
    """The partition of a batch [n_views][H][W] over `world` ranks, from the previous frame's sample counts."""
    n = np.asarray(nsamples_prev)
    n_views, H, W = n.shape
    tiles_x, tiles_y = tile_grid(W, H)
    if n_views >= world and n_views % world == 0 or n_views >= 2 * world:
        vc = view_costs(n, pixel_cost)
        parts = assign_views(vc, world)
        loads = [float(vc[p].sum()) for p in parts]
        samples = [int(n[p].sum(dtype=np.int64)) if p else 0 for p in parts]
        return [Plan("views", r, world, views=parts[r], cost=loads[r], samples=samples[r], imbalance=imbalance(loads),
                     sample_imbalance=imbalance(samples)) for r in range(world)]
    rc = tile_row_costs(n, pixel_cost)
    b = split_rows(rc, world)
    loads = [float(rc[b[r]:b[r + 1]].sum()) for r in range(world)]
    rows_s = tile_row_costs(n, 0.0)
    samples = [int(rows_s[b[r]:b[r + 1]].sum()) for r in range(world)]
    return [Plan("rows", r, world, row_first=int(b[r]), row_end=int(b[r + 1]), tile_first=int(b[r]) * tiles_x,
                 tile_end=int(b[r + 1]) * tiles_x, cost=loads[r], samples=samples[r], imbalance=imbalance(loads),
                 sample_imbalance=imbalance(samples)) for r in range(world)]


def pixel_row_range(plan: Plan, H: int) -> tuple[int, int]:
    """Flattened pixel rows [r0, r1) (view * H + v) that a "rows" plan covers."""
    _, tiles_y = tile_grid(1, H)

    def first(R):
        view, ty = divmod(R, tiles_y)
        return view * H + min(ty * TILE_H, H)

    return first(plan.row_first), first(plan.row_end)


def stitch(plans: list[Plan], parts: list[tuple[np.ndarray, np.ndarray]], n_views: int, H: int, W: int):
    """Assemble the full batch (rgb [n][H][W][3], nsamples [n][H][W]) from every rank's share.
    parts[r] = (rgb, nsamples): mode "views": arrays of that rank's views in `plan.views` order;
    mode "rows": the rank's flattened pixel rows [r0, r1) as [(r1 - r0)][W][...]."""
    rgb = np.zeros((n_views, H, W, 3), dtype=parts[0][0].dtype)
    ns = np.zeros((n_views, H, W), dtype=parts[0][1].dtype)
    seen = np.zeros(n_views * H, dtype=np.int32)
    for plan, (p_rgb, p_ns) in zip(plans, parts):
        if plan.mode == "views":
            for i, v in enumerate(plan.views):
                rgb[v], ns[v] = p_rgb[i], p_ns[i]
                seen[v * H:(v + 1) * H] += 1
        else:
            r0, r1 = pixel_row_range(plan, H)
            rgb.reshape(n_views * H, W, 3)[r0:r1] = p_rgb
            ns.reshape(n_views * H, W)[r0:r1] = p_ns
            seen[r0:r1] += 1
    assert np.all(seen == 1), "every pixel row must be rendered by exactly one rank"
    return rgb, ns
