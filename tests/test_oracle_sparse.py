"""Pins of the oracle's sparse-block grid bake (R24), -m "not gpu".

The bake rule is pinned against what it is for - the set of voxels the renderer's trilinear lookup can touch -
by brute force over points of the slab, and against closed forms for flat slabs."""
import math

import numpy as np
import pytest
from scipy.ndimage import binary_dilation

import oracle
import synth


def _random_scene(seed, hf=13, grid_n=(20, 18, 12), box=(10.0, 9.0, 6.0), empty_frac=0.15):
    rng = np.random.default_rng(seed)
    lo = (0.5 + 2.0 * rng.random((hf, hf))).astype(np.float32)
    hi = (lo + 0.05 + 2.5 * rng.random((hf, hf))).astype(np.float32)
    kill = rng.random((hf, hf)) < empty_frac
    hi[kill] = lo[kill] - 1.0                                   # empty columns (R17)
    return synth.custom_scene(box=box, hf_n=(hf, hf), h_lo=lo, h_up=hi, grid_n=grid_n, seed=seed, smooth=False)


def _slab_points(O, sc, rng, n):
    p = (rng.random((n, 3)) * np.array(sc.box)).astype(np.float32)
    p = p[np.all(p < np.array(sc.box, dtype=np.float32), axis=1)]
    return [q for q in p if O.occupied(q)]


@pytest.mark.parametrize("seed,B", [(1, 4), (2, 8), (3, 2)])
def test_every_corner_the_lookup_touches_is_needed_and_allocated(seed, B):
    """Soundness by brute force: random points that pass the per-sample predicate (Eq. 7, fp32) only ever touch
    needed voxels, the sparse lookup never hits an unallocated block and returns the dense lookup's integers."""
    sc = _random_scene(seed)
    O = oracle.OracleScene(sc)
    S = oracle.SparseBlocks(O, B)
    need = S.need_mask()
    pts = _slab_points(O, sc, np.random.default_rng(100 + seed), 12000)
    assert len(pts) > 1200
    for p in pts:
        c = oracle.grid_corners(O, p)
        for x in c[0:2]:
            for y in c[2:4]:
                for z in c[4:6]:
                    assert need[x, y, z], (p, c)
                    assert S.mark[x // B, y // B, z // B]
        rc, got = S.lookup(p)
        assert rc == 0
        assert np.array_equal(got, O.grid_lookup(p))


def test_need_mask_is_tight_on_a_tiny_scene():
    """The rule may only over-mark by its stated padding: every needed voxel is within one voxel of a voxel that a
    dense sampling of the slab really touches, and everything touched is needed."""
    sc = _random_scene(7, hf=9, grid_n=(10, 9, 8), box=(8.0, 8.0, 4.0), empty_frac=0.2)
    O = oracle.OracleScene(sc)
    need = oracle.SparseBlocks(O, 4).need_mask().astype(bool)
    touched = np.zeros_like(need)
    xs = np.linspace(0.0, 8.0, 161, dtype=np.float32)[:-1] + np.float32(0.013)
    zs = np.linspace(0.0, 4.0, 201, dtype=np.float32)[:-1] + np.float32(0.007)
    for x in xs:
        for y in xs:
            ix, iy = int(math.floor(x + 0.5)), int(math.floor(y + 0.5))
            lo, hi = sc.h_lo[ix, iy], sc.h_up[ix, iy]
            for z in zs[(zs >= lo) & (zs <= hi)]:
                p = np.array([x, y, z], dtype=np.float32)
                assert O.occupied(p)
                c = oracle.grid_corners(O, p)
                touched[c[0]:c[1] + 1, c[2]:c[3] + 1, c[4]:c[5] + 1] = True
    assert touched.sum() > 50
    assert not (touched & ~need).any()
    assert not (need & ~binary_dilation(touched, structure=np.ones((3, 3, 3), bool))).any()


@pytest.mark.parametrize("za,zb", [(1.0, 3.0), (0.0, 6.0), (2.26, 2.27)])
def test_flat_slab_closed_form(za, zb):
    """Flat slab: every (i,j) column needs the corner range [floor(za Gz/Z - 1/2 - 1/64), floor(zb Gz/Z - 1/2 + 1/64) + 1]."""
    G, Z, B = (16, 12, 24), 6.0, 4
    sc = synth.custom_scene(box=(8.0, 6.0, Z), hf_n=(9, 7), h_lo=za, h_up=zb, grid_n=G, seed=1)
    S = oracle.SparseBlocks(oracle.OracleScene(sc), B)
    k0 = max(math.floor(za * G[2] / Z - 0.5 - 1 / 64), 0)
    k1 = min(math.floor(zb * G[2] / Z - 0.5 + 1 / 64) + 1, G[2] - 1)
    need = S.need_mask()
    assert need.sum() == G[0] * G[1] * (k1 - k0 + 1)
    assert need[:, :, k0:k1 + 1].all()
    nbz = k1 // B - k0 // B + 1
    assert S.n_alloc == (G[0] // B) * (G[1] // B) * nbz
    assert S.mark[:, :, k0 // B:k1 // B + 1].all() and S.mark.sum() == S.n_alloc


def test_table_and_atlas_layout():
    """Blocks are numbered in C order of (bx,by,bz); the atlas holds the dense grid's texels, zeros past the edge."""
    sc = _random_scene(5, grid_n=(21, 18, 10))                  # 21 and 10 are not multiples of the block size
    O = oracle.OracleScene(sc)
    S = oracle.SparseBlocks(O, 4)
    flat = S.table.ravel()
    alloc = flat[flat >= 0]
    assert np.array_equal(alloc, np.arange(S.n_alloc)) and S.n_alloc == int(S.mark.sum())
    assert np.array_equal(flat >= 0, S.mark.ravel().astype(bool))
    pad = np.zeros((24, 20, 12, 8), dtype=np.uint8)
    pad[:21, :18, :10] = sc.grid
    for (bx, by, bz), bid in np.ndenumerate(S.table):
        if bid >= 0:
            assert np.array_equal(S.atlas[bid], pad[4 * bx:4 * bx + 4, 4 * by:4 * by + 4, 4 * bz:4 * bz + 4])


def test_empty_plane_allocates_nothing_and_block_count_is_monotone():
    sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=3.0, h_up=1.0, grid_n=(8, 8, 8), seed=1)
    S = oracle.SparseBlocks(oracle.OracleScene(sc), 4)
    assert S.n_alloc == 0 and (S.table == -1).all()
    # widening the slab can only add blocks; the whole box needs every block
    prev = 0
    for zb in (1.2, 2.0, 3.0, 4.0):
        sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=1.0, h_up=zb, grid_n=(8, 8, 8), seed=1)
        n = oracle.SparseBlocks(oracle.OracleScene(sc), 4).n_alloc
        assert n >= prev
        prev = n
    sc = synth.custom_scene(box=(8.0, 8.0, 4.0), hf_n=(9, 9), h_lo=0.0, h_up=4.0, grid_n=(8, 8, 8), seed=1)
    assert oracle.SparseBlocks(oracle.OracleScene(sc), 4).n_alloc == 8
