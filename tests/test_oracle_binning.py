"""Pins of the oracle's tile lists (twin_index rect, orc_bin) -- CPU only.

The paper says only "sorted by depth" and "tile-based rasterizer from 3DGS"; the
rules are readings C7, C9, C10, C12, C13 of DESIGN.md.  Pinned here by brute force written as plain
inequalities in numpy (no trunc/clamp chain), by numpy's own stable sort, and by eigvalsh for the radius.
"""
import numpy as np

from oracle import gabsplat_oracle as orc
from paper_2508_05343_b200 import scenes


def _brute_lists(pr, cam):
    """For each tile, the primitives whose square [mu-r, mu+r] reaches it (reading C10 as inequalities:
    tile t spans pixels 16t..16t+15 and is hit iff mu-r < 16(t+1) and mu+r >= 16t+1), by (depth bits, id)."""
    m = pr["mean2d_f32"].astype(np.float64)
    r = pr["radius"].astype(np.float64)
    lists = []
    for ty in range(cam.tiles_y):
        for tx in range(cam.tiles_x):
            hit = (pr["visible"] > 0) & (m[:, 0] - r < 16 * (tx + 1)) & (m[:, 0] + r >= 16 * tx + 1) \
                & (m[:, 1] - r < 16 * (ty + 1)) & (m[:, 1] + r >= 16 * ty + 1)
            ids = np.nonzero(hit)[0]
            ids = ids[np.lexsort((ids, pr["depth_bits"][ids]))]
            lists.append(ids)
    return lists


def _check(s, cam):
    pr = orc.project(s, cam)
    lists = _brute_lists(pr, cam)
    counts = np.zeros(s.N, np.int64)
    for l in lists:
        counts[l] += 1
    # a primitive whose square misses every tile is culled; otherwise tiles_touched is its tile count
    assert np.array_equal(counts, pr["tiles_touched"].astype(np.int64))
    for brute in (True, False):
        b = orc.bin_sort(s, cam, brute=brute)
        assert b["num_instances"] == counts.sum()
        at = 0
        for t, l in enumerate(lists):
            assert b["tile_ranges"][t, 0] == (at if len(l) else b["tile_ranges"][t, 0]) and \
                b["tile_ranges"][t, 1] - b["tile_ranges"][t, 0] == len(l)
            seg = slice(at, at + len(l))
            assert np.array_equal(b["ids"][seg], l.astype(np.uint32))
            assert np.array_equal(b["keys"][seg], (np.uint64(t) << np.uint64(32)) | pr["depth_bits"][l].astype(np.uint64))
            at += len(l)
        assert np.all(np.diff(b["keys"].astype(np.uint64)) >= 0) or b["num_instances"] < 2
    return pr, lists


def test_tile_lists_brute_force_tiny():
    s = scenes.make_scene("tiny")
    pr, lists = _check(s, scenes.make_cameras("tiny")[0])
    assert sum(len(l) for l in lists) > 3000 and max(len(l) for l in lists) > 100


def test_tile_lists_ragged_image_and_offscreen():
    s = scenes.make_scene("unbounded", N=3000)
    s.scales *= 6.0
    cam = scenes.make_camera(150, 70, 60.0, scenes.make_cameras("unbounded")[2].world_to_cam)   # 10x5 tiles, ragged
    pr, lists = _check(s, cam)
    v = pr["visible"] > 0
    assert 0 < v.sum() < s.N                  # some culled (behind / off screen)
    assert (pr["tiles_touched"][v] == cam.tiles_x * cam.tiles_y).any()   # some cover the whole screen


def test_depth_ties_are_stable_by_index():
    s = scenes.make_scene("tiny", N=64)
    s.means[:] = s.means[0]                   # identical depth for all: order must be the primitive index
    s.scales *= 3.0
    cam = scenes.make_cameras("tiny")[0]
    pr, lists = _check(s, cam)
    assert len(np.unique(pr["depth_bits"])) == 1
    for l in lists:
        assert np.all(np.diff(l) > 0)


def test_radius_is_three_sigma_of_largest_eigenvalue():
    s = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    pr = orc.project(s, cam)
    v = pr["visible"] > 0
    U = pr["cov2d"][v]
    lam = np.array([np.linalg.eigvalsh([[u[0] + 0.3, u[1]], [u[1], u[2] + 0.3]])[1] for u in U])
    want = np.ceil(3 * np.sqrt(lam))
    diff = pr["radius"][v] - want
    assert np.abs(diff).max() <= 1 and (diff != 0).mean() < 0.01     # float32 twin vs double, ceil boundary only
