"""CPU pins of two oracle parts that finite differences cannot see.

1. `absmean2d` (oracle/gabsplat_oracle.cpp backward_pixels): the AbsGS densification statistic, the sum over pixels of
   the ABSOLUTE per-pixel dL/dmu2D (PAPER.md:224 "+AbsGS", :175 "view-space positional gradient").  Pinned by
   (a) dL/dimage non-zero at ONE pixel => |d_mean2d| == d_absmean2d exactly; (b) d_absmean2d >= |d_mean2d|
   element-wise, and additivity over disjoint pixel sets; (c) a two-pixel, one-primitive case computed by hand from
   Eq.12-13 with opposite-sign terms.

2. The decision-injected mode (reading C18): injecting the oracle's own decisions changes nothing and
   reports no violation; a flipped decision far from its threshold is reported; a flipped decision within the
   margin is accepted and produces the rendering in which that pair is skipped / blended.
"""
import numpy as np

from oracle import gabsplat_oracle as orc
from paper_2508_05343_b200 import scenes


def _one_hot_grad(cam, x, y, rng):
    g = np.zeros((3, cam.height, cam.width), np.float32)
    g[:, y, x] = rng.normal(size=3).astype(np.float32)
    return g


def test_absgrad_single_pixel_equals_abs_of_gradient():
    s, cam = scenes.small_scene(31, 12, 3)
    rng = np.random.default_rng(5)
    hit = 0
    for x, y in ((6, 7), (8, 8), (9, 6), (7, 9)):
        a = orc.render_backward(s, cam, _one_hot_grad(cam, x, y, rng))
        assert np.array_equal(np.abs(a["d_mean2d"]), a["d_absmean2d"])
        hit += int(np.abs(a["d_mean2d"]).max() > 0)
    assert hit >= 3


def test_absgrad_dominates_and_is_additive_over_pixels():
    s, cam = scenes.small_scene(32, 16, 4)
    rng = np.random.default_rng(6)
    g = rng.normal(size=(3, cam.height, cam.width)).astype(np.float32)
    full = orc.render_backward(s, cam, g)
    assert np.all(full["d_absmean2d"] >= np.abs(full["d_mean2d"]) - 1e-15)
    assert (full["d_absmean2d"] > np.abs(full["d_mean2d"]) * 1.01).any()      # cancellation does occur
    # additivity: the statistic of the whole image is the sum of the statistics of its two halves
    left, right = g.copy(), g.copy()
    left[:, :, cam.width // 2:] = 0
    right[:, :, :cam.width // 2] = 0
    a, b = orc.render_backward(s, cam, left), orc.render_backward(s, cam, right)
    assert np.allclose(a["d_absmean2d"] + b["d_absmean2d"], full["d_absmean2d"], rtol=1e-12, atol=1e-15)
    assert np.allclose(a["d_mean2d"] + b["d_mean2d"], full["d_mean2d"], rtol=1e-10, atol=1e-14)
    # ... and the sum over one-hot images of |per-pixel gradient| (brute force on a 4x4 block)
    acc = np.zeros_like(full["d_absmean2d"])
    blk = np.zeros_like(g)
    for y in range(6, 10):
        for x in range(6, 10):
            h = np.zeros_like(g)
            h[:, y, x] = g[:, y, x]
            blk[:, y, x] = g[:, y, x]
            acc += np.abs(orc.render_backward(s, cam, h)["d_mean2d"])
    assert np.allclose(orc.render_backward(s, cam, blk)["d_absmean2d"], acc, rtol=1e-12, atol=1e-15)


def test_absgrad_two_pixels_by_hand():
    """One isotropic on-axis Gaussian-only primitive (K=0), two pixels on opposite sides of its centre with the same
    dL/dC: the x gradients cancel exactly, their absolute values add.  Hand computation from Eq.12-13:
    C = c a + (1 - a) bg, a = o exp(-r^2 / (2 sigma^2)), dC/dmu_x = (c - bg) a (x - mu_x) / sigma^2."""
    z, sc, o, fx = 4.0, float(np.float32(0.05)), float(np.float32(0.6)), 64.0   # the float32 values the scene stores
    cam = scenes.make_camera(17, 17, fx, np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 0]], np.float32), bg=(0.1, 0.2, 0.3))
    s = scenes.Scene(np.array([[0, 0, z]], np.float32), np.full((1, 3), sc, np.float32),
                     np.array([[1, 0, 0, 0]], np.float32), np.array([o], np.float32), np.zeros((1, 16, 3), np.float32),
                     np.zeros((1, 0, 3), np.float32), np.zeros((1, 0), np.float32))
    s.sh[0, 0] = [1.0, 0.5, -0.2]
    pr = orc.project(s, cam)
    assert pr["visible"][0] and np.allclose(pr["mean2d"][0], [8.0, 8.0])
    sigma2 = sc * sc * fx * fx / (z * z) + 0.3
    rgb = pr["rgb"][0]
    g = np.zeros((3, 17, 17), np.float32)
    gc = np.array([0.7, -0.4, 1.1], np.float32)
    g[:, 8, 7] = gc
    g[:, 8, 9] = gc
    a = orc.render_backward(s, cam, g)
    alpha = o * np.exp(-1.0 / (2 * sigma2))
    assert alpha > 1.0 / 255
    term = float(np.dot(gc.astype(np.float64), rgb - np.array(cam.bg))) * alpha / sigma2     # |dL/dmu_x| of one pixel
    assert abs(a["d_mean2d"][0, 0]) < 1e-15 * max(1.0, abs(term))
    assert np.isclose(a["d_absmean2d"][0, 0], 2 * abs(term), rtol=1e-12)
    assert a["d_absmean2d"][0, 1] == 0 and a["d_mean2d"][0, 1] == 0


# ---- decision-injected mode ---------------------------------------------------------------------------

def _all_pixels(cam):
    ys, xs = np.mgrid[0:cam.height, 0:cam.width]
    return np.stack([xs.ravel(), ys.ravel()], axis=1).astype(np.int32)


def test_injecting_own_decisions_is_identity():
    s, cam = scenes.small_scene(33, 16, 4)
    s.opacities[:8] = 0.9999                              # some clamped pairs and saturating pixels
    s.weights[:8] = 0.0
    s.scales[:8] *= 3
    rng = np.random.default_rng(7)
    g = rng.normal(size=(3, cam.height, cam.width)).astype(np.float32)
    ref = orc.render_backward(s, cam, g)
    tr = orc.trace_pixels(s, cam, _all_pixels(cam))
    fwd = orc.render_forward(s, cam)
    assert np.array_equal(tr["counts"].reshape(cam.height, cam.width), fwd["counters"][..., 2])
    assert (tr["entries"] >> 31).any()                    # the clamp flag is exercised
    assert (tr["stop_pos"] > 0).any()                     # ... and the saturation stop
    inj = orc.render_backward(s, cam, g, inject=dict(tr, delta=0.0))
    assert inj["violations"] == 0
    for k in ref:
        if k != "violations":
            assert np.array_equal(ref[k], inj[k]), k


def test_flipped_decision_far_from_threshold_is_a_violation():
    s, cam = scenes.small_scene(34, 10, 2)
    g = np.ones((3, cam.height, cam.width), np.float32)
    px = np.array([[8, 8]], np.int32)
    tr = orc.trace_pixels(s, cam, px)
    assert tr["counts"][0] >= 2
    # drop the first blended entry: alpha there is far above 1/255
    bad = dict(pixels=px, offsets=np.array([0, tr["counts"][0] - 1], np.uint32), entries=tr["entries"][1:],
               stop_pos=tr["stop_pos"], delta=1e-4)
    assert orc.render_backward(s, cam, g, inject=bad)["violations"] > 0
    # flip a clamp flag on a pair that is nowhere near 0.99
    ent = tr["entries"].copy()
    ent[0] ^= np.uint32(0x80000000)
    bad = dict(tr, entries=ent, delta=1e-4)
    assert orc.render_backward(s, cam, g, inject=bad)["violations"] > 0
    # a stop where nothing stops
    bad = dict(tr, stop_pos=np.array([tr["entries"][0] & 0x7fffffff], np.uint32), delta=1e-4)
    assert orc.render_backward(s, cam, g, inject=bad)["violations"] > 0


def test_flip_within_margin_is_accepted_and_changes_the_rendering():
    """Tune one opacity so that alpha at one pixel is 1/255 (1 + 3e-5): the oracle blends it; a list without it is
    a correct rendering at delta = 1e-4, and the image / gradient there are those of the skipped pair."""
    s, cam = scenes.small_scene(35, 6, 2)
    x, y = 8, 8
    px = np.array([[x, y]], np.int32)
    tr0 = orc.trace_pixels(s, cam, px)
    ids = orc.render_forward(s, cam)
    assert tr0["counts"][0] >= 2
    # the last blended entry at the pixel: find its primitive, scale its opacity so alpha lands just above 1/255
    order = orc.bin_sort(s, cam)
    tile_ids = order["ids"]                                # one tile (16x16)
    last_pos = int(tr0["entries"][tr0["counts"][0] - 1] & 0x7fffffff)
    prim = int(tile_ids[last_pos - 1])
    lo, hi = 0.0, float(s.opacities[prim])
    for _ in range(200):                                   # bisection on the float32 opacity
        mid = np.float32(0.5 * (lo + hi))
        s.opacities[prim] = mid
        t = orc.trace_pixels(s, cam, px)
        blended = last_pos in set((t["entries"] & 0x7fffffff).tolist())
        if blended:
            hi = float(mid)
        else:
            lo = float(mid)
    s.opacities[prim] = np.float32(hi)
    fwd = orc.render_forward(s, cam)
    assert fwd["margin"][y, x, 0] < 1e-4                   # the pixel is undecidable at delta = 1e-4
    tr = orc.trace_pixels(s, cam, px)
    assert last_pos in set((tr["entries"] & 0x7fffffff).tolist())
    keep = (tr["entries"] & 0x7fffffff) != last_pos
    flipped = dict(pixels=px, offsets=np.array([0, keep.sum()], np.uint32), entries=tr["entries"][keep],
                   stop_pos=tr["stop_pos"], delta=1e-4)
    g = np.zeros((3, cam.height, cam.width), np.float32)
    g[:, y, x] = 1.0
    a = orc.render_backward(s, cam, g)
    b = orc.render_backward(s, cam, g, inject=flipped)
    assert b["violations"] == 0
    assert orc.render_backward(s, cam, g, inject=dict(flipped, delta=1e-9))["violations"] > 0
    assert b["n_contrib"][y, x] <= a["n_contrib"][y, x]
    jump = np.abs(a["image"][:, y, x] - b["image"][:, y, x]).max()
    assert 0 < jump <= (1.0 / 255) * 1.001                 # one alpha_min step, scaled by T |c - B| <= 1
    assert b["d_opacities"][prim] == 0 and a["d_opacities"][prim] != 0
    # every other pixel is untouched
    mask = np.ones((cam.height, cam.width), bool)
    mask[y, x] = False
    assert np.array_equal(a["image"][:, mask], b["image"][:, mask])
