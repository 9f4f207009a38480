"""Pins of the oracle's auxiliary renders: frequency map, depth, accumulated alpha."""
import numpy as np

from oracle import gabsplat_oracle as orc
from paper_2508_05343_b200 import scenes


def test_alpha_channel_telescopes_and_T_is_unchanged():
    """sum_i alpha_i T_i = 1 - T_final for the blended primitives (telescoping), and replacing the colours does
    not change which primitives are blended."""
    s = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    a, f = orc.render_aux(s, cam), orc.render_forward(s, cam)
    assert np.array_equal(a["final_T"], f["final_T"])
    assert np.max(np.abs(a["image"][2] - (1.0 - f["final_T"]))) < 1e-14


def test_depth_channel_is_bounded_by_the_visible_depths():
    s = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    a, p = orc.render_aux(s, cam), orc.project(s, cam)
    z = p["t"][p["tiles_touched"] > 0, 2]
    alpha = a["image"][2]
    assert np.all(a["image"][1] <= z.max() * alpha + 1e-12) and np.all(a["image"][1] >= z.min() * alpha - 1e-12)


def test_zero_weights_give_a_zero_frequency_map():
    s = scenes.make_scene("tiny", zero_weights=True)
    cam = scenes.make_cameras("tiny")[0]
    assert np.all(orc.render_aux(s, cam)["image"][0] == 0.0)


def test_single_primitive_closed_form():
    """One isotropic primitive on the optical axis (the north_star pin): at its centre pixel alpha = o, so the
    channels are o * sum_k omega_k |f_k,xy| z / fx, o * z and o."""
    s = scenes.make_scene("tiny", N=1, K=2)
    s.means[:] = [[0.0, 0.0, 0.0]]
    s.scales[:] = 0.05
    s.rotations[:] = [[1.0, 0.0, 0.0, 0.0]]
    s.opacities[:] = 0.6
    s.freqs[:] = [[[3.0, 4.0, 1.0], [0.0, 2.0, 5.0]]]
    s.weights[:] = [[0.25, 0.5]]
    base = scenes.make_cameras("tiny")[0]
    cam = scenes.make_camera(129, 129, 150.0, base.world_to_cam, base.bg)   # odd size: a pixel at the centre
    a = orc.render_aux(s, cam)["image"][:, 64, 64]
    z, fx, o = 4.0, 150.0, float(np.float32(0.6))
    fm = (0.25 * 5.0 + 0.5 * 2.0) * z / fx
    assert abs(a[2] - o) < 1e-12 and abs(a[1] - o * z) < 1e-9 and abs(a[0] - o * fm) < 1e-9
