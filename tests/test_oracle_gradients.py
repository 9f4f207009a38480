"""Pin of the oracle's analytic backward (backward_pixels / backward_primitive) by central finite
differences of the oracle's own double-precision forward image -- CPU only.

The paper gives no backward equations (PAPER.md:48 "differentiable", :129 "optimized ... during training");
the chain rule is derived in DESIGN.md "Backward".  Scenes: <=16 primitives at 16x16 (one tile, so the tile
rectangle cannot change), all seven parameter groups, plus the cases of readings C14 (alpha clamp) and C15
(clamped ray direction, SH clamp).  A coordinate is compared only when the blended sets at +h and -h are
identical (the image is discontinuous at the 1/255 and 1e-4 thresholds, reading C18).
"""
import numpy as np
import pytest

from oracle import gabsplat_oracle as orc
from paper_2508_05343_b200 import scenes

GROUPS = [("means", "d_means"), ("scales", "d_scales"), ("rotations", "d_rotations"), ("opacities", "d_opacities"),
          ("sh", "d_sh"), ("freqs", "d_freqs"), ("weights", "d_weights")]


def _loss(s, cam, g):
    o = orc.render_forward(s, cam)
    return float((o["image"] * g).sum()), o


def _fd_check(s, cam, seed=0, rel_h=2.0 ** -12, tol=2e-5, min_fraction=0.9):
    rng = np.random.default_rng(seed)
    g = rng.normal(size=(3, cam.height, cam.width)).astype(np.float32)
    ana = orc.render_backward(s, cam, g)
    base = orc.render_forward(s, cam)
    assert np.abs(ana["image"] - base["image"]).max() == 0
    report = {}
    for name, gname in GROUPS:
        arr = getattr(s, name)
        flat = arr.reshape(-1)
        fd = np.full(flat.shape, np.nan)
        typical = float(np.abs(flat).mean()) + 1e-3
        for j in range(flat.size):
            x0 = flat[j]
            for shrink in (1.0, 1.0 / 16, 1.0 / 256):          # "else resample": retry with a smaller step
                h = np.float32(shrink * rel_h * max(abs(float(x0)), typical))
                flat[j] = x0 + h
                xp = float(flat[j]); Lp, op = _loss(s, cam, g)
                flat[j] = x0 - h
                xm = float(flat[j]); Lm, om = _loss(s, cam, g)
                flat[j] = x0
                same = np.array_equal(op["counters"][..., 2], om["counters"][..., 2]) and \
                    np.array_equal(op["last_id"], om["last_id"]) and np.array_equal(op["last_id"], base["last_id"])
                if same:
                    fd[j] = (Lp - Lm) / (xp - xm)
                    break
        a = ana[gname].reshape(-1)
        ok = ~np.isnan(fd)
        scale = np.abs(a).max()
        assert ok.mean() >= min_fraction, (name, ok.mean())
        err = np.abs(fd[ok] - a[ok]).max() / scale if scale > 0 else np.abs(fd[ok]).max()
        report[name] = (err, ok.mean(), scale)
        assert err < tol, (name, err)
    return report, ana


def test_gradients_match_finite_differences_all_groups():
    s, cam = scenes.small_scene(21, 12, 3)
    rep, ana = _fd_check(s, cam)
    for name, gname in GROUPS:
        assert np.abs(ana[gname]).max() > 0, name             # every group receives gradient


def test_gradients_k4_sixteen_primitives():
    s, cam = scenes.small_scene(22, 16, 4)
    _fd_check(s, cam, seed=1)


def test_gradients_with_clamps():
    """Readings C14/C15: alpha clamp at 0.99, ray direction clamp outside 1.3x the field of view, SH clamp at 0."""
    s, cam = scenes.small_scene(23, 8, 2)
    s.opacities[0] = 0.9999                                   # o*G*M > 0.99 near its centre
    s.weights[0] = 0.0
    s.means[1] = [3.2, 0.0, 0.5]                              # far off axis: t_x/t_z beyond the clamp
    s.scales[1] = 1.5                                         # but large enough to reach the tile
    s.sh[2, 0, 0] = -3.0                                      # red channel clamps at 0
    pr = orc.project(s, cam)
    t = pr["t"][1]
    assert pr["visible"][1] and abs(t[0] / t[2]) > 1.3 * 0.5 * cam.width / cam.fx
    assert pr["clamped"][2, 0] == 1
    base = orc.render_forward(s, cam)
    assert (base["margin"][..., 1] < 1e290).any()
    rep, ana = _fd_check(s, cam, seed=2)
    assert np.all(ana["d_sh"][2, :, 0] == 0)


def test_zero_weights_give_zero_frequency_gradient_and_gaussian_gradients():
    """with w=0 the primitive is a Gaussian: dL/df = 0, other gradients equal those of K=0."""
    s, cam = scenes.small_scene(24, 10, 2)
    g = np.random.default_rng(3).normal(size=(3, cam.height, cam.width)).astype(np.float32)
    z = s.copy(); z.weights[:] = 0
    k0 = scenes.Scene(s.means, s.scales, s.rotations, s.opacities, s.sh,
                      np.zeros((s.N, 0, 3), np.float32), np.zeros((s.N, 0), np.float32))
    a, b = orc.render_backward(z, cam, g), orc.render_backward(k0, cam, g)
    assert np.all(a["d_freqs"] == 0)
    assert np.abs(a["d_weights"]).max() > 0                    # dL/dw is not zero at w=0
    for n in ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh"):
        assert np.abs(a[n] - b[n]).max() <= 1e-12 * max(1.0, np.abs(b[n]).max()), n


def test_culled_primitive_has_zero_gradient():
    s, cam = scenes.small_scene(25, 6, 2)
    s.means[3] = [0, 0, -10.0]                                # behind the camera
    g = np.ones((3, cam.height, cam.width), np.float32)
    a = orc.render_backward(s, cam, g)
    for _, gname in GROUPS:
        assert np.all(a[gname][3] == 0)
