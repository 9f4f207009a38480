"""Pins of the oracle's compositing (oracle/gabsplat_oracle.cpp visit / forward_painter) -- CPU only.

  * Single isotropic primitive at the image centre: closed-form 2D Gabor profile (BASELINE.json north_star;
    PAPER.md:158 Eq.12 with the on-axis projection of reading C21).
  * Two overlapping primitives: Eq.13 written out by hand, front one first.
  * w = 0 or f = 0 reduces to plain Gaussian splatting: compared with a separately written
    numpy Gaussian-only compositor (Eq.3-4).
  * Partition of unity (reading C23), permutation invariance ("sorted by depth"), splitting a
    component (Eq.7 is a sum), literal O(N W H) loop == painter's loop bit for bit.
"""
import numpy as np

from oracle import gabsplat_oracle as orc
from paper_2508_05343_b200 import scenes

K0 = np.sqrt(1.0 / (4 * np.pi))


def _set_flat_colour(s, rgb):
    s.sh[:] = 0
    s.sh[:, 0, :] = (np.asarray(rgb, np.float64) - 0.5) / K0


def _central_primitive(K=2, z=4.0, fx=150.0, size=65, sc=0.12, opac=0.8):
    s, _ = scenes.small_scene(2, 1, K)
    s.means[:] = [0, 0, 0]
    s.scales[:] = sc
    s.rotations[:] = [1, 0, 0, 0]
    s.opacities[:] = opac
    _set_flat_colour(s, [0.9, 0.5, 0.2])
    cam = scenes.make_camera(size, size, fx, scenes.look_at([0, 0, -z], [0, 0, 1.0]), bg=(0.1, 0.2, 0.3))
    return s, cam, z, fx


def test_single_isotropic_primitive_closed_form():
    s, cam, z, fx = _central_primitive()
    s.freqs[0] = [[3.0, 1.0, 5.0], [-2.0, 4.0, -7.0]]      # f_z must drop out on axis
    s.weights[0] = [0.45, 0.35]
    out = orc.render_forward(s, cam, literal=True)
    sc, o = float(s.scales[0, 0]), float(s.opacities[0])
    sig2 = sc * sc * fx * fx / (z * z) + 0.3
    yy, xx = np.mgrid[0:cam.height, 0:cam.width].astype(np.float64)
    dx, dy = xx - cam.cx, yy - cam.cy
    G = np.exp(-(dx * dx + dy * dy) / (2 * sig2))
    M = 1.0 - sum(float(s.weights[0, k]) * (1 - np.cos(2 * np.pi * (z / fx) * (float(s.freqs[0, k, 0]) * dx + float(s.freqs[0, k, 1]) * dy)))
                  for k in range(2))
    alpha = np.minimum(0.99, o * G * M)
    alpha[alpha < 1 / 255] = 0
    rgb = 0.5 + K0 * s.sh[0, 0].astype(np.float64)
    want = rgb[:, None, None] * alpha + (1 - alpha) * np.asarray(cam.bg)[:, None, None]
    # radius covers the whole 65x65 image here (3 sigma ~ 14 px -> rect clamps to all 5x5 tiles)
    assert np.abs(out["image"] - want).max() < 1e-12
    assert np.abs(out["final_T"] - (1 - alpha)).max() < 1e-12
    assert np.array_equal(out["n_contrib"] > 0, alpha > 0)
    # centre value: modulation is exactly 1 at d = 0 for any f, w (weights sum to one)
    c = cam.height // 2
    assert np.allclose(out["image"][:, c, c], rgb * o + (1 - o) * np.asarray(cam.bg), atol=1e-12)
    # M goes negative somewhere with these weights (reading C6) and those pixels are skipped
    assert (M < 0).any() and np.all(out["n_contrib"][M < 0] == 0)


def test_alpha_clamp_at_099():
    s, cam, z, fx = _central_primitive(opac=0.999)
    s.weights[:] = 0
    out = orc.render_forward(s, cam)
    c = cam.height // 2
    assert abs(out["final_T"][c, c] - 0.01) < 1e-12


def test_two_primitives_eq13_written_out():
    s, _ = scenes.small_scene(3, 2, 1)
    s.means[:] = [[0, 0, 0.5], [0, 0, -0.5]]               # index 1 is nearer to the camera at z=-4
    s.scales[:] = 0.1
    s.rotations[:] = [1, 0, 0, 0]
    s.opacities[:] = [0.7, 0.6]
    s.freqs[:] = [[[2.0, 0, 0]], [[0, 3.0, 0]]]
    s.weights[:] = [[0.3], [0.2]]
    s.sh[:] = 0
    s.sh[0, 0] = (np.array([1.0, 0.0, 0.5]) - 0.5) / K0
    s.sh[1, 0] = (np.array([0.0, 1.0, 0.25]) - 0.5) / K0
    fx = 100.0
    cam = scenes.make_camera(33, 33, fx, scenes.look_at([0, 0, -4.0], [0, 0, 1.0]))
    out = orc.render_forward(s, cam)
    for (x, y) in [(16, 16), (18, 15), (12, 20), (16, 22)]:
        dx, dy = x - 16.0, y - 16.0
        a = []
        for i, zc in ((1, 3.5), (0, 4.5)):                 # front to back
            sig2 = float(s.scales[i, 0]) ** 2 * fx * fx / zc ** 2 + 0.3
            G = np.exp(-(dx * dx + dy * dy) / (2 * sig2))
            f = s.freqs[i, 0].astype(np.float64) * zc / fx
            w = float(s.weights[i, 0])
            a.append(float(s.opacities[i]) * G * (1 - w + w * np.cos(2 * np.pi * (f[0] * dx + f[1] * dy))))
        assert min(a) > 1 / 255 and max(a) < 0.99
        c1 = 0.5 + K0 * s.sh[1, 0].astype(np.float64)
        c0 = 0.5 + K0 * s.sh[0, 0].astype(np.float64)
        want = c1 * a[0] + c0 * a[1] * (1 - a[0])
        assert np.allclose(out["image"][:, y, x], want, atol=1e-12)
        assert abs(out["final_T"][y, x] - (1 - a[0]) * (1 - a[1])) < 1e-12
        assert out["last_id"][y, x] == 0 and out["n_contrib"][y, x] == 2


def _numpy_gaussian_splat(s, cam):
    """Plain 3D Gaussian splatting (Eq.1-4) in numpy.  Separately written: own projection, own loop.
    Takes only the tile rectangle and depth order from the oracle (pinned in test_oracle_binning.py)."""
    pr = orc.project(s, cam)
    Wm = cam.world_to_cam.astype(np.float64)
    N = s.N
    order = sorted([i for i in range(N) if pr["visible"][i]], key=lambda i: (int(pr["depth_bits"][i]), i))
    H, W = cam.height, cam.width
    img = np.zeros((3, H, W)); T = np.ones((H, W)); done = np.zeros((H, W), bool)
    yy, xx = np.mgrid[0:H, 0:W].astype(np.float64)
    cam_pos = -Wm[:, :3].T @ Wm[:, 3]
    limx, limy = 1.3 * 0.5 * W / cam.fx, 1.3 * 0.5 * H / cam.fy
    for i in order:
        mu = s.means[i].astype(np.float64)
        t = Wm[:, :3] @ mu + Wm[:, 3]
        qw, qx, qy, qz = s.rotations[i].astype(np.float64)
        R = np.array([[1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qw * qz), 2 * (qx * qz + qw * qy)],
                      [2 * (qx * qy + qw * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qw * qx)],
                      [2 * (qx * qz - qw * qy), 2 * (qy * qz + qw * qx), 1 - 2 * (qx * qx + qy * qy)]])
        Sg = R @ np.diag(s.scales[i].astype(np.float64) ** 2) @ R.T
        ux, uy = np.clip(t[0] / t[2], -limx, limx), np.clip(t[1] / t[2], -limy, limy)
        J = np.array([[cam.fx / t[2], 0, -cam.fx * ux / t[2]], [0, cam.fy / t[2], -cam.fy * uy / t[2]]])
        U = J @ Wm[:, :3] @ Sg @ Wm[:, :3].T @ J.T + 0.3 * np.eye(2)
        Ci = np.linalg.inv(U)
        m2 = np.array([cam.fx * t[0] / t[2] + cam.cx, cam.fy * t[1] / t[2] + cam.cy])
        d = (mu - cam_pos) / np.linalg.norm(mu - cam_pos)
        Y, _ = orc.sh_basis(d[None])                        # SH basis pinned in test_oracle_projection.py
        rgb = np.maximum(0.0, 0.5 + Y[0] @ s.sh[i].astype(np.float64))
        x0, y0, x1, y1 = pr["rect"][i]
        mask = (xx >= 16 * x0) & (xx < 16 * x1) & (yy >= 16 * y0) & (yy < 16 * y1) & ~done
        dx, dy = xx - m2[0], yy - m2[1]
        power = -0.5 * (Ci[0, 0] * dx * dx + Ci[1, 1] * dy * dy) - Ci[0, 1] * dx * dy
        alpha = np.minimum(0.99, float(s.opacities[i]) * np.exp(power))
        mask &= (power <= 0) & (alpha >= 1 / 255)
        stop = mask & (T * (1 - alpha) < 1e-4)
        done |= stop
        mask &= ~stop
        img += rgb[:, None, None] * np.where(mask, alpha * T, 0.0)
        T = np.where(mask, T * (1 - alpha), T)
    return img + T * np.asarray(cam.bg)[:, None, None], T


def test_zero_weights_or_zero_freqs_reduce_to_gaussian_splatting():
    s = scenes.make_scene("tiny", N=300)
    s.scales *= 2.0
    cam = scenes.make_camera(64, 48, 75.0, scenes.look_at([0.2, 0.1, -4.0], [0, 0, 1.0]), bg=(0.3, 0.1, 0.6))
    zw = s.copy(); zw.weights[:] = 0
    zf = s.copy(); zf.freqs[:] = 0
    want, wantT = _numpy_gaussian_splat(s, cam)
    for variant in (zw, zf):
        out = orc.render_forward(variant, cam)
        assert np.abs(out["image"] - want).max() < 1e-10
        assert np.abs(out["final_T"] - wantT).max() < 1e-10
    full = orc.render_forward(s, cam)
    assert np.abs(full["image"] - want).max() > 1e-2        # the Gabor terms do change the image


def test_partition_of_unity():
    s = scenes.make_scene("tiny", N=400)
    s.scales *= 3.0
    _set_flat_colour(s, [1.0, 1.0, 1.0])
    cam = scenes.make_camera(48, 48, 60.0, scenes.look_at([0, 0, -4.0], [0, 0, 1.0]), bg=(1.0, 1.0, 1.0))
    out = orc.render_forward(s, cam)
    assert out["n_contrib"].max() > 3
    assert np.abs(out["image"] - 1.0).max() < 1e-6          # float32 SH coefficient rounding only


def test_permutation_invariance_and_component_split():
    s = scenes.make_scene("tiny", N=256)
    s.scales *= 2.0
    cam = scenes.make_cameras("tiny")[0]
    base = orc.render_forward(s, cam)
    perm = np.random.default_rng(1).permutation(s.N)
    assert len(np.unique(orc.project(s, cam)["depth_bits"][orc.project(s, cam)["visible"] > 0])) == \
        int((orc.project(s, cam)["visible"] > 0).sum())     # distinct depths, so order is unique
    p = scenes.Scene(*(a[perm].copy() for a in (s.means, s.scales, s.rotations, s.opacities, s.sh, s.freqs, s.weights)))
    outp = orc.render_forward(p, cam)
    assert np.abs(outp["image"] - base["image"]).max() < 1e-13
    assert np.array_equal(perm[outp["last_id"]][outp["last_id"] >= 0], base["last_id"][base["last_id"] >= 0])
    # split every component into two halves with the same frequency: Eq.7 is linear in w
    sp = scenes.Scene(s.means, s.scales, s.rotations, s.opacities, s.sh,
                      np.ascontiguousarray(np.repeat(s.freqs, 2, axis=1)),
                      np.ascontiguousarray(np.repeat(s.weights * np.float32(0.5), 2, axis=1)))
    outs = orc.render_forward(sp, cam)
    assert np.abs(outs["image"] - base["image"]).max() < 1e-12


def test_literal_equals_painter_and_pixel_sampler():
    s = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    a = orc.render_forward(s, cam, literal=True)
    b = orc.render_forward(s, cam, literal=False)
    for k in ("image", "final_T", "n_contrib", "last_id", "counters"):
        assert np.array_equal(a[k], b[k]), k
    px = np.array([[5, 7], [64, 64], [127, 0], [33, 90]])
    c = orc.render_pixels(s, cam, px)
    for j, (x, y) in enumerate(px):
        assert np.array_equal(c["colour"][j], a["image"][:, y, x]) and c["n_contrib"][j] == a["n_contrib"][y, x]
    assert a["counters"][..., 2].sum() > 10000 and a["n_contrib"].max() > 10
