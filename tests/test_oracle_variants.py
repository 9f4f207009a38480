"""CPU pins of the primitive variants in the oracle (oracle/gabsplat_oracle.cpp, Scene.variant).

VARIANT_LINE_INTEGRAL -- the amplitude of the exact line integral that Eq.12 drops (Eq.25-27; the
printed constants are garbled, reading C4): component k is attenuated by C2_k = exp(-2 pi^2 f_z''^2 / S22).
  * numerical z-quadrature of the ray-space 3D Gabor divided by that of the Gaussian alone = C2_k cos(2 pi f2D.p):
    the amplitude is INCLUDED in the comparison (the test of Eq.18-29 in test_oracle_projection.py computes its own);
  * C2_k does not depend on how J's third row is completed (reading C2) and equals exp(-2 pi^2 (v.f)^2 / (v^T Sigma^-1 v))
    with v the null vector of the finite-difference Jacobian of the pinhole map;
  * on-axis isotropic closed form C2 = exp(-2 pi^2 f_z^2 s^2), and the rendered profile of a single such primitive;
  * f = 0 or w = 0 leaves the render unchanged; finite differences on all seven parameter groups.

VARIANT_MIP_FILTER -- Mip-Splatting's 2D filter in place of the 0.3 dilation:
  * closed form on the on-axis isotropic primitive: sigma^2 = sigma0^2 + 0.1, alpha scaled by sigma0^2 / (sigma0^2 + 0.1);
  * rho^2 = det U / det(U + 0.1 I) from the oracle's own U; the integral of the splat over the plane is independent of
    the dilation (what the filter is for); radius from the 0.1 dilation; finite differences.
"""
import numpy as np

from oracle import gabsplat_oracle as orc
from paper_2508_05343_b200 import scenes
from test_oracle_gradients import _fd_check, GROUPS
from test_oracle_projection import _scene, _fd_T, _sigma_world
from test_oracle_render import _central_primitive, K0

LINE, MIP = orc.VARIANT_LINE_INTEGRAL, orc.VARIANT_MIP_FILTER


def test_attenuation_is_the_amplitude_of_the_z_integral():
    s, cam = _scene(seed=5, N=4, K=2)
    s.freqs *= 0.5                         # keep C2 well away from 0 so that the ratio is well conditioned
    o = orc.project(s, cam, third_row=1)   # the EWA ray-space completion (z'' = distance along the ray)
    seen = 0
    for i in range(s.N):
        S = np.linalg.inv(o["Sigma3"][i])
        U = o["Sigma3"][i][:2, :2]
        sz = 1.0 / np.sqrt(S[2, 2])
        sd = np.sqrt(np.diag(U))
        for k in range(s.K):
            fp, f2 = o["fproj"][i, k], o["freq2d"][i, k]
            for p in (np.array([0.3, -0.2]) * sd, np.array([-0.7, 0.5]) * sd, np.array([0.0, 0.0])):
                zc = -(S[0, 2] * p[0] + S[1, 2] * p[1]) / S[2, 2]
                z = zc + np.linspace(-12, 12, 48001) * sz
                X = np.stack([np.full_like(z, p[0]), np.full_like(z, p[1]), z], 1)
                env = np.exp(-0.5 * np.einsum("na,ab,nb->n", X, S, X))
                ratio = (env * np.cos(2 * np.pi * X @ fp)).sum() / env.sum()
                assert abs(ratio - o["att"][i, k] * np.cos(2 * np.pi * f2 @ p)) <= 1e-9
                seen += 1
    assert seen == 24 and 0.0 < o["att"].min() < 0.99 and o["att"].max() <= 1.0


def test_attenuation_independent_of_third_row_and_null_space_form():
    s, cam = _scene()
    a0, a1, a2 = (orc.project(s, cam, third_row=r)["att"] for r in (0, 1, 2))
    vis = orc.project(s, cam)["visible"].astype(bool)
    assert vis.sum() >= 6
    assert np.allclose(a0[vis], a1[vis], rtol=1e-9, atol=1e-300) and np.allclose(a0[vis], a2[vis], rtol=1e-9, atol=1e-300)
    for i in np.nonzero(vis)[0]:
        T = _fd_T(cam, s.means[i].astype(np.float64))
        v = np.linalg.svd(T)[2][2]                       # null vector of the 2x3 Jacobian: the ray direction
        b = v @ np.linalg.solve(_sigma_world(s, i), v)
        for k in range(s.K):
            a = v @ s.freqs[i, k].astype(np.float64)
            assert np.isclose(a0[i, k], np.exp(-2 * np.pi ** 2 * a * a / b), rtol=1e-5)


def test_attenuation_on_axis_closed_form_and_rendered_profile():
    s, cam, z, fx = _central_primitive()
    s.freqs[0] = [[3.0, 1.0, 1.5], [-2.0, 4.0, -0.8]]
    s.weights[0] = [0.45, 0.35]
    s.variant = LINE
    sc, o = float(s.scales[0, 0]), float(s.opacities[0])
    att = np.exp(-2 * np.pi ** 2 * s.freqs[0, :, 2].astype(np.float64) ** 2 * sc * sc)
    assert np.allclose(orc.project(s, cam)["att"][0], att, rtol=1e-12)
    assert 0.05 < att.min() < 0.9
    out = orc.render_forward(s, cam, literal=True)
    sig2 = sc * sc * fx * fx / (z * z) + 0.3
    yy, xx = np.mgrid[0:cam.height, 0:cam.width].astype(np.float64)
    dx, dy = xx - cam.cx, yy - cam.cy
    G = np.exp(-(dx * dx + dy * dy) / (2 * sig2))
    w = s.weights[0].astype(np.float64)
    M = (1.0 - w.sum()) + sum(w[k] * att[k] * np.cos(2 * np.pi * (z / fx) * (float(s.freqs[0, k, 0]) * dx + float(s.freqs[0, k, 1]) * dy))
                              for k in range(2))
    alpha = np.minimum(0.99, o * G * M)
    alpha[alpha < 1 / 255] = 0
    rgb = 0.5 + K0 * s.sh[0, 0].astype(np.float64)
    want = rgb[:, None, None] * alpha + (1 - alpha) * np.asarray(cam.bg)[:, None, None]
    assert np.abs(out["image"] - want).max() < 1e-12
    # the centre value is no longer o: the cosine terms lost amplitude, the Gaussian term did not
    c = cam.height // 2
    assert np.isclose(out["final_T"][c, c], 1 - o * ((1 - w.sum()) + (w * att).sum()), atol=1e-12)


def test_line_integral_variant_is_inert_without_frequency_or_weight():
    s, cam = scenes.small_scene(41, 10, 3)
    base = orc.render_forward(s, cam)["image"]
    v = s.copy(); v.variant = LINE
    assert np.abs(orc.render_forward(v, cam)["image"] - base).max() > 1e-6      # it does something ...
    for mod in ("freqs", "weights"):
        a, b = s.copy(), s.copy()
        getattr(a, mod)[:] = 0
        getattr(b, mod)[:] = 0
        b.variant = LINE
        assert np.array_equal(orc.render_forward(a, cam)["image"], orc.render_forward(b, cam)["image"])   # ... unless f = 0 or w = 0


def test_mip_filter_closed_form():
    s, cam, z, fx = _central_primitive(sc=0.02)          # sigma0^2 = 0.5625 px^2: the filter matters
    s.freqs[0] = [[3.0, 1.0, 5.0], [-2.0, 4.0, -7.0]]
    s.weights[0] = [0.2, 0.1]
    s.variant = MIP
    sc, o = float(s.scales[0, 0]), float(s.opacities[0])
    sig0 = sc * sc * fx * fx / (z * z)
    pr = orc.project(s, cam)
    assert np.isclose(pr["rho"][0], sig0 / (sig0 + 0.1), rtol=1e-12)
    assert pr["radius"][0] == int(np.ceil(3 * np.sqrt(sig0 + 0.1)))
    assert np.allclose(pr["conic"][0], [1 / (sig0 + 0.1), 0, 1 / (sig0 + 0.1)], rtol=1e-12, atol=1e-15)
    out = orc.render_forward(s, cam, literal=True)
    yy, xx = np.mgrid[0:cam.height, 0:cam.width].astype(np.float64)
    dx, dy = xx - cam.cx, yy - cam.cy
    G = np.exp(-(dx * dx + dy * dy) / (2 * (sig0 + 0.1)))
    w = s.weights[0].astype(np.float64)
    M = 1.0 - sum(w[k] * (1 - np.cos(2 * np.pi * (z / fx) * (float(s.freqs[0, k, 0]) * dx + float(s.freqs[0, k, 1]) * dy))) for k in range(2))
    alpha = np.minimum(0.99, o * (sig0 / (sig0 + 0.1)) * G * M)
    inside = (np.abs(dx) <= pr["radius"][0] + 16) & (np.abs(dy) <= pr["radius"][0] + 16)   # its tile rectangle, generously
    alpha[alpha < 1 / 255] = 0
    rgb = 0.5 + K0 * s.sh[0, 0].astype(np.float64)
    want = rgb[:, None, None] * alpha + (1 - alpha) * np.asarray(cam.bg)[:, None, None]
    rect = pr["rect"][0]
    tile = np.zeros_like(inside)
    tile[rect[1] * 16:rect[3] * 16, rect[0] * 16:rect[2] * 16] = True
    assert np.abs(out["image"] - want)[:, tile].max() < 1e-12
    assert np.all(out["n_contrib"][~tile] == 0)


def test_mip_filter_preserves_the_integral_of_the_splat():
    """What the filter is for: rho * 2 pi sqrt(det(U + 0.1 I)) = 2 pi sqrt(det U), the integral of the unfiltered splat."""
    s, cam = _scene(seed=9, N=12, K=1)
    s.variant = MIP
    pr = orc.project(s, cam)
    vis = pr["visible"].astype(bool)
    U = pr["cov2d"][vis]
    detU = U[:, 0] * U[:, 2] - U[:, 1] ** 2
    detD = (U[:, 0] + 0.1) * (U[:, 2] + 0.1) - U[:, 1] ** 2
    assert np.allclose(pr["rho"][vis] ** 2, detU / detD, rtol=1e-12)
    con = pr["conic"][vis]
    assert np.allclose(con[:, 0] * con[:, 2] - con[:, 1] ** 2, 1.0 / detD, rtol=1e-10)
    assert np.allclose(pr["rho"][vis] * np.sqrt(detD), np.sqrt(detU), rtol=1e-12)
    base = s.copy(); base.variant = 0
    assert np.all(orc.project(base, cam)["rho"][vis] == 1.0)


def test_variant_gradients_match_finite_differences():
    for variant, seed in ((LINE, 51), (MIP, 52), (LINE | MIP, 53)):
        s, cam = scenes.small_scene(seed, 10, 3)
        s.freqs *= 3.0                                   # attenuations between ~0.3 and 1
        s.variant = variant
        if variant & LINE:
            att = orc.project(s, cam)["att"]
            assert att.min() < 0.8
        rep, ana = _fd_check(s, cam, seed=seed)
        for name, gname in GROUPS:
            assert np.abs(ana[gname]).max() > 0, (variant, name)


def test_variant_gradients_with_clamped_ray_direction():
    """The attenuation depends on the ray direction, which is the CLAMPED direction of J (reading C15): no gradient
    flows through a clamped coordinate."""
    s, cam = scenes.small_scene(54, 8, 2)
    s.variant = LINE | MIP
    s.means[1] = [3.2, 0.0, 0.5]
    s.scales[1] = 1.5
    pr = orc.project(s, cam)
    t = pr["t"][1]
    assert pr["visible"][1] and abs(t[0] / t[2]) > 1.3 * 0.5 * cam.width / cam.fx
    _fd_check(s, cam, seed=4)
