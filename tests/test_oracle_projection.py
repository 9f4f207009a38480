"""Pins of the oracle's per-primitive projection (oracle/gabsplat_oracle.cpp project_values / twin_index)
against what the paper and the mathematics fix -- nothing here calls the CUDA path.

  * SH basis (reading C22): orthonormal over the sphere by Gauss-Legendre x uniform-azimuth quadrature;
    gradient of the polynomial extension by finite differences.
  * Sigma = R S S^T R^T with scipy's quaternion->matrix as the independent rotation.
  * Eq.2: U = J Sigma_cam J^T with J taken as the FINITE-DIFFERENCE Jacobian of the pinhole
    map, i.e. the "local affine approximation" of PAPER.md:89 computed without writing J down.
  * Eq.16-17: phase invariance f^T(x-mu) = f_proj^T A (x-mu), off axis -- decides the
    transpose of Eq.9 (reading C1).
  * Eq.10-11: f2D independent of the completion of J's third row (reading C2) and equal
    to U^-1 T Sigma f.
  * Eq.18-29: numerical z-quadrature of the ray-space 3D Gabor equals
    const * G2D * cos(2 pi f2D.p), with const = sqrt(2 pi/S22) exp(-2 pi^2 fz^2/S22) (reading C4).
  * On-axis isotropic closed form (reading C21): sigma^2 = s^2 fx^2/z^2, f2D = f_xy z/fx.
"""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import gabsplat_oracle as orc
from paper_2508_05343_b200 import scenes


def _scene(seed=11, N=12, K=3):
    # primitives spread off axis in front of a camera with a general pose
    s, _ = scenes.small_scene(seed, N, K, spread=0.8)
    cam = scenes.make_camera(96, 64, 70.0, scenes.look_at([0.4, -0.3, -3.0], [-0.1, 0.15, 1.0]))
    return s, cam


def _sigma_world(s, i):
    q = s.rotations[i].astype(np.float64)
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()   # scipy is scalar-last
    S = np.diag(s.scales[i].astype(np.float64))
    return R @ S @ S.T @ R.T


def _pinhole(cam, mu):
    Wm = cam.world_to_cam.astype(np.float64)
    t = Wm[:, :3] @ mu + Wm[:, 3]
    return np.array([cam.fx * t[0] / t[2] + cam.cx, cam.fy * t[1] / t[2] + cam.cy]), t


def _fd_T(cam, mu, h=1e-6):
    """d(mu2D)/d(mu): the 2x3 matrix T = J W by central differences of the pinhole map."""
    T = np.zeros((2, 3))
    for a in range(3):
        e = np.zeros(3); e[a] = h
        T[:, a] = (_pinhole(cam, mu + e)[0] - _pinhole(cam, mu - e)[0]) / (2 * h)
    return T


def test_sh_basis_orthonormal_and_gradient():
    n = 24
    x, w = np.polynomial.legendre.leggauss(n)          # cos(theta) nodes
    phi = (np.arange(2 * n) + 0.5) * np.pi / n
    ct, ph = np.meshgrid(x, phi, indexing="ij")
    st = np.sqrt(1 - ct ** 2)
    d = np.stack([st * np.cos(ph), st * np.sin(ph), ct], -1).reshape(-1, 3)
    wt = (w[:, None] * np.full_like(ph, np.pi / n)).reshape(-1)
    Y, _ = orc.sh_basis(d)
    gram = (Y * wt[:, None]).T @ Y
    assert np.abs(gram - np.eye(16)).max() < 1e-12
    # l=1 sign/order convention of reading C22: (-y, z, -x)
    Y1, dY1 = orc.sh_basis(np.array([[0.0, 0.0, 1.0], [1.0, 0, 0], [0, 1.0, 0]]))
    k1 = np.sqrt(3 / (4 * np.pi))
    assert np.allclose(Y1[:, 1:4], k1 * np.array([[0, 1, 0], [0, 0, -1], [-1, 0, 0]]))
    # gradient of the polynomial extension
    rng = np.random.default_rng(0)
    p = rng.normal(size=(5, 3)); p /= np.linalg.norm(p, axis=1, keepdims=True)
    _, dY = orc.sh_basis(p)
    h = 1e-6
    for a in range(3):
        e = np.zeros(3); e[a] = h
        fd = (orc.sh_basis(p + e)[0] - orc.sh_basis(p - e)[0]) / (2 * h)
        assert np.abs(fd - dY[:, :, a]).max() < 1e-8


def test_cov2d_is_fd_jacobian_congruence_and_conic_inverse():
    s, cam = _scene()
    o = orc.project(s, cam)
    assert o["visible"].all()
    for i in range(s.N):
        mu = s.means[i].astype(np.float64)
        m2, t = _pinhole(cam, mu)
        assert np.allclose(o["mean2d"][i], m2, rtol=0, atol=1e-9) and np.allclose(o["t"][i], t, atol=1e-12)
        T = _fd_T(cam, mu)
        U = T @ _sigma_world(s, i) @ T.T
        got = o["cov2d"][i]
        # float32 quaternions are unit only to ~1e-7; scipy renormalises, the ABI does not (reading C20)
        assert np.allclose([U[0, 0], U[0, 1], U[1, 1]], got, rtol=1e-6, atol=2e-6 * np.abs(U).max())
        a, b, c = o["conic"][i]
        Ud = np.array([[got[0] + 0.3, got[1]], [got[1], got[2] + 0.3]])
        assert np.allclose(np.array([[a, b], [b, c]]) @ Ud, np.eye(2), atol=1e-12)
        # float32 twin agrees with the double values to float32 accuracy; depth key is bits(t_z)
        assert np.allclose(o["mean2d_f32"][i], m2, rtol=2e-6, atol=1e-4)
        assert o["depth_bits"][i] == np.float32(o["t"][i][2]).view(np.uint32) or \
            abs(int(o["depth_bits"][i]) - int(np.float32(t[2]).view(np.uint32))) <= 2


def test_phase_invariance_decides_transpose_of_eq9():
    s, cam = _scene()
    rng = np.random.default_rng(3)
    for third in (0, 1, 2):
        o = orc.project(s, cam, third_row=third)
        for i in range(s.N):
            A = o["A3"][i]
            for k in range(s.K):
                f = s.freqs[i, k].astype(np.float64)
                for _ in range(3):
                    dx = rng.normal(size=3)
                    lhs = f @ dx                          # f^T (x - mu)
                    rhs = o["fproj"][i, k] @ (A @ dx)     # f_proj^T (x'' - mu'')
                    assert abs(lhs - rhs) <= 1e-9 * (1 + abs(lhs))
                    wrong = (np.linalg.inv(A) @ f) @ (A @ dx)   # Eq.9 as printed in the main text
                    assert abs(lhs - wrong) > 1e-6 * abs(lhs) or abs(lhs) < 1e-3


def test_freq2d_independent_of_third_row_and_closed_form():
    s, cam = _scene()
    o0, o1, o2 = (orc.project(s, cam, third_row=r) for r in (0, 1, 2))
    scale = np.abs(o0["freq2d"]).max()
    assert np.abs(o0["freq2d"] - o1["freq2d"]).max() < 1e-10 * scale
    assert np.abs(o0["freq2d"] - o2["freq2d"]).max() < 1e-10 * scale
    for i in range(s.N):
        T = _fd_T(cam, s.means[i].astype(np.float64))
        Sg = _sigma_world(s, i)
        U = T @ Sg @ T.T
        for k in range(s.K):
            want = np.linalg.solve(U, T @ Sg @ s.freqs[i, k].astype(np.float64))
            assert np.allclose(o0["freq2d"][i, k], want, rtol=1e-5, atol=1e-5 * scale)


def test_z_quadrature_of_ray_space_gabor():
    s, cam = _scene(seed=5, N=4, K=2)
    o = orc.project(s, cam, third_row=1)
    for i in range(s.N):
        Sig3 = o["Sigma3"][i]
        S = np.linalg.inv(Sig3)
        U = Sig3[:2, :2]
        Ui = np.linalg.inv(U)
        sz = 1.0 / np.sqrt(S[2, 2])
        for k in range(s.K):
            fp = o["fproj"][i, k]
            f2 = o["freq2d"][i, k]
            const = np.sqrt(2 * np.pi / S[2, 2]) * np.exp(-2 * np.pi ** 2 * fp[2] ** 2 / S[2, 2])
            sd = np.sqrt(np.diag(U))
            for p in (np.array([0.3, -0.2]) * sd, np.array([-0.7, 0.5]) * sd, np.array([0.0, 0.0])):
                zc = -(S[0, 2] * p[0] + S[1, 2] * p[1]) / S[2, 2]
                z = zc + np.linspace(-12, 12, 48001) * sz
                X = np.stack([np.full_like(z, p[0]), np.full_like(z, p[1]), z], 1)
                g = np.exp(-0.5 * np.einsum("na,ab,nb->n", X, S, X)) * np.cos(2 * np.pi * X @ fp)
                integral = g.sum() * (z[1] - z[0])      # integrand is ~0 at both ends; rectangle rule is spectral
                want = const * np.exp(-0.5 * p @ Ui @ p) * np.cos(2 * np.pi * f2 @ p)
                assert abs(integral - want) <= 1e-7 * const + 1e-12


def test_on_axis_isotropic_closed_form():
    z, fx, sc = 5.0, 120.0, 0.07
    s, _ = scenes.small_scene(1, 1, 3)
    s.means[:] = [0, 0, 1.0]
    s.scales[:] = sc
    s.rotations[:] = [1, 0, 0, 0]
    cam = scenes.make_camera(65, 65, fx, scenes.look_at([0, 0, 1.0 - z], [0, 0, 1.0]))
    o = orc.project(s, cam)
    sig2 = float(np.float32(sc)) ** 2 * fx ** 2 / z ** 2
    assert np.allclose(o["cov2d"][0], [sig2, 0, sig2], rtol=1e-12, atol=1e-12)
    assert np.allclose(o["mean2d"][0], [32, 32])
    assert np.allclose(o["freq2d"][0], s.freqs[0, :, :2].astype(np.float64) * z / fx, rtol=1e-10)
    lam = sig2 + 0.3
    assert o["radius"][0] == int(np.ceil(3 * np.sqrt(lam)))


def test_culling_behind_camera_and_z_near():
    s, cam = _scene()
    s.means[0] = [0.4, -0.3, -3.0 - 1.0]     # behind
    Wm = cam.world_to_cam.astype(np.float64)
    o = orc.project(s, cam)
    assert o["visible"][0] == 0 and o["tiles_touched"][0] == 0
    t = Wm[:, :3] @ s.means.astype(np.float64).T + Wm[:, 3:4]
    assert np.array_equal(o["visible"][1:] != 0, (t[2, 1:] > cam.z_near) & (o["tiles_touched"][1:] > 0))
