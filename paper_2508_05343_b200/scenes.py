"""Seeded synthetic scenes, cameras and image gradients for the 3DGabSplat rasterizer.

This module holds NONE of the method's arithmetic (no projection, no blending): it only
draws the inputs that both the CPU oracle (``oracle/``) and the CUDA path consume, so that
the two sides see bit-identical float32 arrays.  The recipes are the BASELINE.json configs
(concretised in SURVEY.md section 8(d), restated in DESIGN.md "Input recipe"); they stand
in for the paper's datasets (PAPER.md:183, :232 -- Mip-NeRF 360 / NeRF-Synthetic shaped),
which are not available here.

Random numbers come from a hand-written counter-based SplitMix64 (uniforms) and Box-Muller
(normals), vectorised with numpy, so any language can regenerate the same streams.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
BASE_SEED = 20250805  # seed = BASE_SEED + 1000*config + view


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


class Stream:
    """Counter-based SplitMix64: output i of stream (seed, name_id) = mix(s0 + (i+1)*GAMMA)."""

    def __init__(self, seed: int, stream_id: int):
        with np.errstate(over="ignore"):
            s = _mix(np.array([np.uint64(seed) * _GAMMA + np.uint64(stream_id) * _M1], dtype=np.uint64))
        self.s0 = s[0]
        self.pos = 0

    def u64(self, n: int) -> np.ndarray:
        with np.errstate(over="ignore"):
            idx = np.arange(self.pos + 1, self.pos + n + 1, dtype=np.uint64)
            out = _mix(self.s0 + idx * _GAMMA)
        self.pos += n
        return out

    def uniform(self, n: int) -> np.ndarray:
        """float64 in [0,1) with 53 random bits."""
        return (self.u64(n) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)

    def normal(self, n: int) -> np.ndarray:
        """float64 standard normals by Box-Muller (cosine branch), two uniforms per normal."""
        u = self.uniform(2 * n)
        u1, u2 = u[0::2], u[1::2]
        return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)


@dataclass
class Scene:
    """Activated primitive parameters, float32, C-contiguous."""
    means: np.ndarray       # [N,3]
    scales: np.ndarray      # [N,3]   > 0 (already exp'ed)
    rotations: np.ndarray   # [N,4]   unit quaternion (w,x,y,z)
    opacities: np.ndarray   # [N]     in (0,1)
    sh: np.ndarray          # [N,16,3]
    freqs: np.ndarray       # [N,K,3] cycles per world unit
    weights: np.ndarray     # [N,K]   in [0,1)
    sh_degree: int = 3
    variant: int = 0        # primitive variant flags (gabsplat.h GABSPLAT_VARIANT_*): 1 line-integral amplitude, 2 Mip filter

    @property
    def N(self) -> int:
        return int(self.means.shape[0])

    @property
    def K(self) -> int:
        return int(self.freqs.shape[1])

    def copy(self) -> "Scene":
        return Scene(*(a.copy() for a in (self.means, self.scales, self.rotations, self.opacities,
                                           self.sh, self.freqs, self.weights)), sh_degree=self.sh_degree,
                     variant=self.variant)


@dataclass
class Camera:
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    world_to_cam: np.ndarray            # [3,4] float32 row-major [W|tau]: t = W mu + tau
    z_near: float = 0.2
    bg: tuple = (0.0, 0.0, 0.0)

    @property
    def tiles_x(self) -> int:
        return (self.width + 15) // 16

    @property
    def tiles_y(self) -> int:
        return (self.height + 15) // 16


def look_at(pos, forward) -> np.ndarray:
    """Rows of W are (right, down, forward) with up=(0,1,0); tau = -W pos.  float32 [3,4]."""
    pos = np.asarray(pos, np.float64)
    fwd = np.asarray(forward, np.float64)
    fwd = fwd / np.linalg.norm(fwd)
    up = np.array([0.0, 1.0, 0.0])
    right = np.cross(up, fwd)
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    W = np.stack([right, down, fwd])
    tau = -W @ pos
    return np.concatenate([W, tau[:, None]], axis=1).astype(np.float32)


def make_camera(width, height, f, world_to_cam, bg=(0.0, 0.0, 0.0)) -> Camera:
    f32 = np.float32
    return Camera(int(width), int(height), float(f32(f)), float(f32(f)),
                  float(f32((width - 1) / 2.0)), float(f32((height - 1) / 2.0)),
                  np.ascontiguousarray(world_to_cam, dtype=np.float32), float(f32(0.2)),
                  tuple(float(f32(b)) for b in bg))


def _common_attributes(seed: int, N: int, K: int, log_scale_mu: float, log_scale_sigma: float):
    """Everything except the means (same distributions in every config)."""
    f32 = np.float32
    scales = np.exp(log_scale_mu + log_scale_sigma * Stream(seed, 2).normal(3 * N)).reshape(N, 3)
    q = Stream(seed, 3).normal(4 * N).reshape(N, 4)
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    opac = 1.0 / (1.0 + np.exp(-Stream(seed, 4).normal(N)))
    sh = 0.3 * Stream(seed, 5).normal(48 * N).reshape(N, 16, 3)
    d = Stream(seed, 6).normal(3 * N * max(K, 1)).reshape(N, max(K, 1), 3)[:, :K]
    d = d / np.maximum(np.linalg.norm(d, axis=2, keepdims=True), 1e-300)
    mag = 8.0 * Stream(seed, 7).uniform(N * max(K, 1)).reshape(N, max(K, 1), 1)[:, :K]
    freqs = d * mag
    weights = Stream(seed, 8).uniform(N * max(K, 1)).reshape(N, max(K, 1))[:, :K]
    # renormalise quaternions after the float32 cast is NOT done: the ABI takes them as given.
    return (np.ascontiguousarray(scales, f32), np.ascontiguousarray(q, f32),
            np.ascontiguousarray(np.clip(opac, 1e-6, 1 - 1e-6), f32), np.ascontiguousarray(sh, f32),
            np.ascontiguousarray(freqs, f32).reshape(N, K, 3),
            np.ascontiguousarray(np.minimum(weights, 1 - 2.0 ** -24), f32).reshape(N, K))


def _means_box(seed, N):
    return 2.0 * Stream(seed, 1).uniform(3 * N).reshape(N, 3) - 1.0


def _means_ball(seed, N):
    d = Stream(seed, 1).normal(3 * N).reshape(N, 3)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    r = Stream(seed, 9).uniform(N) ** (1.0 / 3.0)
    return d * r[:, None]


def _means_unbounded(seed, N):
    n_in = int(round(0.7 * N))
    inner = Stream(seed, 1).normal(3 * n_in).reshape(n_in, 3) * np.array([3.0, 1.0, 3.0])
    n_out = N - n_in
    d = Stream(seed, 9).normal(3 * n_out).reshape(n_out, 3)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    r = 20.0 + 30.0 * Stream(seed, 10).uniform(n_out)
    return np.concatenate([inner, d * r[:, None]], axis=0)


CONFIGS = {
    # name: (config index, N, K, means fn, log-scale mu, sigma, W, H, focal, bg, n_views)
    "tiny":      (1, 1024,      4, _means_box,       -3.0, 0.5, 128,  128,  150.0,  (0, 0, 0), 1),
    "object":    (2, 300_000,   4, _means_ball,      -4.5, 0.7, 800,  800,  1111.0, (1, 1, 1), 8),
    "unbounded": (3, 1_000_000, 4, _means_unbounded, -4.0, 1.0, 1297, 840,  1150.0, (0, 0, 0), 8),
    "large":     (4, 3_000_000, 4, _means_unbounded, -4.5, 1.2, 1957, 1266, 1700.0, (0, 0, 0), 8),
}


def config_seed(name: str, view: int = 0) -> int:
    return BASE_SEED + 1000 * CONFIGS[name][0] + view


def make_scene(name: str, K: int | None = None, N: int | None = None, zero_weights: bool = False) -> Scene:
    """Scene of a BASELINE.json config.  ``K`` overrides the filter-bank size (config 5, the K
    sweep, is ``make_scene('unbounded', K=k)``; its all-zero-weight case sets ``zero_weights``).
    ``N`` overrides the primitive count (reduced-size parity cases keep the distributions)."""
    idx, N0, K0, means_fn, mu, sigma, *_ = CONFIGS[name]
    N = N0 if N is None else int(N)
    K = K0 if K is None else int(K)
    seed = BASE_SEED + 1000 * idx
    means = np.ascontiguousarray(means_fn(seed, N), np.float32)
    scales, q, opac, sh, freqs, weights = _common_attributes(seed, N, K, mu, sigma)
    if zero_weights:
        weights = np.zeros_like(weights)
    return Scene(means, scales, q, opac, sh, freqs, weights, 3)


def make_cameras(name: str) -> list[Camera]:
    idx, _, _, _, _, _, W, H, f, bg, n_views = CONFIGS[name]
    seed = BASE_SEED + 1000 * idx
    cams = []
    if name == "tiny":
        cams.append(make_camera(W, H, f, look_at([0, 0, -4.0], [0, 0, 1.0]), bg))
    elif name == "object":
        d = Stream(seed, 20).normal(3 * n_views).reshape(n_views, 3)
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        for v in range(n_views):
            pos = 4.0 * d[v]
            cams.append(make_camera(W, H, f, look_at(pos, -pos), bg))
    else:
        p = np.clip(Stream(seed, 20).normal(3 * n_views).reshape(n_views, 3), -2, 2) * 0.5 * np.array([3.0, 1.0, 3.0])
        az = 2 * np.pi * Stream(seed, 21).uniform(n_views)
        el = np.deg2rad(-10.0 + 20.0 * Stream(seed, 22).uniform(n_views))
        for v in range(n_views):
            fwd = [np.cos(el[v]) * np.sin(az[v]), np.sin(el[v]), np.cos(el[v]) * np.cos(az[v])]
            cams.append(make_camera(W, H, f, look_at(p[v], fwd), bg))
    return cams


def make_image_grad(name: str, view: int, cam: Camera) -> np.ndarray:
    """dL/dimage ~ N(0,1) i.i.d., planar [3,H,W] float32."""
    g = Stream(config_seed(name, view), 30).normal(3 * cam.height * cam.width)
    return np.ascontiguousarray(g.reshape(3, cam.height, cam.width), np.float32)


def small_scene(seed: int, N: int, K: int, size: int = 16, f: float = 40.0, spread: float = 0.15,
                log_scale=(-2.6, 0.3)) -> tuple[Scene, Camera]:
    """A few primitives in front of a one-tile camera: finite-difference and unit-test scenes."""
    scales, q, opac, sh, freqs, weights = _common_attributes(seed, N, K, log_scale[0], log_scale[1])
    means = (2.0 * Stream(seed, 1).uniform(3 * N).reshape(N, 3) - 1.0) * spread
    freqs = freqs * np.float32(0.25)
    cam = make_camera(size, size, f, look_at([0.02, -0.03, -3.0], [0.01, 0.02, 1.0]))
    return Scene(np.ascontiguousarray(means, np.float32), scales, q, opac, sh, freqs, weights, 3), cam
