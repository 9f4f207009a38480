"""ORACLE -- TEST INFRASTRUCTURE ONLY (see gabsplat_oracle.cpp for what it computes and its pins).

ctypes wrapper around ``oracle/liboracle_gabsplat.so`` (built by ``oracle/build.py`` with g++).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this module.  It imports nothing from the CUDA path; scenes and cameras are
duck-typed (any object with the attribute names of ``paper_2508_05343_b200.scenes``).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np

VARIANT_LINE_INTEGRAL, VARIANT_MIP_FILTER = 1, 2     # scene.variant bit flags

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle_gabsplat.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "gabsplat_oracle.cpp")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        subprocess.check_call([sys.executable, os.path.join(_HERE, "build.py")])
    return _LIB_PATH


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB_PATH)
        _lib.orc_bin.restype = C.c_uint64
        _lib.orc_max_threads.restype = C.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def cam_vector(cam) -> np.ndarray:
    v = np.zeros(22, np.float64)
    v[0], v[1] = cam.width, cam.height
    v[2:6] = [cam.fx, cam.fy, cam.cx, cam.cy]
    v[6:18] = np.asarray(cam.world_to_cam, np.float64).reshape(12)
    v[18] = cam.z_near
    v[19:22] = cam.bg
    return v


def _scene_args(scene):
    arrs = [np.ascontiguousarray(a, np.float32) for a in
            (scene.means, scene.scales, scene.rotations, scene.opacities, scene.sh, scene.freqs, scene.weights)]
    deg = int(scene.sh_degree) | (int(getattr(scene, "variant", 0)) << 8)     # variant flags ride in the second byte
    return arrs, [C.c_int(scene.N), C.c_int(scene.K), C.c_int(deg)] + [_p(a) for a in arrs]


def max_threads() -> int:
    return int(lib().orc_max_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(C.c_int(n))


def sh_basis(dirs):
    d = np.ascontiguousarray(dirs, np.float64).reshape(-1, 3)
    Y = np.zeros((d.shape[0], 16))
    dY = np.zeros((d.shape[0], 16, 3))
    lib().orc_sh_basis(C.c_int(d.shape[0]), _p(d), _p(Y), _p(dY))
    return Y, dY


def project(scene, cam, third_row: int = 0) -> dict:
    N, K = scene.N, scene.K
    keep, args = _scene_args(scene)
    cv = cam_vector(cam)
    o = dict(
        visible=np.zeros(N, np.uint8), t=np.zeros((N, 3)), mean2d=np.zeros((N, 2)), cov2d=np.zeros((N, 3)),
        conic=np.zeros((N, 3)), freq2d=np.zeros((N, K, 2)), rgb=np.zeros((N, 3)), clamped=np.zeros((N, 3), np.uint8),
        depth_bits=np.zeros(N, np.uint32), mean2d_f32=np.zeros((N, 2), np.float32), radius=np.zeros(N, np.int32),
        rect=np.zeros((N, 4), np.int32), tiles_touched=np.zeros(N, np.uint32),
        A3=np.zeros((N, 3, 3)), fproj=np.zeros((N, K, 3)), Sigma3=np.zeros((N, 3, 3)),
        att=np.zeros((N, K)), rho=np.zeros(N))
    lib().orc_project(*args, _p(cv), C.c_int(third_row), *[_p(o[k]) for k in (
        "visible", "t", "mean2d", "cov2d", "conic", "freq2d", "rgb", "clamped", "depth_bits", "mean2d_f32",
        "radius", "rect", "tiles_touched", "A3", "fproj", "Sigma3", "att", "rho")])
    return o


def bin_sort(scene, cam, brute: bool = False) -> dict:
    keep, args = _scene_args(scene)
    cv = cam_vector(cam)
    D = int(lib().orc_bin(*args, _p(cv), C.c_int(0 if brute else 1), C.c_uint64(0), None, None, None))
    keys = np.zeros(max(D, 1), np.uint64)
    ids = np.zeros(max(D, 1), np.uint32)
    ranges = np.zeros((cam.tiles_x * cam.tiles_y, 2), np.uint32)
    lib().orc_bin(*args, _p(cv), C.c_int(0 if brute else 1), C.c_uint64(max(D, 1)), _p(keys), _p(ids), _p(ranges))
    return dict(num_instances=D, keys=keys[:D], ids=ids[:D], tile_ranges=ranges)


def render_forward(scene, cam, literal: bool = False) -> dict:
    keep, args = _scene_args(scene)
    cv = cam_vector(cam)
    H, W = cam.height, cam.width
    o = dict(image=np.zeros((3, H, W)), final_T=np.zeros((H, W)), n_contrib=np.zeros((H, W), np.uint32),
             last_id=np.zeros((H, W), np.int32), counters=np.zeros((H, W, 3), np.uint32), margin=np.zeros((H, W, 2)))
    lib().orc_render_forward(*args, _p(cv), C.c_int(1 if literal else 0), *[_p(o[k]) for k in (
        "image", "final_T", "n_contrib", "last_id", "counters", "margin")])
    return o


def render_aux(scene, cam) -> dict:
    """Auxiliary renders: image[0] = blended sum_k omega_k |f2D_k|, image[1] = blended depth, image[2] = accumulated alpha."""
    keep, args = _scene_args(scene)
    cv = cam_vector(cam)
    H, W = cam.height, cam.width
    o = dict(image=np.zeros((3, H, W)), final_T=np.zeros((H, W)))
    lib().orc_render_aux(*args, _p(cv), _p(o["image"]), _p(o["final_T"]))
    return o


def render_pixels(scene, cam, pixels) -> dict:
    keep, args = _scene_args(scene)
    cv = cam_vector(cam)
    px = np.ascontiguousarray(pixels, np.int32).reshape(-1, 2)
    n = px.shape[0]
    o = dict(colour=np.zeros((n, 3)), final_T=np.zeros(n), n_contrib=np.zeros(n, np.uint32),
             last_id=np.zeros(n, np.int32), margin=np.zeros((n, 2)))
    lib().orc_render_pixels(*args, _p(cv), C.c_int(n), _p(px), *[_p(o[k]) for k in (
        "colour", "final_T", "n_contrib", "last_id", "margin")])
    return o


def trace_pixels(scene, cam, pixels, max_entries: int = 4096) -> dict:
    """The oracle's own blend decisions at the pixels [n][2] (x, y), in the format render_backward's `inject` takes."""
    keep, args = _scene_args(scene)
    cv = cam_vector(cam)
    px = np.ascontiguousarray(pixels, np.int32).reshape(-1, 2)
    n = px.shape[0]
    off = (np.arange(n + 1, dtype=np.uint64) * max_entries).astype(np.uint32)
    ent = np.zeros(max(1, n * max_entries), np.uint32)
    counts = np.zeros(n, np.uint32)
    stop = np.zeros(n, np.uint32)
    lib().orc_trace_pixels(*args, _p(cv), C.c_int(n), _p(px), _p(off), _p(ent), _p(counts), _p(stop))
    assert n == 0 or counts.max() <= max_entries
    # compact to CSR
    offsets = np.zeros(n + 1, np.uint32)
    offsets[1:] = np.cumsum(counts)
    entries = np.concatenate([ent[off[k]:off[k] + counts[k]] for k in range(n)]) if n else np.zeros(0, np.uint32)
    return dict(pixels=px, offsets=offsets, entries=entries.astype(np.uint32), stop_pos=stop, counts=counts)


def render_backward(scene, cam, dL_dimage, inject: dict | None = None) -> dict:
    """Forward + analytic backward.  `inject` (decision-injected mode, reading C18): dict with
    pixels [n][2] int32 (x, y), offsets [n+1] uint32, entries uint32 (1-based list positions of the blended
    entries, bit 31 = clamp active), stop_pos [n] uint32, delta (relative margin).  The result then carries
    `violations`: the number of injected outcomes that are not correct renderings within delta (must be 0)."""
    keep, args = _scene_args(scene)
    cv = cam_vector(cam)
    N, K, H, W = scene.N, scene.K, cam.height, cam.width
    g = np.ascontiguousarray(dL_dimage, np.float32)
    assert g.shape == (3, H, W)
    o = dict(image=np.zeros((3, H, W)), final_T=np.zeros((H, W)), n_contrib=np.zeros((H, W), np.uint32),
             d_means=np.zeros((N, 3)), d_scales=np.zeros((N, 3)),
             d_rotations=np.zeros((N, 4)), d_opacities=np.zeros(N), d_sh=np.zeros((N, 16, 3)),
             d_freqs=np.zeros((N, K, 3)), d_weights=np.zeros((N, K)), d_mean2d=np.zeros((N, 2)),
             d_conic=np.zeros((N, 3)), d_rgb=np.zeros((N, 3)), d_freq2d=np.zeros((N, K, 2)),
             d_absmean2d=np.zeros((N, 2)))
    viol = np.zeros(1, np.uint64)
    if inject is not None and len(inject["pixels"]):
        px = np.ascontiguousarray(inject["pixels"], np.int32).reshape(-1, 2)
        off = np.ascontiguousarray(inject["offsets"], np.uint32)
        ent = np.ascontiguousarray(inject["entries"], np.uint32)
        stop = np.ascontiguousarray(inject["stop_pos"], np.uint32)
        assert off.shape == (px.shape[0] + 1,) and stop.shape == (px.shape[0],) and ent.size >= int(off[-1])
        assert np.all(px[:, 0] >= 0) and np.all(px[:, 0] < W) and np.all(px[:, 1] >= 0) and np.all(px[:, 1] < H)
        inj = [C.c_int(px.shape[0]), _p(px), _p(off), _p(ent), _p(stop), C.c_double(float(inject["delta"])), _p(viol)]
    else:
        inj = [C.c_int(0), None, None, None, None, C.c_double(0.0), _p(viol)]
    lib().orc_render_backward_ex(*args, _p(cv), _p(g), *[_p(o[k]) for k in (
        "image", "final_T", "n_contrib", "d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs",
        "d_weights", "d_mean2d", "d_conic", "d_rgb", "d_freq2d", "d_absmean2d")], *inj)
    o["violations"] = int(viol[0])
    return o
