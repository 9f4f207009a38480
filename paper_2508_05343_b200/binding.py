"""Thin ctypes binding of libgabsplat.so (include/gabsplat.h).  Argument marshalling only: every step of
the path runs in the library's CUDA kernels.  torch is used for device memory and streams.

The functions carry the names of the C entry points (gabsplat_preprocess, gabsplat_bin_sort,
gabsplat_render_forward, gabsplat_render_backward, gabsplat_render_host).  There is no fallback:
importing this module without the built library, or creating a Context without a B200, raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgabsplat.so")

OK, INVALID_ARG, CAPACITY, CUDA_ERROR, UNSUPPORTED = 0, 1, 2, 3, 4
CHUNK = 1024   # GABSPLAT_CHUNK
TILE = 16


class GabsplatError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("libgabsplat status %d: %s" % (code, msg))
        self.code = code


class _Camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("world_to_cam", C.c_float * 12), ("z_near", C.c_float),
                ("bg", C.c_float * 3)]


class _Scene(C.Structure):
    _fields_ = [("N", C.c_int32), ("K", C.c_int32), ("sh_degree", C.c_int32), ("variant", C.c_int32)] + [
        (n, C.c_void_p) for n in ("means", "scales", "rotations", "opacities", "sh", "freqs", "weights")]


class _Projected(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("mean2d", "depth", "radius", "conic_opacity", "rgb", "rgb_clamped",
                                          "freq2d", "tiles_touched", "rect", "packed", "chunk_visible")]


class _Binning(C.Structure):
    _fields_ = [("offsets", C.c_void_p), ("keys", C.c_void_p), ("ids", C.c_void_p), ("tile_ranges", C.c_void_p),
                ("tile_order", C.c_void_p), ("capacity", C.c_uint64), ("num_instances", C.c_void_p), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_uint64), ("tile_work_hint", C.c_void_p)]


class _FwdOut(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("image", "final_T", "n_contrib", "blend_state")] + [
        ("blend_state_bytes", C.c_uint64), ("tile_work", C.c_void_p)]


class _Grads(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs",
                                          "d_weights", "d_mean2d", "d_mean2d_abs")]


_lib = None


def lib():
    """The loaded library; raises if it has not been built (python -m paper_2508_05343_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libgabsplat.so is not built: run `python -m paper_2508_05343_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.gabsplat_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32]
        L.gabsplat_create.restype = C.c_int32
        L.gabsplat_destroy.argtypes = [C.c_void_p]
        L.gabsplat_destroy.restype = None
        L.gabsplat_last_error.argtypes = [C.c_void_p]
        L.gabsplat_last_error.restype = C.c_char_p
        L.gabsplat_packed_floats.argtypes = [C.c_int32]
        L.gabsplat_packed_floats.restype = C.c_int32
        L.gabsplat_sort_workspace_bytes.argtypes = [C.c_int32, C.c_uint64, C.c_int32, C.c_int32]
        L.gabsplat_sort_workspace_bytes.restype = C.c_uint64
        L.gabsplat_blend_state_bytes.argtypes = [C.c_int32, C.c_int32, C.c_uint64]
        L.gabsplat_blend_state_bytes.restype = C.c_uint64
        L.gabsplat_grad_workspace_bytes.argtypes = [C.c_int32, C.c_int32]
        L.gabsplat_grad_workspace_bytes.restype = C.c_uint64
        L.gabsplat_host_arena_bytes.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_uint64]
        L.gabsplat_host_arena_bytes.restype = C.c_uint64
        P = C.c_void_p
        L.gabsplat_preprocess.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.POINTER(_Projected), P]
        L.gabsplat_bin_sort.argtypes = [P, C.c_int32, C.POINTER(_Projected), C.POINTER(_Camera), C.POINTER(_Binning),
                                        C.POINTER(C.c_uint64), P]
        L.gabsplat_preprocess_bin_sort.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.POINTER(_Projected),
                                                   C.POINTER(_Binning), C.POINTER(C.c_uint64), P]
        L.gabsplat_preprocess_bin_sort.restype = C.c_int32
        L.gabsplat_render_forward.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.POINTER(_Projected),
                                              C.POINTER(_Binning), C.POINTER(_FwdOut), P]
        L.gabsplat_render_backward.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.POINTER(_Projected),
                                               C.POINTER(_Binning), C.POINTER(_FwdOut), P, C.POINTER(_Grads), P,
                                               C.c_uint64, P]
        L.gabsplat_render_host.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.c_uint64, P, P,
                                           C.POINTER(_Grads), P, C.c_uint64, P]
        L.gabsplat_aux_workspace_bytes.argtypes = [C.c_int32, C.c_int32, C.c_int32]
        L.gabsplat_aux_workspace_bytes.restype = C.c_uint64
        L.gabsplat_render_aux.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.POINTER(_Projected),
                                          C.POINTER(_Binning), P, P, C.c_uint64, P]
        L.gabsplat_render_aux.restype = C.c_int32
        L.gabsplat_chunk_visible_count.argtypes = [C.c_int32]
        L.gabsplat_chunk_visible_count.restype = C.c_uint64
        L.gabsplat_loss_workspace_bytes.argtypes = [C.c_int32, C.c_int32]
        L.gabsplat_loss_workspace_bytes.restype = C.c_uint64
        L.gabsplat_loss.argtypes = [P, C.c_int32, C.c_int32, P, P, C.c_float, P, P, P, C.c_uint64, P]
        L.gabsplat_loss.restype = C.c_int32
        L.gabsplat_loss_static_max_pixels.argtypes = []
        L.gabsplat_loss_static_max_pixels.restype = C.c_uint64
        L.gabsplat_loss_static_last_error.argtypes = []
        L.gabsplat_loss_static_last_error.restype = C.c_char_p
        L.gabsplat_loss_static.argtypes = [C.c_int32, C.c_int32, P, P, C.c_float, P, P, P]
        L.gabsplat_loss_static.restype = C.c_int32
        L.gabsplat_kernel_launches.argtypes = []
        L.gabsplat_kernel_launches.restype = C.c_uint64
        L.gabsplat_timing_enable.argtypes = [P, C.c_int32]
        L.gabsplat_timing_read.argtypes = [P, C.POINTER(C.c_int32), C.POINTER(C.c_float), C.c_int32,
                                           C.POINTER(C.c_int32)]
        L.gabsplat_count_pairs.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.POINTER(_Projected),
                                           C.POINTER(_Binning), P, P]
        L.gabsplat_trace_pixels.argtypes = [P, C.POINTER(_Scene), C.POINTER(_Camera), C.POINTER(_Projected),
                                            C.POINTER(_Binning), C.c_int32, P, P, P, P, P, P]
        L.gabsplat_trace_pixels.restype = C.c_int32
        L.gabsplat_probe_sincos.argtypes = [P, C.c_int32, P, P, P, P]
        L.gabsplat_probe_sincos.restype = C.c_int32
        L.gabsplat_set_place_bands.argtypes = [P, C.c_int32]
        L.gabsplat_set_place_bands.restype = C.c_int32
        L.gabsplat_measure_peaks.argtypes = [P, C.POINTER(C.c_float), P]
        L.gabsplat_measure_peaks.restype = C.c_int32
        for f in (L.gabsplat_preprocess, L.gabsplat_bin_sort, L.gabsplat_render_forward, L.gabsplat_render_backward,
                  L.gabsplat_render_host, L.gabsplat_timing_enable, L.gabsplat_timing_read, L.gabsplat_count_pairs):
            f.restype = C.c_int32
        _lib = L
    return _lib


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream) -> C.c_void_p:
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def camera_struct(cam) -> _Camera:
    c = _Camera()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = cam.fx, cam.fy, cam.cx, cam.cy
    w = np.asarray(cam.world_to_cam, np.float32).reshape(12)
    for i in range(12):
        c.world_to_cam[i] = float(w[i])
    c.z_near = cam.z_near
    for i in range(3):
        c.bg[i] = float(cam.bg[i])
    return c


class Context:
    """gabsplat_ctx bound to one CUDA device."""

    def __init__(self, device: int = 0):
        self._h = C.c_void_p()
        rc = lib().gabsplat_create(C.byref(self._h), device)
        if rc != OK:
            raise GabsplatError(rc, "gabsplat_create failed (needs an sm_100 device; there is no CPU fallback)")
        self.device = torch.device("cuda", device)

    def check(self, rc: int) -> None:
        if rc != OK:
            raise GabsplatError(rc, lib().gabsplat_last_error(self._h).decode())

    def close(self) -> None:
        if self._h:
            lib().gabsplat_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


@dataclass
class DeviceScene:
    """The primitives in device memory (float32, contiguous; layouts of gabsplat_scene)."""
    means: torch.Tensor
    scales: torch.Tensor
    rotations: torch.Tensor
    opacities: torch.Tensor
    sh: torch.Tensor
    freqs: torch.Tensor
    weights: torch.Tensor
    sh_degree: int = 3
    variant: int = 0        # GABSPLAT_VARIANT_* flags

    @property
    def N(self) -> int:
        return int(self.means.shape[0])

    @property
    def K(self) -> int:
        return int(self.freqs.shape[1])

    def struct(self) -> _Scene:
        s = _Scene()
        s.N, s.K, s.sh_degree, s.variant = self.N, self.K, self.sh_degree, int(self.variant)
        for n in ("means", "scales", "rotations", "opacities", "sh", "freqs", "weights"):
            t = getattr(self, n)
            assert t.dtype == torch.float32 and t.is_contiguous()
            setattr(s, n, t.data_ptr() if t.numel() else None)
        return s


def upload_scene(scene, device="cuda:0") -> DeviceScene:
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(device)
    return DeviceScene(f(scene.means), f(scene.scales), f(scene.rotations), f(scene.opacities), f(scene.sh),
                       f(scene.freqs), f(scene.weights), scene.sh_degree, int(getattr(scene, "variant", 0)))


class Projected:
    """Device buffers of gabsplat_projected for N primitives, K components."""

    def __init__(self, N: int, K: int, device):
        z = lambda shape, dt: torch.zeros(shape, dtype=dt, device=device)
        self.N, self.K = N, K
        self.mean2d = z((N, 2), torch.float32)
        self.depth = z((N,), torch.float32)
        self.radius = z((N,), torch.int32)
        self.conic_opacity = z((N, 4), torch.float32)
        self.rgb = z((N, 3), torch.float32)
        self.rgb_clamped = z((N, 4), torch.uint8)
        self.freq2d = z((N, K, 2), torch.float32)
        self.tiles_touched = z((N,), torch.int32)  # uint32 on the device; torch has no uint32 arithmetic
        self.rect = z((N, 4), torch.int32)
        self.packed = z((N, lib().gabsplat_packed_floats(K)), torch.float32)
        self.chunk_visible = z((int(lib().gabsplat_chunk_visible_count(N)),), torch.int32)

    def struct(self) -> _Projected:
        p = _Projected()
        for n, _ in _Projected._fields_:
            t = getattr(self, n)
            setattr(p, n, t.data_ptr() if t.numel() else None)
        return p


class Binning:
    """Device buffers of gabsplat_binning for N primitives and `capacity` instances."""

    def __init__(self, N: int, cam, capacity: int, device, with_keys: bool = True):
        z = lambda shape, dt: torch.zeros(shape, dtype=dt, device=device)
        self.N, self.capacity = N, int(capacity)
        self.n_tiles = ((cam.width + TILE - 1) // TILE) * ((cam.height + TILE - 1) // TILE)
        self.offsets = z((max(N, 1),), torch.int32)
        self.keys = z((max(self.capacity, 1),), torch.int64) if with_keys else None
        self.ids = z((max(self.capacity, 1),), torch.int32)
        self.tile_ranges = z((self.n_tiles, 2), torch.int32)
        self.tile_order = z((self.n_tiles,), torch.int32)
        self.num_instances = z((4,), torch.int32)
        self.workspace_bytes = int(lib().gabsplat_sort_workspace_bytes(N, self.capacity, cam.width, cam.height))
        self.workspace = z((self.workspace_bytes + 256,), torch.uint8)
        self.D = None  # host copy of the instance count when the call read it back
        self.tile_work_hint = None  # optional int32 [n_tiles]: FwdOut.tile_work of an earlier render of the view

    def struct(self) -> _Binning:
        b = _Binning()
        b.offsets, b.ids = self.offsets.data_ptr(), self.ids.data_ptr()
        b.keys = self.keys.data_ptr() if self.keys is not None else None
        b.tile_ranges = self.tile_ranges.data_ptr()
        b.tile_order = self.tile_order.data_ptr()
        b.capacity = self.capacity
        b.num_instances = self.num_instances.data_ptr()
        b.workspace = (self.workspace.data_ptr() + 255) // 256 * 256
        b.workspace_bytes = self.workspace_bytes
        b.tile_work_hint = self.tile_work_hint.data_ptr() if self.tile_work_hint is not None else None
        return b


class FwdOut:
    """capacity = the binning's instance capacity allocates the blend state the backward replays;
    capacity=None is inference mode (gabsplat_render_backward then refuses this output)."""

    def __init__(self, cam, device, capacity: int | None = None):
        H, W = cam.height, cam.width
        self.image = torch.zeros((3, H, W), dtype=torch.float32, device=device)
        self.final_T = torch.zeros((H, W), dtype=torch.float32, device=device)
        self.n_contrib = torch.zeros((H, W), dtype=torch.int32, device=device)
        self.blend_state = None
        self.blend_state_bytes = 0
        self.tile_work = None   # optional int32 [n_tiles] output: list entries every tile consumed (the next render's hint)
        if capacity is not None:
            self.blend_state_bytes = int(lib().gabsplat_blend_state_bytes(W, H, int(capacity)))
            self.blend_state = torch.empty((self.blend_state_bytes,), dtype=torch.uint8, device=device)

    def struct(self, save_state: bool = True) -> _FwdOut:
        o = _FwdOut()
        o.image, o.final_T, o.n_contrib = self.image.data_ptr(), self.final_T.data_ptr(), self.n_contrib.data_ptr()
        o.tile_work = self.tile_work.data_ptr() if self.tile_work is not None else None
        if save_state and self.blend_state is not None:
            o.blend_state, o.blend_state_bytes = self.blend_state.data_ptr(), self.blend_state_bytes
        else:
            o.blend_state, o.blend_state_bytes = None, 0
        return o


class Grads:
    def __init__(self, N: int, K: int, device, with_mean2d: bool = True):
        z = lambda shape: torch.zeros(shape, dtype=torch.float32, device=device)
        self.N, self.K = N, K
        self.d_means, self.d_scales, self.d_rotations = z((N, 3)), z((N, 3)), z((N, 4))
        self.d_opacities, self.d_sh = z((N,)), z((N, 16, 3))
        self.d_freqs, self.d_weights = z((N, K, 3)), z((N, K))
        self.d_mean2d = z((N, 2)) if with_mean2d else None
        self.d_mean2d_abs = z((N, 2)) if with_mean2d else None
        self.workspace_bytes = int(lib().gabsplat_grad_workspace_bytes(N, K))
        self.workspace = torch.zeros((self.workspace_bytes,), dtype=torch.uint8, device=device)

    def struct(self) -> _Grads:
        g = _Grads()
        for n, _ in _Grads._fields_:
            t = getattr(self, n)
            setattr(g, n, t.data_ptr() if (t is not None and t.numel()) else None)
        return g


# ---- the four calls (same names as the C entry points) ---------------------------------------------

def gabsplat_preprocess(ctx: Context, scene: DeviceScene, cam, out: Projected | None = None, stream=None) -> Projected:
    out = Projected(scene.N, scene.K, scene.means.device) if out is None else out
    s, c, p = scene.struct(), camera_struct(cam), out.struct()
    ctx.check(lib().gabsplat_preprocess(ctx._h, C.byref(s), C.byref(c), C.byref(p), _stream(stream)))
    return out


def gabsplat_bin_sort(ctx: Context, N: int, proj: Projected, cam, bin: Binning | None = None, capacity: int | None = None,
                      read_count: bool = True, stream=None) -> Binning:
    """With bin=None and capacity=None the instance count is taken from a first pass with zero capacity."""
    dev = proj.depth.device
    if bin is None:
        if capacity is None:
            probe = Binning(N, cam, 0, dev)
            p, c, b = proj.struct(), camera_struct(cam), probe.struct()
            d = C.c_uint64(0)
            rc = lib().gabsplat_bin_sort(ctx._h, N, C.byref(p), C.byref(c), C.byref(b), C.byref(d), _stream(stream))
            if rc not in (OK, CAPACITY):
                ctx.check(rc)
            capacity = int(d.value)
        bin = Binning(N, cam, capacity, dev)
    p, c, b = proj.struct(), camera_struct(cam), bin.struct()
    d = C.c_uint64(0)
    ctx.check(lib().gabsplat_bin_sort(ctx._h, N, C.byref(p), C.byref(c), C.byref(b),
                                      C.byref(d) if read_count else None, _stream(stream)))
    bin.D = int(d.value) if read_count else None
    return bin


def gabsplat_preprocess_bin_sort(ctx: Context, scene: DeviceScene, cam, proj: Projected, bin: Binning,
                                 read_count: bool = True, stream=None) -> Binning:
    """S1 + S2 in one call (the value track of the projection overlaps the binning); buffers are the caller's."""
    s, c, p, b = scene.struct(), camera_struct(cam), proj.struct(), bin.struct()
    d = C.c_uint64(0)
    ctx.check(lib().gabsplat_preprocess_bin_sort(ctx._h, C.byref(s), C.byref(c), C.byref(p), C.byref(b),
                                                 C.byref(d) if read_count else None, _stream(stream)))
    bin.D = int(d.value) if read_count else None
    return bin


def gabsplat_render_forward(ctx: Context, scene: DeviceScene, cam, proj: Projected, bin: Binning,
                            out: FwdOut | None = None, stream=None, save_state: bool = True) -> FwdOut:
    """save_state=False renders without recording the blend state (inference; no backward afterwards)."""
    out = FwdOut(cam, scene.means.device, bin.capacity if save_state else None) if out is None else out
    s, c, p, b, o = scene.struct(), camera_struct(cam), proj.struct(), bin.struct(), out.struct(save_state)
    ctx.check(lib().gabsplat_render_forward(ctx._h, C.byref(s), C.byref(c), C.byref(p), C.byref(b), C.byref(o),
                                            _stream(stream)))
    return out


def gabsplat_render_backward(ctx: Context, scene: DeviceScene, cam, proj: Projected, bin: Binning, fwd: FwdOut,
                             dL_dimage: torch.Tensor, grads: Grads | None = None, stream=None) -> Grads:
    grads = Grads(scene.N, scene.K, scene.means.device) if grads is None else grads
    assert dL_dimage.dtype == torch.float32 and dL_dimage.is_contiguous()
    assert tuple(dL_dimage.shape) == (3, cam.height, cam.width)
    s, c, p, b, o, g = (scene.struct(), camera_struct(cam), proj.struct(), bin.struct(), fwd.struct(), grads.struct())
    ctx.check(lib().gabsplat_render_backward(ctx._h, C.byref(s), C.byref(c), C.byref(p), C.byref(b), C.byref(o),
                                             _ptr(dL_dimage), C.byref(g), _ptr(grads.workspace),
                                             grads.workspace_bytes, _stream(stream)))
    return grads


def gabsplat_render_host(ctx: Context, scene, cam, capacity: int, image_host: torch.Tensor,
                         dL_dimage_host: torch.Tensor | None, grads_host: dict | None, arena: torch.Tensor,
                         stream=None) -> None:
    """End-to-end call with HOST buffers (torch CPU tensors, ideally pinned).  `scene` holds CPU tensors
    under the attribute names of gabsplat_scene; `grads_host` maps d_* names to CPU tensors."""
    s = _Scene()
    s.N, s.K, s.sh_degree = int(scene.means.shape[0]), int(scene.freqs.shape[1]), int(scene.sh_degree)
    s.variant = int(getattr(scene, "variant", 0))
    for n in ("means", "scales", "rotations", "opacities", "sh", "freqs", "weights"):
        t = getattr(scene, n)
        setattr(s, n, t.data_ptr() if t.numel() else None)
    g = _Grads()
    if grads_host is not None:
        for n, _ in _Grads._fields_:
            t = grads_host.get(n)
            setattr(g, n, t.data_ptr() if (t is not None and t.numel()) else None)
    c = camera_struct(cam)
    base = (arena.data_ptr() + 255) // 256 * 256
    nbytes = arena.numel() - (base - arena.data_ptr())
    ctx.check(lib().gabsplat_render_host(ctx._h, C.byref(s), C.byref(c), int(capacity), _ptr(image_host),
                                         _ptr(dL_dimage_host), C.byref(g) if grads_host is not None else None,
                                         C.c_void_p(base), nbytes, _stream(stream)))


STAGES = ("preprocess", "scan", "duplicate", "sort", "ranges", "blend_forward", "blend_backward",
          "preprocess_backward", "depth_sort")          # indexed by GABSPLAT_STAGE_*
# stage records of one forward + backward pass, in launch order (images of at most 26000 tiles: the tile ranges
# are known before the instances are placed; larger images run "duplicate", "sort", "ranges")
LAUNCH_ORDER = ("preprocess", "depth_sort", "scan", "duplicate", "ranges", "sort", "blend_forward", "blend_backward",
                "preprocess_backward")


def gabsplat_render_aux(ctx: Context, scene: DeviceScene, cam, proj: Projected, bin: Binning, stream=None) -> torch.Tensor:
    """Auxiliary renders [3][H][W]: blended sum_k omega_k |f2D_k|, blended depth, accumulated alpha."""
    dev = scene.means.device
    out = torch.empty((3, cam.height, cam.width), dtype=torch.float32, device=dev)
    nbytes = int(lib().gabsplat_aux_workspace_bytes(scene.N, cam.width, cam.height))
    ws = torch.empty((nbytes,), dtype=torch.uint8, device=dev)
    s, c, p, b = scene.struct(), camera_struct(cam), proj.struct(), bin.struct()
    ctx.check(lib().gabsplat_render_aux(ctx._h, C.byref(s), C.byref(c), C.byref(p), C.byref(b), _ptr(out), _ptr(ws), nbytes,
                                        _stream(stream)))
    return out


def gabsplat_loss(ctx: Context, image: torch.Tensor, target: torch.Tensor, lam: float = 0.2, want_grad: bool = True,
                  workspace: torch.Tensor | None = None, stream=None):
    """Eq.14 on the device: returns (loss_out [3] = (L, L1, mean SSIM) device tensor, dL_dimage or None)."""
    assert image.dtype == torch.float32 and target.dtype == torch.float32 and image.shape == target.shape
    assert image.is_contiguous() and target.is_contiguous() and image.dim() == 3 and image.shape[0] == 3
    H, W = int(image.shape[1]), int(image.shape[2])
    nbytes = int(lib().gabsplat_loss_workspace_bytes(W, H))
    if workspace is None:
        workspace = torch.empty((nbytes,), dtype=torch.uint8, device=image.device)
    out = torch.zeros((3,), dtype=torch.float32, device=image.device)
    grad = torch.empty_like(image) if want_grad else None
    ctx.check(lib().gabsplat_loss(ctx._h, W, H, _ptr(image), _ptr(target), float(lam), _ptr(out),
                                  _ptr(grad) if want_grad else None, _ptr(workspace), workspace.numel(), _stream(stream)))
    return out, grad


def gabsplat_loss_static_max_pixels() -> int:
    return int(lib().gabsplat_loss_static_max_pixels())


def gabsplat_loss_static(image: torch.Tensor, target: torch.Tensor, lam: float = 0.2, out: torch.Tensor | None = None,
                         grad: torch.Tensor | None = None, want_grad: bool = True, stream=None):
    """gabsplat_loss without a workspace and without a context, for callers that may not allocate device memory
    (plugins that only own their inputs and outputs, loops that must stay off the allocator): the scratch is a fixed
    array inside the library, one per GPU, shared by all calls.  Pass `out` ([3]) and `grad` (like image) to keep this
    wrapper from allocating them with torch; images beyond gabsplat_loss_static_max_pixels() raise (status CAPACITY).
    Calls that may overlap on the GPU race on the shared scratch: keep them on one stream."""
    assert image.dtype == torch.float32 and target.dtype == torch.float32 and image.shape == target.shape
    assert image.is_contiguous() and target.is_contiguous() and image.dim() == 3 and image.shape[0] == 3
    H, W = int(image.shape[1]), int(image.shape[2])
    if out is None:
        out = torch.empty((3,), dtype=torch.float32, device=image.device)
    if want_grad and grad is None:
        grad = torch.empty_like(image)
    with torch.cuda.device(image.device):      # the scratch that is used is the current device's
        rc = lib().gabsplat_loss_static(W, H, _ptr(image), _ptr(target), float(lam), _ptr(out),
                                        _ptr(grad) if want_grad else None, _stream(stream))
    if rc != 0:
        raise GabsplatError(rc, lib().gabsplat_loss_static_last_error().decode())
    return out, (grad if want_grad else None)


def gabsplat_kernel_launches() -> int:
    return int(lib().gabsplat_kernel_launches())


def gabsplat_timing_enable(ctx: Context, on: bool) -> None:
    ctx.check(lib().gabsplat_timing_enable(ctx._h, 1 if on else 0))


def gabsplat_timing_read(ctx: Context, max_records: int = 1 << 16) -> list[tuple[str, float]]:
    """(stage name, milliseconds) of every stage launched since timing was enabled / last read."""
    ids = (C.c_int32 * max_records)()
    ms = (C.c_float * max_records)()
    n = C.c_int32(0)
    ctx.check(lib().gabsplat_timing_read(ctx._h, ids, ms, max_records, C.byref(n)))
    return [(STAGES[ids[i]], float(ms[i])) for i in range(min(n.value, max_records))]


def gabsplat_count_pairs(ctx: Context, scene: DeviceScene, cam, proj: Projected, bin: Binning, stream=None) -> torch.Tensor:
    """[H][W][4] int32 per-pixel counters (examined, past the envelope test, blended, past the envelope
    test at positions <= the last contributor)."""
    out = torch.zeros((cam.height, cam.width, 4), dtype=torch.int32, device=scene.means.device)
    s, c, p, b = scene.struct(), camera_struct(cam), proj.struct(), bin.struct()
    ctx.check(lib().gabsplat_count_pairs(ctx._h, C.byref(s), C.byref(c), C.byref(p), C.byref(b), _ptr(out),
                                         _stream(stream)))
    return out


def gabsplat_trace_pixels(ctx: Context, scene: DeviceScene, cam, proj: Projected, bin: Binning, pixels: torch.Tensor,
                          offsets: torch.Tensor, stream=None):
    """The forward's decisions at the pixels [n][2] (x, y) int32: returns (entries, colour_T [n][4], info [n][4]);
    entries[offsets[i]:offsets[i+1]] = 1-based list positions of the entries blended at pixel i (bit 31: clamp active)."""
    dev = scene.means.device
    n = int(pixels.shape[0])
    assert pixels.dtype == torch.int32 and pixels.is_contiguous() and offsets.dtype == torch.int32 and offsets.numel() == n + 1
    entries = torch.zeros((max(1, int(offsets[-1].item())),), dtype=torch.int32, device=dev)
    colour_T = torch.zeros((max(n, 1), 4), dtype=torch.float32, device=dev)
    info = torch.zeros((max(n, 1), 4), dtype=torch.int32, device=dev)
    s, c, p, b = scene.struct(), camera_struct(cam), proj.struct(), bin.struct()
    ctx.check(lib().gabsplat_trace_pixels(ctx._h, C.byref(s), C.byref(c), C.byref(p), C.byref(b), n, _ptr(pixels),
                                          _ptr(offsets), _ptr(entries), _ptr(colour_T), _ptr(info), _stream(stream)))
    return entries, colour_T[:n], info[:n]


def gabsplat_probe_sincos(ctx: Context, phase: torch.Tensor, stream=None):
    """(cos, sin) of raw radian phases as the blend kernels evaluate them."""
    assert phase.dtype == torch.float32 and phase.is_contiguous()
    c, s = torch.empty_like(phase), torch.empty_like(phase)
    ctx.check(lib().gabsplat_probe_sincos(ctx._h, phase.numel(), _ptr(phase), _ptr(c), _ptr(s), _stream(stream)))
    return c, s


def gabsplat_set_place_bands(ctx: Context, bands: int) -> None:
    ctx.check(lib().gabsplat_set_place_bands(ctx._h, int(bands)))


PEAK_NAMES = ("ffma", "ffma2", "mufu_ex2", "mufu_cos", "mix_4ffma_1mufu", "alu_iadd")


def gabsplat_measure_peaks(ctx: Context, stream=None) -> dict:
    """Measured ALU rooflines of this device: lane-instructions (lane-ops) per second and per SM per clock."""
    r = (C.c_float * 16)()
    ctx.check(lib().gabsplat_measure_peaks(ctx._h, r, _stream(stream)))
    out = {n: float(r[i]) for i, n in enumerate(PEAK_NAMES)}
    out.update({n + "_per_sm_clk": float(r[8 + i]) for i, n in enumerate(PEAK_NAMES)})
    out["sm_clock_hz"], out["sms"] = float(r[6]), int(r[7])
    return out


def host_arena_bytes(N: int, K: int, cam, capacity: int) -> int:
    return int(lib().gabsplat_host_arena_bytes(N, K, cam.width, cam.height, int(capacity))) + 256
