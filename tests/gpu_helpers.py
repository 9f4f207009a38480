"""Helpers of the -m gpu parity tests: run the CUDA path through the C ABI binding, return numpy arrays."""
from __future__ import annotations

import numpy as np
import torch

from paper_2508_05343_b200 import binding as gb

_ctx = None


def ctx() -> gb.Context:
    global _ctx
    if _ctx is None:
        _ctx = gb.Context(0)
    return _ctx


def u32(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().numpy().view(np.uint32)


def run_gpu(scene, cam, dL=None, capacity=None):
    """All four calls; returns (dict of numpy results, device objects)."""
    c = ctx()
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(c, ds, cam)
    bins = gb.gabsplat_bin_sort(c, ds.N, proj, cam, capacity=capacity)
    fwd = gb.gabsplat_render_forward(c, ds, cam, proj, bins)
    torch.cuda.synchronize()
    D = bins.D
    out = dict(
        D=D,
        mean2d=proj.mean2d.cpu().numpy(), depth_bits=u32(proj.depth), radius=proj.radius.cpu().numpy(),
        conic_opacity=proj.conic_opacity.cpu().numpy(), rgb=proj.rgb.cpu().numpy(),
        rgb_clamped=proj.rgb_clamped.cpu().numpy(), freq2d=proj.freq2d.cpu().numpy(),
        tiles_touched=u32(proj.tiles_touched), rect=proj.rect.cpu().numpy(),
        offsets=u32(bins.offsets)[:ds.N],
        keys=bins.keys.cpu().numpy().view(np.uint64)[:D], ids=u32(bins.ids)[:D],
        tile_ranges=u32(bins.tile_ranges),
        image=fwd.image.cpu().numpy(), final_T=fwd.final_T.cpu().numpy(), n_contrib=u32(fwd.n_contrib),
    )
    dev = dict(scene=ds, proj=proj, bins=bins, fwd=fwd)
    if dL is not None:
        g = gb.gabsplat_render_backward(c, ds, cam, proj, bins, fwd, torch.from_numpy(dL).cuda())
        torch.cuda.synchronize()
        for n in ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs", "d_weights", "d_mean2d",
                  "d_mean2d_abs"):
            out[n] = getattr(g, n).cpu().numpy()
        dev["grads"] = g
    return out, dev


def rel_inf(a: np.ndarray, ref: np.ndarray) -> float:
    """|| a - ref ||_inf / || ref ||_inf  (reading C19)."""
    den = float(np.max(np.abs(ref))) if ref.size else 0.0
    if den == 0.0:
        return float(np.max(np.abs(a))) if a.size else 0.0
    return float(np.max(np.abs(a.astype(np.float64) - ref)) / den)
