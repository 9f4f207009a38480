"""-m gpu parity of gabsplat_render_aux against the oracle's auxiliary renders: same lists and
alpha rules as the colour render, so the same tolerance on decidable pixels (1e-4 of the channel's range)."""
import numpy as np
import pytest

from paper_2508_05343_b200 import scenes

pytestmark = pytest.mark.gpu


def _run(scene, cam):
    import torch
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx
    c = ctx()
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(c, ds, cam)
    bins = gb.gabsplat_bin_sort(c, ds.N, proj, cam)
    aux = gb.gabsplat_render_aux(c, ds, cam, proj, bins)
    fwd = gb.gabsplat_render_forward(c, ds, cam, proj, bins, save_state=False)
    torch.cuda.synchronize()
    return aux.cpu().numpy().astype(np.float64), fwd.final_T.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("name,N,W,H,f", [("tiny", 1024, 128, 128, 150.0), ("unbounded", 40000, 203, 131, 180.0)])
def test_aux_renders(name, N, W, H, f):
    from oracle import gabsplat_oracle as orc
    scene = scenes.make_scene(name, N=N)
    base = scenes.make_cameras(name)[0]
    cam = scenes.make_camera(W, H, f, base.world_to_cam, base.bg)
    aux, final_T = _run(scene, cam)
    ref = orc.render_aux(scene, cam)
    margin = orc.render_forward(scene, cam)["margin"]
    dec = np.minimum(margin[..., 0], margin[..., 1]) > 1e-4
    assert dec.mean() > 0.97
    for ch in range(3):
        scale = max(1.0, np.abs(ref["image"][ch]).max())
        err = np.abs(aux[ch] - ref["image"][ch])
        assert err[dec].max() <= 1e-4 * scale, (ch, err[dec].max(), scale)
    # accumulated alpha is 1 - T of the colour render, to fp32 rounding of two different summation orders
    assert np.abs(aux[2] - (1.0 - final_T)).max() <= 2e-5
