"""-m gpu parity of gabsplat_loss (Eq.14) against oracle/loss_oracle.py:
loss terms to 2e-6 absolute (fp32 outputs of fp64 sums), dL/dimage to 1e-4 of its max norm."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _mods():
    import torch
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx
    from oracle import loss_oracle as lo
    return torch, gb, ctx(), lo


def _pair(seed, H, W):
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:H, 0:W]
    base = np.stack([0.5 + 0.4 * np.sin(0.05 * xx + c) * np.cos(0.07 * yy - c) for c in range(3)])
    target = np.clip(base + 0.05 * rng.standard_normal(base.shape), 0, 1).astype(np.float32)
    image = np.clip(base + 0.1 * rng.standard_normal(base.shape), 0, 1).astype(np.float32)
    return image, target


def _check(image, target, lam):
    torch, gb, ctx, lo = _mods()
    out, grad = gb.gabsplat_loss(ctx, torch.from_numpy(image).cuda(), torch.from_numpy(target).cuda(), lam)
    torch.cuda.synchronize()
    ref = lo.loss_forward(image, target, lam)
    got = out.cpu().numpy().astype(np.float64)
    assert abs(got[0] - ref["loss"]) <= 2e-6 and abs(got[1] - ref["l1"]) <= 2e-6 and abs(got[2] - ref["ssim"]) <= 2e-6, (got, ref)
    gref = lo.loss_backward(image, target, lam)
    err = np.abs(grad.cpu().numpy().astype(np.float64) - gref).max()
    assert err <= 1e-4 * np.abs(gref).max(), (err, np.abs(gref).max())


@pytest.mark.parametrize("lam", [0.2, 0.0, 1.0])
def test_loss_ragged(lam):
    """203 x 131: several 32x8 tiles and a ragged right / bottom edge, borders with a partial window."""
    image, target = _pair(1, 131, 203)
    _check(image, target, lam)


def test_loss_tiny_image_smaller_than_the_window():
    image, target = _pair(2, 7, 9)
    _check(image, target, 0.2)


def test_identical_images_give_zero_loss_and_gradient():
    torch, gb, ctx, lo = _mods()
    image, _ = _pair(3, 64, 96)
    x = torch.from_numpy(image).cuda()
    out, grad = gb.gabsplat_loss(ctx, x, x.clone(), 0.2)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    assert o[1] == 0.0 and abs(o[2] - 1.0) <= 1e-6 and abs(o[0]) <= 1e-6
    assert float(grad.abs().max()) <= 1e-9          # SSIM is maximal and |x - y| has sign 0
    out2, none = gb.gabsplat_loss(ctx, x, x.clone(), 0.2, want_grad=False)
    torch.cuda.synchronize()
    assert none is None and torch.equal(out, out2)  # deterministic


def test_loss_full_size():
    """The headline image size, 1297 x 840 (not a multiple of the tile in either direction)."""
    image, target = _pair(4, 840, 1297)
    _check(image, target, 0.2)


def test_loss_feeds_the_backward():
    """dL/dimage of the loss is a valid dL_dimage of gabsplat_render_backward (shapes, layout): one training step's
    worth of calls on config 1."""
    torch, gb, ctx, lo = _mods()
    from paper_2508_05343_b200 import scenes
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(ctx, ds, cam)
    bins = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam)
    fwd = gb.gabsplat_render_forward(ctx, ds, cam, proj, bins)
    target = torch.full_like(fwd.image, 0.5)
    out, dL = gb.gabsplat_loss(ctx, fwd.image, target, 0.2)
    grads = gb.gabsplat_render_backward(ctx, ds, cam, proj, bins, fwd, dL)
    torch.cuda.synchronize()
    assert float(out[0]) > 0 and float(grads.d_sh.abs().max()) > 0
