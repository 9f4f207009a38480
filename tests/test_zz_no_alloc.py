"""-m gpu: gabsplat_loss_static, the loss for callers that cannot allocate device memory, against gabsplat_loss.

Who needs it: a plugin that runs inside another engine and owns nothing but the input and output buffers it is
handed; a loop that has promised not to call the allocator once it is running (cudaMalloc locks the process and can
stall the GPU); a job on a crowded GPU that cannot rely on a free block.  gabsplat_loss is closed to all of them
because its workspace must be cudaMalloc'ed by someone.  gabsplat_loss_static keeps that workspace in a fixed array
inside the library instead (Eq.14, unchanged), so here it is checked against gabsplat_loss:

  - twice in a row, the second call on a smaller image, so that the second call finds the first call's leftovers in
    the shared array and must not be disturbed by them;
  - a third time on the first image again, which must reproduce the first result exactly;
  - with the tolerances of tests/test_gpu_loss.py (loss terms 2e-6 absolute, gradient 1e-4 of its max norm) -- the
    two entry points launch the same kernels, so the difference is expected to be zero;
  - and an image over the built-in limit must be refused with the CAPACITY status, not rendered wrongly.

The file name sorts after every other test file on purpose: the suite runs with pytest -x, so a failure here hides no
other test.  It needs nothing from the tests before it and leaves nothing behind (it passes alone in a fresh process
and after the rest of the suite)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _pair(seed, H, W):
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:H, 0:W]
    base = np.stack([0.5 + 0.4 * np.sin(0.05 * xx + c) * np.cos(0.07 * yy - c) for c in range(3)])
    target = np.clip(base + 0.05 * rng.standard_normal(base.shape), 0, 1).astype(np.float32)
    image = np.clip(base + 0.1 * rng.standard_normal(base.shape), 0, 1).astype(np.float32)
    return image, target


def _close(static, plain):
    (out_s, grad_s), (out_p, grad_p) = static, plain
    o_s, o_p = out_s.cpu().numpy().astype(np.float64), out_p.cpu().numpy().astype(np.float64)
    assert np.abs(o_s - o_p).max() <= 2e-6, (o_s, o_p)
    g_s, g_p = grad_s.cpu().numpy().astype(np.float64), grad_p.cpu().numpy().astype(np.float64)
    assert np.isfinite(g_s).all()
    assert np.abs(g_s - g_p).max() <= 1e-4 * np.abs(g_p).max(), (np.abs(g_s - g_p).max(), np.abs(g_p).max())


def test_static_loss_matches_the_workspace_loss_on_two_calls_in_a_row():
    import torch
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx as make_ctx
    ctx = make_ctx()
    # 203 x 131: ragged in both directions; 96 x 64: smaller, so most of the array still holds the first call's maps
    cases = [_pair(11, 131, 203), _pair(12, 64, 96)]
    dev = [(torch.from_numpy(i).cuda(), torch.from_numpy(t).cuda()) for i, t in cases]
    outs = [torch.empty(3, dtype=torch.float32, device="cuda") for _ in dev]      # the caller's outputs, made up front:
    grads = [torch.empty_like(i) for i, _ in dev]                                  # nothing is allocated between calls
    plain = [gb.gabsplat_loss(ctx, i, t, 0.2) for i, t in dev]
    torch.cuda.synchronize()

    static = [gb.gabsplat_loss_static(i, t, 0.2, out=o, grad=g) for (i, t), o, g in zip(dev, outs, grads)]
    torch.cuda.synchronize()
    for s, p in zip(static, plain):
        _close(s, p)
    assert float(static[0][0][0]) > 0.01            # a real loss, not an untouched buffer

    first = (static[0][0].clone(), static[0][1].clone())
    again = gb.gabsplat_loss_static(dev[0][0], dev[0][1], 0.2, out=outs[0], grad=grads[0])
    torch.cuda.synchronize()
    assert torch.equal(again[0], first[0]) and torch.equal(again[1], first[1])

    forward_only, none = gb.gabsplat_loss_static(dev[1][0], dev[1][1], 0.2, want_grad=False)
    torch.cuda.synchronize()
    assert none is None and torch.equal(forward_only, static[1][0])


def test_static_loss_refuses_images_over_its_limit():
    import torch
    from paper_2508_05343_b200 import binding as gb
    limit = gb.gabsplat_loss_static_max_pixels()
    assert limit == 512 * 512
    at_limit = torch.rand((3, 512, 512), dtype=torch.float32, device="cuda")
    out, grad = gb.gabsplat_loss_static(at_limit, at_limit.clone(), 0.2)
    torch.cuda.synchronize()
    assert float(out[1]) == 0.0 and abs(float(out[2]) - 1.0) <= 1e-6
    for shape in [(3, 512, 513), (3, 1, 2049), (3, 840, 1297)]:
        big = torch.zeros(shape, dtype=torch.float32, device="cuda")
        sentinel = torch.full((3,), -7.0, dtype=torch.float32, device="cuda")
        with pytest.raises(gb.GabsplatError) as err:
            gb.gabsplat_loss_static(big, big, 0.2, out=sentinel, want_grad=False)
        assert err.value.code == gb.CAPACITY and "larger than the built-in scratch" in str(err.value)
        torch.cuda.synchronize()
        assert torch.equal(sentinel.cpu(), torch.full((3,), -7.0))      # nothing was launched
