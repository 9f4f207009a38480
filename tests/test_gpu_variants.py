"""-m gpu parity of the primitive variants (gabsplat_scene.variant) against the oracle: the line-integral
amplitude C2_k and the Mip 2D filter, alone and together -- every stage, forward
and backward, on config 1 and on a ragged mid-size case; the blend kernels are the unchanged ones (the variants fold
into the gathered record)."""
import numpy as np
import pytest

from paper_2508_05343_b200 import scenes
from test_gpu_parity import check_projection, check_binning, check_forward, check_gradients, _gpu, _oracle, _ragged_case

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("variant", [1, 2, 3])
@pytest.mark.parametrize("K", [4, 1])
def test_tiny_variants(variant, K):
    orc = _oracle()
    scene = scenes.make_scene("tiny", K=K)
    scene.freqs *= np.float32(0.25)          # attenuations spread over (0, 1) instead of underflowing to 0
    scene.variant = variant
    cam = scenes.make_cameras("tiny")[0]
    dL = scenes.make_image_grad("tiny", 0, cam)
    g = _gpu(scene, cam, dL)
    o = orc.project(scene, cam)
    if variant & 1:
        att = o["att"][o["visible"].astype(bool)]
        assert att.min() < 0.75 and att.max() > 0.9   # the scene exercises the attenuation (a precondition, not a tolerance)
    check_projection(g, o, K)
    check_binning(g, orc.bin_sort(scene, cam))
    check_forward(g, orc.render_forward(scene, cam))
    check_gradients(g, orc.render_backward(scene, cam, dL))
    # the variant changes the picture
    base = scenes.make_scene("tiny", K=K)
    base.freqs *= np.float32(0.25)
    assert np.abs(_gpu(base, cam)["image"] - g["image"]).max() > 1e-3


@pytest.mark.parametrize("variant", [1, 3])
def test_ragged_midsize_variants(variant):
    orc = _oracle()
    scene, cam = _ragged_case("unbounded", 40000, 203, 131, 180.0)
    scene.freqs *= np.float32(0.1)
    scene.variant = variant
    dL = np.random.default_rng(8).standard_normal((3, cam.height, cam.width)).astype(np.float32)
    g = _gpu(scene, cam, dL)
    check_projection(g, orc.project(scene, cam), scene.K)
    check_binning(g, orc.bin_sort(scene, cam))
    check_forward(g, orc.render_forward(scene, cam))
    check_gradients(g, orc.render_backward(scene, cam, dL))


def test_full_attenuation_never_blends():
    """Weights summing to more than one with fully attenuated cosines: beta <= 0, the modulation is negative everywhere
    and the primitive must vanish (effective opacity 0) without poisoning anything."""
    orc = _oracle()
    scene = scenes.make_scene("tiny", K=2)
    scene.freqs[:] = np.float32(40.0)        # C2 underflows: the cosine terms vanish
    scene.weights[:] = np.float32(0.7)       # 1 - sum w = -0.4 < 0
    scene.weights[::2] = np.float32(0.2)     # every other primitive keeps a positive Gaussian term
    scene.variant = 1
    cam = scenes.make_cameras("tiny")[0]
    dL = scenes.make_image_grad("tiny", 0, cam)
    g = _gpu(scene, cam, dL)
    o = orc.render_backward(scene, cam, dL)
    check_forward(g, orc.render_forward(scene, cam))
    check_gradients(g, o)
    assert np.all(np.isfinite(g["d_weights"])) and np.all(g["d_weights"][1::2] == 0)


@pytest.mark.parametrize("variant,K,zero_axes", [(1, 4, 1), (3, 4, 1), (2, 0, 2), (2, 0, 1)])
def test_degenerate_scales_give_no_nan(variant, K, zero_axes):
    """Outside the value contract (scales > 0), but a trainer can underflow a scale to exactly 0: the variants divide by
    s^2 (line integral: b = v^T Sigma^-1 v = inf) and by det U (Mip filter: rho = 0, U^-1 not finite).  Such a primitive
    must not poison anything: image and every gradient stay finite, and the primitives that are in contract get the
    gradients they get without the degenerate ones' variant terms (those rows are exactly zero or finite)."""
    import torch
    from gpu_helpers import run_gpu
    scene = scenes.make_scene("tiny", K=K)
    scene.variant = variant
    scene.scales[::7, 1] = 0.0
    if zero_axes == 2:
        scene.scales[::7, 2] = 0.0
    cam = scenes.make_cameras("tiny")[0]
    dL = scenes.make_image_grad("tiny", 0, cam)
    g, _ = run_gpu(scene, cam, dL)
    assert np.isfinite(g["image"]).all()
    for n in ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs", "d_weights"):
        assert np.isfinite(g[n]).all(), n
    assert np.abs(g["d_means"]).max() > 0
