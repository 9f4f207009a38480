"""-m gpu: the committed measurements DESIGN.md leans on -- the error of the MUFU cosine / sine path the blend kernels
use on raw radian phases (Eq.12), and the measured ALU rooflines."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

# |cos_gpu - cos| and |sin_gpu - sin| <= A |phase| + B for |phase| <= 500 rad
PHASE_ERR_A, PHASE_ERR_B = 1.6e-7, 5e-7


def test_mufu_phase_error_bound():
    import torch
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx
    g = torch.Generator(device="cuda").manual_seed(3)
    ph = ((torch.rand(1 << 22, device="cuda", dtype=torch.float64, generator=g) * 2 - 1) * 500).float()
    # the phases that matter most: multiples of pi / 2, where one of the two functions crosses zero
    k = torch.arange(-300, 301, device="cuda", dtype=torch.float64) * (np.pi / 2)
    ph = torch.cat([ph, k.float(), torch.zeros(1, device="cuda")])
    c, s = gb.gabsplat_probe_sincos(ctx(), ph)
    torch.cuda.synchronize()
    x = ph.double()
    ec, es = (c.double() - torch.cos(x)).abs(), (s.double() - torch.sin(x)).abs()
    bound = PHASE_ERR_A * x.abs() + PHASE_ERR_B
    ratio = float((torch.maximum(ec, es) / bound).max())
    assert ratio <= 1.0, ratio
    # at |phase| = 300 rad (the largest the 1M-primitive configs produce inside a footprint) the error is <= 5e-5
    m = x.abs() <= 300
    assert float(torch.maximum(ec, es)[m].max()) <= 5e-5
    assert float(c[-1]) == 1.0 and float(s[-1]) == 0.0


def test_measured_peaks_are_sane():
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx
    p = gb.gabsplat_measure_peaks(ctx())
    assert p["sms"] >= 100
    nominal_fp32 = p["sms"] * 128 * 1.965e9          # lane-instructions / s at the maximum SM clock
    nominal_mufu = p["sms"] * 16 * 1.965e9
    assert 0.5 * nominal_fp32 <= p["ffma"] <= 1.05 * nominal_fp32, p
    assert 0.5 * nominal_mufu <= p["mufu_ex2"] <= 1.05 * nominal_mufu, p
    assert 0.5 * nominal_mufu <= p["mufu_cos"] <= 1.05 * nominal_mufu, p
    assert 0.4 * nominal_fp32 <= 2 * p["ffma2"] <= 1.05 * nominal_fp32, p   # packed: two fp32 fmas per lane-instruction
    assert 1.0e9 <= p["sm_clock_hz"] <= 2.2e9, p


def test_trace_pixels_flags_pixels_outside_the_image():
    """gabsplat_trace_pixels must not index tile_ranges with a pixel that is not in the image, nor trust a descending
    offsets pair: such a pixel is flagged (info[3] = 1, nothing else), an inverted slice is empty, and the pixels
    around them are traced as if they were alone."""
    import torch
    from paper_2508_05343_b200 import binding as gb, scenes
    from gpu_helpers import ctx, run_gpu
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    g, dev = run_gpu(scene, cam)
    W, H = cam.width, cam.height
    px = torch.tensor([[64, 64], [-1, 5], [W, 3], [7, H], [1 << 20, 1 << 20], [70, 60], [64, 64]], dtype=torch.int32, device="cuda")
    # 64 entries per pixel, except pixel 5, whose pair is inverted (320 .. 256); pixel 6 reuses an outside pixel's slice
    offsets = torch.tensor([0, 64, 128, 192, 256, 320, 256, 320], dtype=torch.int32, device="cuda")
    entries, colour_T, info = gb.gabsplat_trace_pixels(ctx(), dev["scene"], cam, dev["proj"], dev["bins"], px, offsets)
    torch.cuda.synchronize()
    info, colour_T = info.cpu().numpy(), colour_T.cpu().numpy()
    assert (info[1:5] == np.array([0, 0, 0, 1])).all() and (colour_T[1:5] == 0).all()
    for i, (x, y) in ((0, (64, 64)), (5, (70, 60)), (6, (64, 64))):
        assert info[i, 3] == 0 and info[i, 0] == g["n_contrib"][y, x]
        assert np.array_equal(colour_T[i, :3], g["image"][:, y, x]) and colour_T[i, 3] == g["final_T"][y, x]
    e = entries.cpu().numpy()
    assert info[5, 1] > 0                      # blended entries counted, none written: the slice was empty
    assert info[6, 1] == info[0, 1] and np.array_equal(e[256:320], e[0:64]) and e[0] != 0
    assert (e[64:256] == 0).all()              # the slices of the outside pixels stayed untouched
