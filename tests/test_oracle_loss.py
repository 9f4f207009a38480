"""Pins of the loss oracle (oracle/loss_oracle.py; Eq.14, window and constants of [25], DESIGN.md
reading C25) against things other than itself: a library Gaussian filter, closed forms, symmetries, and central
finite differences of its own forward."""
import numpy as np
import pytest

from oracle import loss_oracle as lo


def _images(seed, C=3, H=23, W=31):
    rng = np.random.default_rng(seed)
    x = rng.uniform(0.0, 1.0, (C, H, W))
    y = np.clip(x + 0.2 * rng.standard_normal((C, H, W)), 0.0, 1.0)
    return x, y


def test_window_is_the_truncated_normalised_gaussian():
    w = lo.gaussian_window()
    assert w.shape == (11, 11) and abs(w.sum() - 1.0) < 1e-15
    assert np.allclose(w, w.T) and np.allclose(w, w[::-1, ::-1])
    assert abs(w[5, 5] / w[5, 6] - np.exp(1.0 / (2 * 1.5 ** 2))) < 1e-12        # ratio of neighbouring taps


def test_window_sum_equals_scipy_gaussian_filter():
    """scipy's gaussian_filter with truncate = 5 / 1.5 uses the same 11 normalised taps; mode constant = zero padding."""
    from scipy.ndimage import gaussian_filter
    x, _ = _images(1)
    ref = np.stack([gaussian_filter(c, sigma=1.5, mode="constant", cval=0.0, truncate=5.0 / 1.5 + 1e-9) for c in x])
    assert np.max(np.abs(lo.window_sum(x) - ref)) < 1e-14


def test_identical_images():
    x, _ = _images(2)
    out = lo.loss_forward(x, x)
    assert out["l1"] == 0.0 and abs(out["ssim"] - 1.0) < 1e-14 and abs(out["loss"]) < 1e-14


def test_constant_images_closed_form():
    """Constant a against constant b: variances vanish, so in the interior (full window inside the image)
    SSIM = (2ab + C1) / (a^2 + b^2 + C1); L1 = |a - b| everywhere."""
    a, b = 0.7, 0.4
    x = np.full((1, 40, 40), a)
    y = np.full((1, 40, 40), b)
    s = lo.ssim_map(x, y)
    assert np.allclose(s[0, 5:-5, 5:-5], (2 * a * b + lo.C1) / (a * a + b * b + lo.C1), rtol=0, atol=1e-11)   # cancellation in Exx - mx^2 against C2 = 9e-4
    assert abs(lo.loss_forward(x, y)["l1"] - abs(a - b)) < 1e-15


def test_ssim_is_symmetric_and_bounded():
    x, y = _images(3)
    assert np.max(np.abs(lo.ssim_map(x, y) - lo.ssim_map(y, x))) < 1e-14
    assert np.all(lo.ssim_map(x, y) <= 1.0 + 1e-12)


def test_lambda_mixes_the_two_terms():
    x, y = _images(4)
    f0, f1, f = lo.loss_forward(x, y, 0.0), lo.loss_forward(x, y, 1.0), lo.loss_forward(x, y, 0.2)
    assert abs(f0["loss"] - f0["l1"]) < 1e-15 and abs(f1["loss"] - (1 - f1["ssim"])) < 1e-15
    assert abs(f["loss"] - (0.8 * f["l1"] + 0.2 * (1 - f["ssim"]))) < 1e-15


@pytest.mark.parametrize("lam", [0.0, 0.2, 1.0])
def test_gradient_against_central_differences(lam):
    x, y = _images(5, C=2, H=17, W=19)
    g = lo.loss_backward(x, y, lam)
    rng = np.random.default_rng(6)
    h = 1e-6
    for _ in range(40):
        c, i, j = rng.integers(0, 2), rng.integers(0, 17), rng.integers(0, 19)   # borders included
        xp, xm = x.copy(), x.copy()
        xp[c, i, j] += h
        xm[c, i, j] -= h
        fd = (lo.loss_forward(xp, y, lam)["loss"] - lo.loss_forward(xm, y, lam)["loss"]) / (2 * h)
        assert abs(fd - g[c, i, j]) <= 1e-6 * max(abs(fd), np.abs(g).max()), (c, i, j, fd, g[c, i, j])
