"""ORACLE -- TEST INFRASTRUCTURE ONLY.  The training loss of PAPER.md:171 Eq.14,

    L = (1 - lambda) L1 + lambda L_D-SSIM,        lambda = 0.2,

"as in 3DGS" [25]: L1 = mean |I - I_gt| over pixels and channels; L_D-SSIM = 1 - mean SSIM; SSIM per channel with
an 11x11 Gaussian window (sigma 1.5, normalised), zero padding, C1 = 0.01^2, C2 = 0.03^2 (reading C25:
the paper gives Eq.14 only; window and constants are [25]'s published choice).

Plain numpy, float64, direct (non-separable) windowed sums written as explicit loops over the 121 taps: slow and
obviously the definition.  The gradient is the analytic derivative of exactly this forward.

Pins (tests/test_oracle_loss.py): the local means equal scipy.ndimage.gaussian_filter(mode="constant") (an
independent library routine with the same 11 taps); SSIM(x, x) = 1 and L(x, x) = 0; constant images give the
closed form (2ab + C1) / (a^2 + b^2 + C1) away from the border; symmetry in the two images; the gradient against
central finite differences.  Only tests/ may import this module; it imports nothing from the CUDA path.
"""
from __future__ import annotations

import numpy as np

WINDOW = 11
SIGMA = 1.5
C1 = 0.01 ** 2
C2 = 0.03 ** 2


def gaussian_window() -> np.ndarray:
    """w[i][j] = g[i] g[j], g[i] = exp(-(i - 5)^2 / (2 sigma^2)) normalised to sum 1."""
    x = np.arange(WINDOW, dtype=np.float64) - WINDOW // 2
    g = np.exp(-(x * x) / (2.0 * SIGMA * SIGMA))
    g /= g.sum()
    return np.outer(g, g)


def window_sum(a: np.ndarray) -> np.ndarray:
    """(w * a)[y][x] = sum_ij w[i][j] a[y + i - 5][x + j - 5], zero outside the image; a is [C][H][W]."""
    w = gaussian_window()
    r = WINDOW // 2
    C, H, W = a.shape
    p = np.zeros((C, H + 2 * r, W + 2 * r), dtype=np.float64)
    p[:, r:r + H, r:r + W] = a
    out = np.zeros((C, H, W), dtype=np.float64)
    for i in range(WINDOW):
        for j in range(WINDOW):
            out += w[i, j] * p[:, i:i + H, j:j + W]
    return out


def ssim_map(x: np.ndarray, y: np.ndarray) -> np.ndarray:
    mx, my = window_sum(x), window_sum(y)
    sxx = window_sum(x * x) - mx * mx
    syy = window_sum(y * y) - my * my
    sxy = window_sum(x * y) - mx * my
    return ((2 * mx * my + C1) * (2 * sxy + C2)) / ((mx * mx + my * my + C1) * (sxx + syy + C2))


def loss_forward(image: np.ndarray, target: np.ndarray, lam: float = 0.2) -> dict:
    x = np.asarray(image, dtype=np.float64)
    y = np.asarray(target, dtype=np.float64)
    l1 = float(np.mean(np.abs(x - y)))
    ssim = float(np.mean(ssim_map(x, y)))
    return {"loss": (1.0 - lam) * l1 + lam * (1.0 - ssim), "l1": l1, "ssim": ssim}


def loss_backward(image: np.ndarray, target: np.ndarray, lam: float = 0.2) -> np.ndarray:
    """dL/dimage, [C][H][W].  With S = A1 A2 / (B1 B2), A1 = 2 mx my + C1, A2 = 2 (Exy - mx my) + C2,
    B1 = mx^2 + my^2 + C1, B2 = (Exx - mx^2) + (Eyy - my^2) + C2 and mx = w*x, Exx = w*x^2, Exy = w*xy:
      dS/dmx  = (2 my A2 - 2 my A1) / (B1 B2) - S (2 mx / B1 - 2 mx / B2)
      dS/dExx = -S / B2
      dS/dExy = 2 A1 / (B1 B2)
    and, the window being symmetric, dL/dx = w*(g dS/dmx) + 2 x w*(g dS/dExx) + y w*(g dS/dExy), g = dL/dS."""
    x = np.asarray(image, dtype=np.float64)
    y = np.asarray(target, dtype=np.float64)
    n = x.size
    mx, my = window_sum(x), window_sum(y)
    exx, eyy, exy = window_sum(x * x), window_sum(y * y), window_sum(x * y)
    a1 = 2 * mx * my + C1
    a2 = 2 * (exy - mx * my) + C2
    b1 = mx * mx + my * my + C1
    b2 = (exx - mx * mx) + (eyy - my * my) + C2
    s = a1 * a2 / (b1 * b2)
    g = -lam / n                                   # dL/dS at every pixel: L_D-SSIM = 1 - mean S
    ds_dmx = (2 * my * a2 - 2 * my * a1) / (b1 * b2) - s * (2 * mx / b1 - 2 * mx / b2)
    ds_dexx = -s / b2
    ds_dexy = 2 * a1 / (b1 * b2)
    grad = window_sum(g * ds_dmx) + 2 * x * window_sum(g * ds_dexx) + y * window_sum(g * ds_dexy)
    grad += (1.0 - lam) / n * np.sign(x - y)
    return grad
