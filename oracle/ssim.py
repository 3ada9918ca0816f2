"""TEST INFRASTRUCTURE - fp64 NumPy oracle of the structure-aware penalty L_SSIM of PAPER.md eq. 17 (P:212-218,
P:228 "L_SSIM is the structure-aware penalty"). Only tests/ may import it.

The paper names the term and gives no formula; reading R14 takes the definition every SVRaster / 3DGS
code base trains with, which is the structural similarity index of Wang, Bovik, Sheikh, Simoncelli (2004) written
out below:

  window   g = 11-tap Gaussian, sigma = 1.5, normalised to sum 1; the 2-D window is g g^T; images are ZERO-padded
           (a "same" correlation), each colour channel on its own.
  moments  mu1 = g * R, mu2 = g * I, s11 = g * R^2 - mu1^2, s22 = g * I^2 - mu2^2, s12 = g * (R I) - mu1 mu2
  index    SSIM(p) = (2 mu1 mu2 + C1) (2 s12 + C2) / ((mu1^2 + mu2^2 + C1) (s11 + s22 + C2)),
           C1 = 0.01^2, C2 = 0.03^2 (dynamic range 1)
  loss     L_SSIM = 1 - mean over pixels and channels of SSIM(p)
  gradient with A1 = 2 mu1 mu2 + C1, A2 = 2 s12 + C2, B1 = mu1^2 + mu2^2 + C1, B2 = s11 + s22 + C2 and the three
           maps the render enters through, m1 = g * R, q11 = g * R^2, q12 = g * (R I):
             dS/dq11 = -A1 A2 / (B1 B2^2)
             dS/dq12 = 2 A1 / (B1 B2)
             dS/dm1  = 2 mu2 A2 / (B1 B2) - 2 mu1 A1 A2 / (B1^2 B2) - 2 mu1 dS/dq11 - mu2 dS/dq12
           dL/dR = -(1 / (3 |P|)) [ g^T * dS/dm1 + 2 R (g^T * dS/dq11) + I (g^T * dS/dq12) ]; the window is symmetric and
           the padding is zero, so the adjoint g^T * is the same correlation.

The correlation is written as 121 shifted adds (no convolution routine), so the taps are visible.

Pins (tests/test_oracle_pins.py): R = I gives SSIM = 1 and L = 0 with zero gradient; two constant images give, at
pixels whose window lies inside the image, the closed form (2ab + C1)/(a^2 + b^2 + C1); the index is symmetric in
(R, I); the analytic gradient equals central finite differences of the loss; the window sums to 1 and its centre
tap is the printed value 0.266011... * 0.266011... (sigma = 1.5, 11 taps).
PARITY UNPINNED (paper silent): window size and sigma, padding rule, C1 / C2, the per-channel mean.
"""
from __future__ import annotations

import numpy as np

C1 = 0.01 ** 2
C2 = 0.03 ** 2
TAPS = 11
SIGMA = 1.5


def gaussian_window() -> np.ndarray:
    """g[k] = exp(-(k - 5)^2 / (2 sigma^2)) / sum, k = 0..10."""
    x = np.arange(TAPS, dtype=np.float64) - (TAPS // 2)
    g = np.exp(-(x * x) / (2.0 * SIGMA * SIGMA))
    return g / g.sum()


def blur(x: np.ndarray) -> np.ndarray:
    """Zero-padded "same" correlation of every channel of x [H, W, C] with g g^T, as 121 shifted adds."""
    g = gaussian_window()
    H, W = x.shape[:2]
    r = TAPS // 2
    pad = np.zeros((H + 2 * r, W + 2 * r) + x.shape[2:], dtype=np.float64)
    pad[r:r + H, r:r + W] = x
    out = np.zeros_like(x, dtype=np.float64)
    for dy in range(TAPS):
        for dx in range(TAPS):
            out += (g[dy] * g[dx]) * pad[dy:dy + H, dx:dx + W]
    return out


def ssim_map(render: np.ndarray, target: np.ndarray):
    """Returns (S, parts) with S [H, W, C] the index per pixel and channel."""
    R = np.asarray(render, dtype=np.float64)
    I = np.asarray(target, dtype=np.float64)
    mu1, mu2 = blur(R), blur(I)
    s11 = blur(R * R) - mu1 * mu1
    s22 = blur(I * I) - mu2 * mu2
    s12 = blur(R * I) - mu1 * mu2
    A1 = 2.0 * mu1 * mu2 + C1
    A2 = 2.0 * s12 + C2
    B1 = mu1 * mu1 + mu2 * mu2 + C1
    B2 = s11 + s22 + C2
    S = (A1 * A2) / (B1 * B2)
    return S, dict(mu1=mu1, mu2=mu2, A1=A1, A2=A2, B1=B1, B2=B2)


def ssim_loss_and_grad(render: np.ndarray, target: np.ndarray):
    """L_SSIM = 1 - mean(S) and dL/dR [H, W, C] (fp64)."""
    R = np.asarray(render, dtype=np.float64)
    I = np.asarray(target, dtype=np.float64)
    S, p = ssim_map(R, I)
    mu1, mu2, A1, A2, B1, B2 = p["mu1"], p["mu2"], p["A1"], p["A2"], p["B1"], p["B2"]
    dq11 = -(A1 * A2) / (B1 * B2 * B2)
    dq12 = 2.0 * A1 / (B1 * B2)
    dm1 = 2.0 * mu2 * A2 / (B1 * B2) - 2.0 * mu1 * A1 * A2 / (B1 * B1 * B2) - 2.0 * mu1 * dq11 - mu2 * dq12
    n = float(S.size)
    grad = -(blur(dm1) + 2.0 * R * blur(dq11) + I * blur(dq12)) / n
    return 1.0 - float(S.mean()), grad
