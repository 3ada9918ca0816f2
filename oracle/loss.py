"""TEST INFRASTRUCTURE - fp64 NumPy oracle of the LF-weighted photometric loss (PAPER.md P:116-141,
eqs. 7-10, and P:220-224 eq. 18). Only tests/, smoke() and bench.py's cpu_baseline leg may import it.

Steps in the paper's order (reading R10 where the paper is silent):
  1. s(p): "percentile-normalized Sobel magnitude ... treated as stop-grad". Grey = channel mean
     of the TARGET image (sobel_source=0) or of the render (1); 3x3 Sobel, replicate border;
     m = sqrt(gx^2 + gy^2); s = min(1, m / m_q), m_q = nearest-rank q-quantile sorted[ceil(q |P|) - 1];
     m_q = 0 => s = 0.
  2. w(p) = (eps + 1 - s(p))^gamma, eps = 1e-3                               (eq. 7)
  3. w~(p) = w(p) / mean_q w(q)                                               (eq. 8)
  4. L = 1/|P| sum_p w~(p) rho(r_p), r_p = R(p) - I(p)                        (eq. 10 P:139 / eq. 18)
     rho = L1 averaged over the 3 channels (R10; BASELINE.json north_star (5) says L1).
  5. dL/dR[p,ch] = w~(p) sign(r) / (3 |P|), sign(0) = 0 (s is stop-grad).
  gamma(t): piecewise-linear ramp, eq. 9.

Pins (tests/test_oracle_pins.py): gamma = 0 => w~ = 1 and the gradient is sign(r)/(3|P|);
mean(w~) = 1 (eq. 8); constant target => s = 0; ramp image I = a x + b y => interior Sobel (8a, 8b);
eq. 9 at t0, (t0+t1)/2, t1 gives 0, gamma_max/2, gamma_max; eq. 7 BY VALUE: a one-step target has Sobel
magnitude {0, 4a}, so w_edge / w_flat = (eps / (1 + eps))^gamma and w~ in closed form; the
nearest-rank rule sorted[ceil(q |P|) - 1] on a dot lattice whose magnitudes are {0, sqrt(2) a, 2a} with the
rank boundary exactly at q |P| (floor(q |P|) or the maximum give another answer). The definitions the paper
leaves open (Sobel source, grey conversion, border rule, the percentile q, rho = L1 and the channel mean) are
the readings R10 of DESIGN.md: the pins fix that the code computes those readings, not that the paper meant them.
q is used as given: callers that mirror the C ABI pass the binary32 value of the percentile.
"""
from __future__ import annotations

import numpy as np


def gamma_schedule(t: float, T: float, t0_frac: float = 0.3, t1_frac: float = 0.6, gamma_max: float = 0.6) -> float:
    """eq. 9, defaults t0 = 0.3 T, t1 = 0.6 T, gamma_max = 0.6."""
    t0, t1 = t0_frac * T, t1_frac * T
    if t < t0:
        return 0.0
    if t < t1:
        return gamma_max * (t - t0) / (t1 - t0)
    return gamma_max


def sobel_magnitude(img: np.ndarray) -> np.ndarray:
    """|grad| of the channel-mean grey image, 3x3 Sobel, replicate border. Written as explicit loops
    over the 3x3 stencil (no convolution routine) so the kernel coefficients are visible."""
    g = np.asarray(img, dtype=np.float64).mean(axis=2)
    H, W = g.shape
    p = np.pad(g, 1, mode="edge")
    kx = np.array([[-1.0, 0.0, 1.0], [-2.0, 0.0, 2.0], [-1.0, 0.0, 1.0]])
    ky = kx.T
    gx = np.zeros_like(g)
    gy = np.zeros_like(g)
    for dy in range(3):
        for dx in range(3):
            win = p[dy:dy + H, dx:dx + W]
            gx += kx[dy, dx] * win
            gy += ky[dy, dx] * win
    return np.sqrt(gx * gx + gy * gy)


def lf_weights(source_img: np.ndarray, gamma: float, eps: float = 1e-3, q: float = 0.99) -> np.ndarray:
    m = sobel_magnitude(source_img)
    flat = np.sort(m.reshape(-1))
    k = int(np.ceil(q * flat.size)) - 1
    k = min(max(k, 0), flat.size - 1)
    mq = flat[k]
    s = np.minimum(1.0, m / mq) if mq > 0 else np.zeros_like(m)
    w = np.power(eps + 1.0 - s, gamma)
    return w / w.mean()


def lf_loss_and_grad(render: np.ndarray, target: np.ndarray, gamma: float, eps: float = 1e-3, q: float = 0.99,
                     sobel_source: int = 0):
    """Returns (L, dL/dRender [H,W,3], w~ [H,W])."""
    R = np.asarray(render, dtype=np.float64)
    I = np.asarray(target, dtype=np.float64)
    wt = lf_weights(I if sobel_source == 0 else R, gamma, eps, q)
    r = R - I
    n_pix = R.shape[0] * R.shape[1]
    L = float((wt[:, :, None] * np.abs(r)).sum() / (3.0 * n_pix))
    dL = wt[:, :, None] * np.sign(r) / (3.0 * n_pix)
    return L, dL, wt
