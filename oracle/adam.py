"""TEST INFRASTRUCTURE - NumPy oracle of the Adam update (Kingma & Ba; "Adam state per voxel", ref. [14]
P:334) that SURVEY 8f lists under NEXT-4 ("fused Adam over voxel parameters"). Only tests/ may import it.
float32, every operation rounded in the written order (the CUDA kernel uses the same sequence, so the result is
bit-identical):
    m <- b1 m + (1 - b1) g
    v <- b2 v + (1 - b2) (g g)
    theta <- theta - (lr (m / c1)) / (sqrt(v / c2) + eps),   c1 = 1 - b1^t, c2 = 1 - b2^t (fp64 powers of the float32 b1, b2; rounded once)
Pins (tests/test_oracle_pins.py): the first step moves every parameter by lr * sign(g) up to eps (textbook property of
the bias correction); a constant gradient keeps |step| -> lr; against a fp64 re-derivation within rounding.
"""
from __future__ import annotations

import numpy as np


def adam_step(theta, g, m, v, lr, b1, b2, eps, t):
    f = np.float32
    theta, g, m, v = (np.asarray(a, dtype=np.float32) for a in (theta, g, m, v))
    one_b1, one_b2 = f(1.0) - f(b1), f(1.0) - f(b2)
    c1, c2 = f(1.0 - float(f(b1)) ** t), f(1.0 - float(f(b2)) ** t)      # b1, b2 are float32 values on both sides
    m2 = (f(b1) * m).astype(f) + (one_b1 * g).astype(f)
    v2 = (f(b2) * v).astype(f) + (one_b2 * (g * g).astype(f)).astype(f)
    mh = (m2 / c1).astype(f)
    vh = (v2 / c2).astype(f)
    th2 = theta - ((f(lr) * mh).astype(f) / (np.sqrt(vh).astype(f) + f(eps)).astype(f)).astype(f)
    return th2.astype(f), m2.astype(f), v2.astype(f)
