"""TEST INFRASTRUCTURE - fp64 NumPy oracle of the total-variation term L_tv of PAPER.md eq. 17 ("L_tv
is the total-variation on the sparse density field to reduce spurious high-frequency noise"). Only tests/ may import it.

The paper names the term and gives no formula. DESIGN.md reading R15: the field is the trilinear raw density of every
voxel (corner c = bx + 2 by + 4 bz), and its anisotropic (L1) total variation is taken over the 12 edges of each cell:

    L_tv = 1 / (12 N) * sum_v sum_{(a,b) in edges} | raw[v,a] - raw[v,b] |
    dL/draw[v,a] = 1 / (12 N) * sum_{b ~ a} sign(raw[v,a] - raw[v,b]),   sign(0) = 0

edges = the 12 corner pairs that differ in exactly one bit. With shared grid points (svr_gather_corners) the per-voxel
gradient is scatter-added to the grid (svr_scatter_add_corners), so an edge shared by k voxels counts k times.

Pins (tests/test_oracle_pins.py): a constant field has L = 0 and zero gradient; corners sampled from the linear field
alpha x + beta y + gamma z give (|alpha| + |beta| + |gamma|) / 3; L(s raw + c) = |s| L(raw); the gradient equals central
finite differences away from ties; every row of the gradient sums to zero.
PARITY UNPINNED (paper silent): L1 over cell edges, raw (pre-activation) values, the 1/(12 N) normalisation.
"""
from __future__ import annotations

import numpy as np

EDGES = [(c, c | (1 << a)) for a in range(3) for c in range(8) if not (c >> a) & 1]      # 12 pairs, a < b


def tv_loss_and_grad(raw: np.ndarray):
    """raw [n, 8] -> (L_tv, dL/draw [n, 8]) in fp64."""
    r = np.asarray(raw, dtype=np.float64)
    n = r.shape[0]
    grad = np.zeros_like(r)
    total = 0.0
    for a, b in EDGES:
        d = r[:, a] - r[:, b]
        total += float(np.abs(d).sum())
        sg = np.sign(d)
        grad[:, a] += sg
        grad[:, b] -= sg
    if n == 0:
        return 0.0, grad
    return total / (12.0 * n), grad / (12.0 * n)
