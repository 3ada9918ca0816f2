"""TEST INFRASTRUCTURE - fp64 oracle of the rendered-normal head (PAPER.md shows normal maps in Fig. 8,
P:312, and names depth-normal consistency terms L_NDm / L_NDM in eq. 17, but gives no formula). Only tests/ may
import it. DESIGN.md reading R16:

  * per-voxel normal: the trilinear raw-density field of voxel v has, at the cell centre q = (1/2, 1/2, 1/2), the gradient
        g_a = (sum of the 4 corner raws with b_a = 1  -  sum of the 4 with b_a = 0) / (4 e),   e = cell edge, corner c = bx + 2 by + 4 bz,
    n_v = -g / |g| (density falls along the outward normal), n_v = 0 where g = 0. World space, independent of the view.
  * rendered normal: N(p) = sum_k w_k n_{v_k} with the blending weights of eqs. 2-4; the background adds nothing. It is
    NOT re-normalised (|N| <= 1 - T_K), so it composes like a colour.
  * gradient of L = sum_p G_N(p) . N(p) w.r.t. the corner raws: through the weights (the compositing chain of the colour pass with
    n_v in the place of c_v and a zero background) and through n_v itself: dn/dg = -(I - n n^T) / |g|.

The compositing itself is NOT restated here: it is the pinned renderer of svr_oracle.cpp used as a library step, fed a degree-0 scene
whose colour is c'_v = (n_v + 1) / 2 in [0, 1] (never clamped) over a zero background: C' = (N + 1 - T_K) / 2, so
N = 2 C' - (1 - T_K), and dL/draw follows from orc_backward_heads with G = 2 G_N and G_T = sum_ch G_N.
Pins (tests/test_oracle_pins.py): the centre gradient of a linear field a + b.x is b exactly; a scene of voxels that all share
one normal renders N = (1 - T_K) n; central finite differences of sum(G_N . N) on an 8-voxel scene. PARITY UNPINNED: the whole
definition is the reading (the paper shows normal maps, not how they are made).
"""
from __future__ import annotations

from dataclasses import replace

import numpy as np

_Y0 = 0.28209479177387814      # 1 / (2 sqrt(pi)): the oracle's colour of a degree-0 voxel is max(0, 0.5 + Y0 sh0)
# sign of corner c = bx + 2 by + 4 bz along axis a: +1 if b_a = 1 else -1
_SIGN = np.array([[1.0 if (c >> a) & 1 else -1.0 for c in range(8)] for a in range(3)])


def voxel_gradients(scene, raw=None) -> np.ndarray:
    """g [n,3]: gradient of the trilinear raw field at the cell centre."""
    raw = np.asarray(scene.raw if raw is None else raw, dtype=np.float64)
    e = float(scene.root_edge) / np.exp2(scene.ijkl[:, 3].astype(np.float64))
    g = np.zeros((raw.shape[0], 3))
    for a in range(3):                                   # the four edges of the cell along axis a: far corner minus near corner
        for c in range(8):
            if not (c >> a) & 1:
                g[:, a] += raw[:, c | (1 << a)] - raw[:, c]
    return g / (4.0 * e[:, None])


def voxel_normals(scene, raw=None) -> np.ndarray:
    g = voxel_gradients(scene, raw)
    norm = np.sqrt((g * g).sum(1))
    n = np.zeros_like(g)
    ok = norm > 0
    n[ok] = -g[ok] / norm[ok, None]
    return n


def _normal_scene(scene, cam, raw=None):
    """Degree-0 copy of the scene whose colour is (n_v + 1) / 2, and the camera with a zero background."""
    n = voxel_normals(scene, raw)
    sh0 = (n / (2.0 * _Y0)).astype(np.float64)[:, None, :]              # 0.5 + Y0 sh0 = (n + 1) / 2
    sc = replace(scene, sh_degree=0, sh=sh0.astype(np.float32))         # (marshalled as float64 below through `sh=`)
    return sc, sh0, replace(cam, bg=np.zeros(3, dtype=np.float32)), n


def render_normals(orc, scene, cam, K: int, mode: str = "pure", xy=None, raw=None):
    """N [H,W,3] (or [n_rays,3]) and T_final."""
    sc, sh0, cam0, _ = _normal_scene(scene, cam, raw)
    r = orc.render(sc, cam0, K, mode=mode, xy=xy, raw=raw, sh=sh0)
    return 2.0 * r["image"] - (1.0 - r["T_final"])[..., None], r["T_final"]


def backward_normals(orc, scene, cam, K: int, G_N: np.ndarray, mode: str = "pure", xy=None, raw=None) -> np.ndarray:
    """d sum(G_N . N) / d raw [n,8]."""
    sc, sh0, cam0, n = _normal_scene(scene, cam, raw)
    G_N = np.asarray(G_N, dtype=np.float64)
    g_raw, g_sh = orc.backward(sc, cam0, K, 2.0 * G_N, mode=mode, xy=xy, raw=raw, sh=sh0, G_T=G_N.sum(axis=-1))
    # through n_v: dL/dc' = g_sh0 / Y0, dL/dn = dL/dc' / 2; dn/dg = -(I - n n^T) / |g|; dg_a/draw_c = sign[a,c] / (4 e)
    dLdn = g_sh[:, 0, :] / (2.0 * _Y0)
    g = voxel_gradients(scene, raw)
    norm = np.sqrt((g * g).sum(1))
    ok = norm > 0
    dLdg = np.zeros_like(g)
    dLdg[ok] = -(dLdn[ok] - n[ok] * (n[ok] * dLdn[ok]).sum(1, keepdims=True)) / norm[ok, None]
    e = float(scene.root_edge) / np.exp2(scene.ijkl[:, 3].astype(np.float64))
    return g_raw + (dLdg @ _SIGN) / (4.0 * e[:, None])
