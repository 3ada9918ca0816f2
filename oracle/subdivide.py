"""TEST INFRASTRUCTURE - NumPy oracle of priority-driven subdivision (Sec. IV-D, eqs. 13-16).
Only tests/ may import it. Steps in the paper's order; DESIGN.md "R12 subdivision" lists the readings.

  1. depth z_v and footprint delta_v as in oracle/prune.py.
  2. eq. 13: eligible iff level < max_level ("not at the finest octree level") and h_v > kappa * delta_v
     (and z_v finite: a voxel no camera sees in front of it cannot be resolved by any).
  3. eq. 14: z~ = clip((z - z_p5) / (z_p95 - z_p5), 0, 1), (z_p5, z_p95) = the 5th / 95th percentile of the
     finite depths (nearest rank) of THIS step, or the running values the caller passes; z_p95 <= z_p5 -> z~ = 0.
  4. eqs. 15-16: priority = P_v * (1 + beta * z~), P_v >= 0 the running usefulness score (an input).
  5. budget: the max_splits eligible voxels of highest priority split, ties by lower index.
  6. split 1 -> 8: children (2i + bx, 2j + by, 2k + bz, L + 1), child order c = bx + 2 by + 4 bz; child corner raws =
     the parent's trilinear field at the child's corners, i.e. at parent coordinates in {0, 1/2, 1}: interpolate along
     x, then y, then z with mix(a, b, 0) = a, mix(a, b, 1) = b, mix(a, b, 1/2) = 0.5 * (a + b) (float32, one rounding
     each); SH coefficients copied (BASELINE.json configs[4]: "seeded 1->8 subdivision").
  Output arrays: the unsplit voxels in their order, then the children grouped by parent in parent order.

Pins (tests/test_oracle_pins.py): eq. 13 on hand-made footprints; eqs. 14-16 against the formulas typed out with
numbers; budget and tie order; children tile the parent exactly and stay disjoint; child raws equal the fp64 trilinear
formula at the child corners and a second split of a child equals sampling the original field.
PARITY UNPINNED (paper silent): percentile convention, finite-depth rule, tie order, child raws, SH inheritance.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .prune import depth_proxy


@dataclass
class SubdivOpts:
    kappa: float = 1.0
    beta: float = 0.2
    max_level: int = 12
    max_splits: int = 1000
    use_current_percentiles: bool = True
    z_p5: float = 0.0
    z_p95: float = 0.0


def nearest_rank(v_sorted: np.ndarray, q: float) -> np.float32:
    rank = int(np.ceil(np.float32(np.float32(q) * np.float32(v_sorted.size))))
    return v_sorted[min(max(rank, 1), v_sorted.size) - 1]


def select_splits(scene, cams, P: np.ndarray, opts: SubdivOpts):
    """Steps 1-5. Returns dict(split [n] bool, priority [n] f32, eligible, z, delta, z_p5, z_p95)."""
    P = np.asarray(P, dtype=np.float32)
    z, delta, half = depth_proxy(scene, cams)
    finite = np.isfinite(z)
    level = scene.ijkl[:, 3].astype(np.int64)
    eligible = finite & (level < opts.max_level) & (half > (np.float32(opts.kappa) * delta).astype(np.float32))
    zf = np.sort(z[finite])
    p5 = nearest_rank(zf, 0.05) if zf.size else np.float32(0)
    p95 = nearest_rank(zf, 0.95) if zf.size else np.float32(0)
    a, b = (p5, p95) if opts.use_current_percentiles else (np.float32(opts.z_p5), np.float32(opts.z_p95))
    den = np.float32(b - a)
    with np.errstate(invalid="ignore", divide="ignore"):
        zt = ((z - a).astype(np.float32) / den).astype(np.float32) if den > 0 else np.zeros_like(z)
    zt = np.where(finite, np.minimum(np.maximum(zt, np.float32(0)), np.float32(1)), np.float32(0)).astype(np.float32)
    bias = (np.float32(1) + (np.float32(opts.beta) * zt).astype(np.float32)).astype(np.float32)        # eq. 15
    pr = (P * bias).astype(np.float32)                                                                  # eq. 16
    idx = np.flatnonzero(eligible)
    k = min(int(opts.max_splits), idx.size)
    split = np.zeros(scene.n, dtype=bool)
    if k > 0:
        order = np.lexsort((idx, -pr[idx].astype(np.float64)))           # highest priority first, ties by lower index
        split[idx[order[:k]]] = True
    return dict(split=split, priority=pr, eligible=eligible, z=z, delta=delta, z_p5=np.float32(p5), z_p95=np.float32(p95))


def _mix(a, b, t2):
    """t2 = 2 t in {0, 1, 2}."""
    if t2 == 0:
        return a
    if t2 == 2:
        return b
    return (np.float32(0.5) * (a + b).astype(np.float32)).astype(np.float32)


def child_raws(raw: np.ndarray) -> np.ndarray:
    """raw [m, 8] float32 (corner c = bx + 2 by + 4 bz) -> [m, 8 children, 8 corners]."""
    raw = np.asarray(raw, dtype=np.float32)
    out = np.empty((raw.shape[0], 8, 8), dtype=np.float32)
    for o in range(8):
        ox, oy, oz = o & 1, (o >> 1) & 1, o >> 2
        for c in range(8):
            tx, ty, tz = ox + (c & 1), oy + ((c >> 1) & 1), oz + (c >> 2)      # 2 x parent coordinate
            x00 = _mix(raw[:, 0], raw[:, 1], tx); x10 = _mix(raw[:, 2], raw[:, 3], tx)
            x01 = _mix(raw[:, 4], raw[:, 5], tx); x11 = _mix(raw[:, 6], raw[:, 7], tx)
            y0 = _mix(x00, x10, ty); y1 = _mix(x01, x11, ty)
            out[:, o, c] = _mix(y0, y1, tz)
    return out


def apply_splits(scene, split: np.ndarray):
    """Step 6. Returns (ijkl, raw, sh) of the new voxel set."""
    keep = np.flatnonzero(~split)
    par = np.flatnonzero(split)
    pij = scene.ijkl[par].astype(np.int64)
    ch = np.empty((par.size, 8, 4), dtype=np.int64)
    for o in range(8):
        ch[:, o, 0] = 2 * pij[:, 0] + (o & 1)
        ch[:, o, 1] = 2 * pij[:, 1] + ((o >> 1) & 1)
        ch[:, o, 2] = 2 * pij[:, 2] + (o >> 2)
        ch[:, o, 3] = pij[:, 3] + 1
    ijkl = np.concatenate([scene.ijkl[keep], ch.reshape(-1, 4).astype(scene.ijkl.dtype)])
    raw = np.concatenate([scene.raw[keep], child_raws(scene.raw[par]).reshape(-1, 8)])
    sh = np.concatenate([scene.sh[keep], np.repeat(scene.sh[par], 8, axis=0)])
    return ijkl, raw, sh


def carry_rows(rows: np.ndarray, split: np.ndarray, mode: str) -> np.ndarray:
    """Per-voxel side state through a split ("refresh the optimizer/scheduler after topology changes"; DESIGN.md
    reading R17). `rows` [n, ...] is any per-voxel array (EMA, hysteresis state, w_max, usefulness, Adam moments). The new
    array follows apply_splits' order: the unsplit voxels' rows in their order, then 8 rows per split voxel grouped by parent
    in parent order, each the parent's row (mode "copy": statistics the children inherit) or zero (mode "zero": state that
    restarts, e.g. Adam moments of parameters that did not exist before)."""
    if mode not in ("copy", "zero"):
        raise ValueError(mode)
    split = np.asarray(split, dtype=bool)
    keep = np.flatnonzero(~split)
    par = np.flatnonzero(split)
    out = np.empty((keep.size + 8 * par.size,) + rows.shape[1:], dtype=rows.dtype)
    for j, i in enumerate(keep):
        out[j] = rows[i]
    for j, i in enumerate(par):
        for o in range(8):
            out[keep.size + 8 * j + o] = rows[i] if mode == "copy" else 0
    return out
