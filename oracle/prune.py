"""TEST INFRASTRUCTURE - NumPy oracle of depth-aware quantile pruning (Sec. IV-C, P:143-172,
eqs. 11-12 and guards i-iii). Only tests/ may import it. It follows the paper's order step by step; where the paper
is silent the reading is DESIGN.md "R11 pruning" (every constant is an argument, none is hidden here).

Steps (one adaptation step, all voxels of the scene, statistics gathered over the views given):
  1. depth proxy z_v ("group voxels by a depth proxy into bins"; P:185 names z_v "camera-space depth"):
     z_v = min over the cameras with Z_c(x_v) > 0 of the camera-space depth Z_c of the voxel centre, +inf if none;
     footprint delta_v = z_v / f_x (size of one pixel at that depth). float32, operations in the
     written order (the bins are integers decided by floating point: both sides use the same precision).
  2. bins V_b, b = 0..B-1: piecewise-linear log2 of z between the smallest and largest finite depth, taken on the
     float32 bit patterns (integer arithmetic, exact): b = min(B-1, (bits(z) - bits(z_min)) * B // (bits(z_max) -
     bits(z_min) + 1)); z = +inf -> bin B-1.
  3. eq. 11 / eq. 12: tau_b = F_b^{-1}(q_b) = nearest-rank quantile sorted_b[ceil(q_b |V_b|) - 1] of
     w_max over ALL voxels of the bin (never-seen voxels have w_max = 0); q_b = q_near + (q_far - q_near) b/(B-1)
     ("a mild near/far relaxation"; the annealing over training is the caller's, through q_near/q_far).
     "We prune v in V_b when w_max <= tau_b": inside score x_t = [w_max > tau_b].
  4. guard i: m_t = (1 - alpha) m_{t-1} + alpha x_t (float32); s_t = out if m_t < m_low, in if
     m_t > m_high, else s_{t-1}.
  5. guard ii (P:171 'Contour/detail dilation ("keep-halo")'): SEEDS are the voxels with h_v < kappa * delta_v ("small relative
     to the local ray footprint") or w_max >= w_keep ("high w_max"); protected = the seeds dilated `halo` times over the
     face-neighbour relation of the leaves (halo = 0: the seeds alone). Two leaves are face neighbours when their cells touch on
     one axis and overlap with positive area on the other two (any level difference); edge or corner contact does not count.
  6. guard iii: at most R = floor(cap_fraction * N) voxels leave per step: the candidates (state out, not
     protected) with the smallest w_max, ties by lower index.
Returns the new EMA, the new state, the keep mask, the thresholds and the bins.

Pins (tests/test_oracle_pins.py): the quantile against a sort written out; eq. 11 F_b(tau_b) >= q_b > F_b(tau_b^-);
the hysteresis on a hand-computed sequence; cap and protection invariants; one bin and no guards = a global quantile
cut; the keep-halo: a row of three cells, a gap of one empty cell, diagonal contact, a coarse cell beside fine ones, and the
neighbour pairs against the O(n^2) geometric definition on a random octree. PARITY UNPINNED (paper silent): the depth proxy, the bin edges, q_b's form, the inside score, kappa / w_keep
protection, the cap's choice among candidates.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class PruneOpts:
    n_bins: int = 8
    q_near: float = 0.10
    q_far: float = 0.05
    ema_alpha: float = 0.5
    m_low: float = 0.3
    m_high: float = 0.7
    kappa: float = 1.0
    w_keep: float = 0.5
    cap_fraction: float = 0.05
    halo: int = 0            # dilation steps of the keep-halo (guard ii)


def voxel_centres_f32(scene) -> np.ndarray:
    """x_v = root_lo + (i + 0.5) * edge in float32 (exact: edge is a power of two)."""
    ijkl = scene.ijkl.astype(np.int64)
    e = (np.float32(scene.root_edge) * np.exp2(-ijkl[:, 3].astype(np.float64)).astype(np.float32)).astype(np.float32)
    lo = np.asarray(scene.root_lo, dtype=np.float32)
    c = np.empty((scene.n, 3), dtype=np.float32)
    for a in range(3):
        c[:, a] = (lo[a] + (ijkl[:, a].astype(np.float32) + np.float32(0.5)) * e).astype(np.float32)
    return c, e


def depth_proxy(scene, cams):
    """Step 1. Returns (z [n] float32, delta [n] float32, half [n] float32)."""
    x, e = voxel_centres_f32(scene)
    z = np.full(scene.n, np.inf, dtype=np.float32)
    delta = np.full(scene.n, np.inf, dtype=np.float32)
    for cam in cams:
        R = np.asarray(cam.R, dtype=np.float32).reshape(3, 3)
        t = np.asarray(cam.t, dtype=np.float32)
        # Z = ((R20 x + R21 y) + R22 z) + t2, every operation rounded to float32
        Z = ((R[2, 0] * x[:, 0] + R[2, 1] * x[:, 1]).astype(np.float32) + (R[2, 2] * x[:, 2]).astype(np.float32)).astype(np.float32)
        Z = (Z + t[2]).astype(np.float32)
        ok = (Z > 0) & (Z < z)
        d = (Z / np.float32(cam.fx)).astype(np.float32)
        z = np.where(ok, Z, z)
        delta = np.where(ok, d, delta)
    return z, delta, (np.float32(0.5) * e).astype(np.float32)


def depth_bins(z: np.ndarray, n_bins: int):
    """Step 2: integer arithmetic on the float32 bit patterns (positive floats order like their bit patterns)."""
    bits = z.view(np.uint32).astype(np.int64)
    finite = np.isfinite(z)
    if not finite.any():
        return np.full(z.shape, n_bins - 1, dtype=np.int32), 0, 0
    lo, hi = int(bits[finite].min()), int(bits[finite].max())
    b = np.minimum(n_bins - 1, (np.clip(bits, lo, hi) - lo) * n_bins // (hi - lo + 1))
    b = np.where(finite, b, n_bins - 1)
    return b.astype(np.int32), lo, hi


def bin_quantiles(w_max: np.ndarray, bins: np.ndarray, opts: PruneOpts):
    """Step 3, eqs. 11-12: tau_b = sorted_b[ceil(q_b |V_b|) - 1]; an empty bin gets tau = -1 (nothing is <= it).
    ceil(q n) is evaluated in float32 (q n rounded once) so that both sides agree on the rank."""
    B = opts.n_bins
    tau = np.full(B, -1.0, dtype=np.float32)
    q = np.empty(B, dtype=np.float32)
    for b in range(B):
        frac = np.float32(b) / np.float32(max(B - 1, 1))
        q[b] = np.float32(opts.q_near) + (np.float32(opts.q_far) - np.float32(opts.q_near)) * frac
        v = np.sort(w_max[bins == b])
        if v.size:
            rank = int(np.ceil(np.float32(q[b] * np.float32(v.size))))
            rank = min(max(rank, 1), v.size)
            tau[b] = v[rank - 1]
    return tau, q


def face_neighbour_pairs(scene):
    """All pairs (a, b) of leaves that share part of a face, listed once from the side of the finer (or equal) leaf a: b is the
    leaf that covers the cell of a's size adjacent to one of a's six faces, i.e. that cell itself or one of its ancestors
    (leaves are disjoint, so at most one of them is a leaf; a coarser-to-finer contact appears from the finer side)."""
    ijkl = scene.ijkl.astype(np.int64)
    n = scene.n
    key_of = lambda L, x, y, z: (L << 48) | (x << 32) | (y << 16) | z          # level, ix, iy, iz: 16 bits each
    keys = key_of(ijkl[:, 3], ijkl[:, 0], ijkl[:, 1], ijkl[:, 2])
    order = np.argsort(keys, kind="stable")
    skeys = keys[order]
    A, B = [], []
    for axis in range(3):
        for step in (-1, 1):
            c = ijkl[:, :3].copy()
            c[:, axis] += step
            inside = (c[:, axis] >= 0) & (c[:, axis] < (1 << ijkl[:, 3]))      # the adjacent cell lies in the root cube
            for up in range(0, 17):                                            # the cell itself, its parent, grandparent, ...
                L = ijkl[:, 3] - up
                ok = inside & (L >= 0)
                if not ok.any():
                    break
                k = key_of(np.maximum(L, 0), c[:, 0] >> up, c[:, 1] >> up, c[:, 2] >> up)
                pos = np.searchsorted(skeys, k)
                hit = ok & (pos < n) & (skeys[np.minimum(pos, n - 1)] == k)
                a = np.flatnonzero(hit)
                A.append(a)
                B.append(order[pos[a]])
    return np.concatenate(A), np.concatenate(B)


def keep_halo(scene, seed: np.ndarray, steps: int) -> np.ndarray:
    """Guard ii: the seed set dilated `steps` times over the face-neighbour relation."""
    prot = np.asarray(seed, dtype=bool).copy()
    if steps <= 0:
        return prot
    a, b = face_neighbour_pairs(scene)
    for _ in range(steps):
        new = prot.copy()
        new[b[prot[a]]] = True
        new[a[prot[b]]] = True
        prot = new
    return prot


def prune_step(scene, cams, w_max: np.ndarray, ema: np.ndarray, state: np.ndarray, opts: PruneOpts):
    """One adaptation step. ema [n] float32 (m_{t-1}), state [n] uint8 (1 = in, 0 = out). Returns a dict."""
    w_max = np.asarray(w_max, dtype=np.float32)
    z, delta, half = depth_proxy(scene, cams)
    bins, _, _ = depth_bins(z, opts.n_bins)
    tau, q = bin_quantiles(w_max, bins, opts)
    x = (w_max > tau[bins]).astype(np.float32)                                  # inside score
    one_minus = np.float32(1.0) - np.float32(opts.ema_alpha)
    m = (one_minus * ema.astype(np.float32)).astype(np.float32) + (np.float32(opts.ema_alpha) * x).astype(np.float32)
    m = m.astype(np.float32)
    s = np.where(m < np.float32(opts.m_low), 0, np.where(m > np.float32(opts.m_high), 1, state)).astype(np.uint8)
    seed = (half < (np.float32(opts.kappa) * delta).astype(np.float32)) | (w_max >= np.float32(opts.w_keep))
    protected = keep_halo(scene, seed, opts.halo)
    cand = (s == 0) & ~protected
    R = int(np.floor(np.float32(opts.cap_fraction) * np.float32(scene.n)))
    remove = np.zeros(scene.n, dtype=bool)
    idx = np.flatnonzero(cand)
    if idx.size > R:
        order = np.lexsort((idx, w_max[idx]))                                   # by w_max, ties by lower index
        idx = idx[order[:R]]
    remove[idx] = True
    return dict(z=z, delta=delta, bins=bins, tau=tau, q=q, ema=m, state=s, seed=seed, protected=protected, candidates=cand,
                keep=~remove, n_removed=int(remove.sum()), cap=R)


def compact(scene, keep: np.ndarray):
    """Stable compaction of the voxel arrays (the order of the survivors is kept)."""
    k = np.flatnonzero(keep)
    return scene.ijkl[k], scene.raw[k], scene.sh[k]
