"""Seeded scene / camera generators for configs C1..C5 (BASELINE.json `configs[0..4]`).

Layout only: which octree cells are leaves, what random numbers fill their parameters, where the
cameras sit. No rendering arithmetic lives here (see package docstring).

Conventions fixed here because both the oracle and the CUDA path consume them as *data*:
  * voxel = octree leaf (ix, iy, iz, level); edge = root_edge / 2**level; larger level = finer
    (reading R1 of PAPER.md line 74).
  * corner index c = bx + 2*by + 4*bz for `raw[n, 8]`.
  * camera: OpenCV axes, p_cam = R p_world + t, stored in float32 (both sides derive the centre
    o = -R^T t from these float32 values themselves).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Callable, List, Optional

import numpy as np

CONFIG_NAMES = ["C1", "C2", "C3", "C4", "C5"]
_SEEDS = {"C1": 1001, "C2": 1002, "C3": 1003, "C4": 1004, "C5": 1005}
# value of the constant (l = 0) real spherical harmonic, 1/(2 sqrt(pi)); used only to turn a drawn
# RGB into a degree-0 coefficient for C1 ("SH degree 0 RGB ~U(0,1)").
_Y0 = 0.28209479177387814
_BG = (0.2, 0.3, 0.4)


@dataclass
class Scene:
    root_lo: np.ndarray          # (3,) float32
    root_edge: float             # power of two
    max_level: int               # Lmax used for Morton codes (>= every voxel level)
    sh_degree: int
    ijkl: np.ndarray             # [n,4] uint16: ix, iy, iz, level
    raw: np.ndarray              # [n,8] float32 corner raw densities
    sh: np.ndarray               # [n,(D+1)^2,3] float32

    @property
    def n(self) -> int:
        return int(self.ijkl.shape[0])

    @property
    def n_basis(self) -> int:
        return (self.sh_degree + 1) ** 2


@dataclass
class Camera:
    W: int
    H: int
    fx: float
    fy: float
    cx: float
    cy: float
    R: np.ndarray                # (3,3) float32, world -> camera, row-major
    t: np.ndarray                # (3,) float32
    z_near: float = 0.01
    bg: np.ndarray = field(default_factory=lambda: np.array(_BG, dtype=np.float32))


@dataclass
class Config:
    name: str
    seed: int
    scene: Scene
    cameras: List[Camera]
    K: int
    T_min: float = 1e-5
    gamma: float = 0.6
    orbit_radius: float = 3.0
    target_kind: str = "uniform"   # "uniform" | "perturbed_render" | "noisy_render"
    target_noise: float = 0.05
    emit_wmax_in_backward: bool = False
    workspace_budget_bytes: int = 0


# ----------------------------------------------------------------------------------------------
# cameras
# ----------------------------------------------------------------------------------------------
def look_at_camera(pos, target, W: int, H: int, hfov_deg: float = 60.0, z_near: float = 0.01,
                   bg=_BG) -> Camera:
    """Pinhole looking from `pos` at `target`, world up = +z, horizontal field of view `hfov_deg`."""
    pos = np.asarray(pos, dtype=np.float64)
    target = np.asarray(target, dtype=np.float64)
    f = target - pos
    f /= np.linalg.norm(f)
    up = np.array([0.0, 0.0, 1.0])
    r = np.cross(f, up)
    r /= np.linalg.norm(r)
    dwn = np.cross(f, r)
    R = np.stack([r, dwn, f]).astype(np.float32)
    t = (-(R.astype(np.float64) @ pos)).astype(np.float32)
    fx = W / (2.0 * np.tan(np.deg2rad(hfov_deg) / 2.0))
    return Camera(W=W, H=H, fx=float(np.float32(fx)), fy=float(np.float32(fx)),
                  cx=float(W) / 2.0, cy=float(H) / 2.0, R=R, t=t, z_near=z_near,
                  bg=np.asarray(bg, dtype=np.float32))


def _orbit(radius, az_deg, el_deg=20.0):
    az, el = np.deg2rad(az_deg), np.deg2rad(el_deg)
    return radius * np.array([np.cos(el) * np.cos(az), np.cos(el) * np.sin(az), np.sin(el)])


# ----------------------------------------------------------------------------------------------
# shells and octrees
# ----------------------------------------------------------------------------------------------
class _Shells:
    """Union of ellipsoid shells; `dist` = approximate (radial) distance to the nearest shell.
    Above `full_level` only the `n_near` shells nearest to the node's coarse ancestor are evaluated
    (a recipe, not geometry: the generator only needs a deterministic refinement field)."""

    def __init__(self, centres: np.ndarray, A: np.ndarray):
        self.c = centres.astype(np.float32)        # [m,3]
        self.A = A.astype(np.float32)              # [m,3,3]: unit-sphere coords = A (x - c)
        self.m = self.c.shape[0]

    @staticmethod
    def random(rng, m, c_range=0.6, ax_lo=0.15, ax_hi=0.5):
        centres = rng.uniform(-c_range, c_range, size=(m, 3))
        axes = rng.uniform(ax_lo, ax_hi, size=(m, 3))
        A = np.empty((m, 3, 3))
        for i in range(m):
            q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
            A[i] = np.diag(1.0 / axes[i]) @ q.T
        return _Shells(centres, A)

    @staticmethod
    def sphere(centre, radius):
        return _Shells(np.asarray(centre, dtype=np.float64)[None], (np.eye(3) / radius)[None])

    def surface_points(self, rng, k):
        """k seeded points lying on the shells (centres of the fine-detail patches)."""
        sid = rng.integers(0, self.m, size=k)
        u = rng.normal(size=(k, 3))
        u /= np.linalg.norm(u, axis=1, keepdims=True)
        Ainv = np.linalg.inv(self.A.astype(np.float64))
        return self.c[sid].astype(np.float64) + np.einsum("kij,kj->ki", Ainv[sid], u)

    def _dist_one(self, xs, i):
        rel = xs - self.c[i]
        rn = np.sqrt(np.einsum("ij,ij->i", rel, rel))
        y = rel @ self.A[i].T
        f = np.sqrt(np.einsum("ij,ij->i", y, y))
        d = np.abs(rn * (1.0 - 1.0 / np.maximum(f, 1e-12)))
        return np.where(f < 1e-12, rn, d).astype(np.float32)

    def dist_all(self, x: np.ndarray) -> np.ndarray:
        """[n, m] distances to every shell (coarse levels only)."""
        x = x.astype(np.float32)
        return np.stack([self._dist_one(x, i) for i in range(self.m)], axis=1)

    def dist_near(self, x: np.ndarray, near: np.ndarray, chunk: int = 1 << 19) -> np.ndarray:
        """min over the shells listed per point in near[n, k]."""
        x = x.astype(np.float32)
        out = np.empty(x.shape[0], dtype=np.float32)
        for s in range(0, x.shape[0], chunk):
            xs, ids = x[s:s + chunk], near[s:s + chunk]
            rel = xs[:, None, :] - self.c[ids]                       # [n,k,3]
            rn = np.sqrt(np.einsum("nkj,nkj->nk", rel, rel))
            y = np.einsum("nkij,nkj->nki", self.A[ids], rel)
            f = np.sqrt(np.einsum("nki,nki->nk", y, y))
            d = np.abs(rn * (1.0 - 1.0 / np.maximum(f, 1e-12)))
            d = np.where(f < 1e-12, rn, d)
            out[s:s + chunk] = d.min(axis=1)
        return out

    def dist(self, x: np.ndarray) -> np.ndarray:
        return self.dist_all(x).min(axis=1)


def _children(ijk: np.ndarray) -> np.ndarray:
    off = np.array([[bx, by, bz] for bz in (0, 1) for by in (0, 1) for bx in (0, 1)], dtype=ijk.dtype)
    return (ijk[:, None, :] * 2 + off[None, :, :]).reshape(-1, 3)


def _grid(level: int) -> np.ndarray:
    g = np.arange(2 ** level, dtype=np.int64)
    return np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)


def _build_octree(root_lo, root_edge, start_ijk, start_level, max_level, level_fn, carry=None):
    """Top-down: a node at level L is subdivided while level_fn(centre, edge, L, carry) > L (and
    L < max_level); level_fn < 0 drops the node. `carry` is a per-node array inherited by children
    (level_fn returns (levels, carry)). Returns leaves (ijk[m,3], level[m], carry[m]) - disjoint."""
    root_lo = np.asarray(root_lo, dtype=np.float64)
    ijk, L = start_ijk, start_level
    out_ijk, out_l, out_c = [], [], []
    while ijk.shape[0] > 0:
        e = root_edge / 2 ** L
        ctr = root_lo + (ijk + 0.5) * e
        tl, carry = level_fn(ctr, e, L, carry)
        split = (tl > L) & (L < max_level)
        leaf = (~split) & (tl >= 0)
        out_ijk.append(ijk[leaf])
        out_l.append(np.full(int(leaf.sum()), L, dtype=np.int64))
        if carry is not None:
            out_c.append(carry[leaf])
            carry = np.repeat(carry[split], 8, axis=0)
        ijk = _children(ijk[split])
        L += 1
    return (np.concatenate(out_ijk), np.concatenate(out_l),
            np.concatenate(out_c) if out_c else None)


def _weighted_subsample(rng, weights: np.ndarray, n: int) -> np.ndarray:
    """Indices of n items drawn without replacement with probability ~ weights (Efraimidis-Spirakis)."""
    m = weights.shape[0]
    if m < n:
        raise ValueError(f"octree generator produced {m} candidate leaves, need {n}")
    u = rng.random(m)
    keys = np.log(np.maximum(u, 1e-300)) / np.maximum(weights, 1e-300)
    idx = np.argpartition(-keys, n - 1)[:n]
    return np.sort(idx)


def _pack(ijk, lvl) -> np.ndarray:
    out = np.empty((ijk.shape[0], 4), dtype=np.uint16)
    out[:, :3] = ijk
    out[:, 3] = lvl
    return out


def _shell_scene(rng, shells: _Shells, root_lo, root_edge, start_ijk, start_level, lmin, lmax, n,
                 n_detail=12, layers=1.5, full_level=6, n_near=4):
    """Exactly n disjoint leaves hugging `shells`.

    Finest level lmax only inside seeded "detail patches" (discs of radius r0 around points on the
    shells); each further r0 of distance from the nearest patch centre costs one level, down to lmin.
    Away from the surface the level also falls (one level per doubling of distance). r0 starts from
    the area estimate for n leaves and grows until the tree has >= 1.05 n candidate leaves; the
    leaves nearest the surface (weight exp(-dist / (0.5 edge))) are kept, so surfaces stay contiguous."""
    root_lo64 = np.asarray(root_lo, dtype=np.float64)
    e_f = root_edge / 2 ** lmax
    patches = shells.surface_points(rng, n_detail)
    r0 = e_f * np.sqrt(1.3 * n / (layers * n_detail * np.pi * 2.2))
    k = min(n_near, shells.m)

    def level_fn_factory(r0):
        def level_fn(ctr, e, L, near):
            if L <= full_level or near is None:
                dall = shells.dist_all(ctr)
                near = np.argsort(dall, axis=1)[:, :k].astype(np.int32)
                d = dall.min(axis=1)
            else:
                d = shells.dist_near(ctr, near)
            d_eff = np.maximum(d - 0.87 * e, 0.0)
            dp = np.sqrt(((ctr[:, None, :] - patches[None, :, :]) ** 2).sum(-1)).min(axis=1)
            pen = np.floor(np.maximum(dp - 0.87 * e, 0.0) / r0)
            tl = np.floor(lmax - pen - np.log2(1.0 + d_eff / (0.25 * e_f))).astype(np.int64)
            tl = np.clip(tl, lmin, lmax)
            tl = np.where(d_eff > 4.0 * e, -1, tl)            # empty space: drop the subtree
            tl = np.where((tl >= 0) & (L < lmin), np.maximum(tl, L + 1), tl)
            return tl, near
        return level_fn

    for _ in range(12):
        ijk, lvl, near = _build_octree(root_lo, root_edge, start_ijk, start_level, lmax,
                                       level_fn_factory(r0))
        if ijk.shape[0] >= int(1.05 * n):
            break
        r0 *= 1.35
    e = root_edge / np.power(2.0, lvl)
    ctr = root_lo64 + (ijk + 0.5) * e[:, None]
    d = shells.dist_near(ctr, near).astype(np.float64)
    w = np.exp(-np.minimum(d / (0.5 * e), 50.0))
    sel = _weighted_subsample(rng, w, n)
    return ijk[sel], lvl[sel]


def _params(rng, n, sh_degree, raw_mu, raw_sd, sh_sd):
    raw = rng.normal(raw_mu, raw_sd, size=(n, 8)).astype(np.float32)
    nb = (sh_degree + 1) ** 2
    sh = rng.normal(0.0, sh_sd, size=(n, nb, 3)).astype(np.float32)
    return raw, sh


# ----------------------------------------------------------------------------------------------
# small hand-sized scenes for pins / finite differences
# ----------------------------------------------------------------------------------------------
def uniform_grid_scene(level: int, seed: int, sh_degree: int = 0, raw_mu=-1.0, raw_sd=1.0) -> Scene:
    rng = np.random.Generator(np.random.PCG64(seed))
    ijk = _grid(level)
    n = ijk.shape[0]
    raw = rng.normal(raw_mu, raw_sd, size=(n, 8)).astype(np.float32)
    nb = (sh_degree + 1) ** 2
    sh = rng.normal(0.0, 0.3, size=(n, nb, 3)).astype(np.float32)
    rgb = rng.uniform(0.0, 1.0, size=(n, 3))
    sh[:, 0, :] = ((rgb - 0.5) / _Y0).astype(np.float32)
    return Scene(root_lo=np.array([-1, -1, -1], dtype=np.float32), root_edge=2.0, max_level=level,
                 sh_degree=sh_degree, ijkl=_pack(ijk, np.full(n, level)), raw=raw, sh=sh)


def tiny_scene(seed: int, n: int = 8, sh_degree: int = 1, max_level: int = 3) -> Scene:
    """<= 8-voxel mixed-level scene of disjoint leaves in [-1,1]^3 (finite-difference pins)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    ijk, lvl = _grid(1), np.ones(8, dtype=np.int64)
    for _ in range(2):                         # split two random leaves one level down
        cand = np.flatnonzero(lvl < max_level)
        j = int(rng.choice(cand))
        ch = _children(ijk[j:j + 1])
        ijk = np.concatenate([np.delete(ijk, j, axis=0), ch])
        lvl = np.concatenate([np.delete(lvl, j), np.full(8, lvl[j] + 1)])
    sel = np.sort(rng.choice(ijk.shape[0], size=n, replace=False))
    ijk, lvl = ijk[sel], lvl[sel]
    raw = rng.normal(-0.5, 1.0, size=(n, 8)).astype(np.float32)
    sh = rng.normal(0.0, 0.3, size=(n, (sh_degree + 1) ** 2, 3)).astype(np.float32)
    return Scene(root_lo=np.array([-1, -1, -1], dtype=np.float32), root_edge=2.0, max_level=max_level,
                 sh_degree=sh_degree, ijkl=_pack(ijk, lvl), raw=raw, sh=sh)


def perturbed_copy(scene: Scene, seed: int, raw_sd: float = 0.3, sh_sd: float = 0.05) -> Scene:
    rng = np.random.Generator(np.random.PCG64(seed))
    raw = (scene.raw + rng.normal(0, raw_sd, size=scene.raw.shape)).astype(np.float32)
    sh = (scene.sh + rng.normal(0, sh_sd, size=scene.sh.shape)).astype(np.float32)
    return replace(scene, raw=raw, sh=sh)


# ----------------------------------------------------------------------------------------------
# the five configs
# ----------------------------------------------------------------------------------------------
def _scaled_res(W, H, s):
    return max(16, int(round(W * s))), max(16, int(round(H * s)))


def _c1(seed, n_voxels, res_scale, n_cams):
    scene = uniform_grid_scene(3, seed, sh_degree=0)
    W, H = _scaled_res(64, 64, res_scale)
    cams = [look_at_camera(_orbit(3.0, 17.0), (0, 0, 0), W, H)]
    return Config("C1", seed, scene, cams, K=2, gamma=0.6, orbit_radius=3.0, target_kind="uniform")


def _c2(seed, n_voxels, res_scale, n_cams):
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_voxels or 50_000
    centre = rng.uniform(-0.05, 0.05, size=3)
    shells = _Shells.sphere(centre, 0.6)
    ijk, lvl = _shell_scene(rng, shells, (-1, -1, -1), 2.0, _grid(3), 3, 5, 8, n, n_detail=6)
    raw, sh = _params(rng, n, 1, -2.0, 1.5, 0.3)
    scene = Scene(np.array([-1, -1, -1], dtype=np.float32), 2.0, 8, 1, _pack(ijk, lvl), raw, sh)
    W, H = _scaled_res(256, 256, res_scale)
    cams = [look_at_camera(_orbit(3.0, 17.0 + 90.0 * i), (0, 0, 0), W, H) for i in range(n_cams or 4)]
    return Config("C2", seed, scene, cams, K=3, orbit_radius=3.0, target_kind="perturbed_render")


def _c3_leaves(rng, n, lmin=6, lmax=11, n_shells=20):
    shells = _Shells.random(rng, n_shells)
    # coarser trees for reduced sizes keep the generator fast in tests
    ijk, lvl = _shell_scene(rng, shells, (-1, -1, -1), 2.0, _grid(3), 3, lmin, lmax, n)
    return ijk, lvl


def _lmax_for(n, full_n, full_lmax, lmin):
    """Reduced copies of a config use a shallower tree so voxel footprints stay comparable."""
    if n >= full_n:
        return full_lmax
    drop = int(np.ceil(np.log2(full_n / n) / 2.0))       # surface count ~ 4^level
    return max(lmin + 1, full_lmax - drop)


def _first_fit(build, lmax0, lmax_full):
    """Reduced copies start from a shallower tree and deepen it until it holds enough leaves."""
    for lm in range(lmax0, lmax_full + 1):
        try:
            return lm, build(lm)
        except ValueError:
            if lm == lmax_full:
                raise


def _c3(seed, n_voxels, res_scale, n_cams):
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_voxels or 1_000_000
    lmax, (ijk, lvl) = _first_fit(lambda lm: _c3_leaves(rng, n, 6, lm), _lmax_for(n, 1_000_000, 11, 6), 11)
    raw, sh = _params(rng, n, 3, -3.0, 2.0, 0.2)
    scene = Scene(np.array([-1, -1, -1], dtype=np.float32), 2.0, lmax, 3, _pack(ijk, lvl), raw, sh)
    W, H = _scaled_res(980, 545, res_scale)
    m = n_cams or 8
    az = np.linspace(-35.0, 35.0, 8)[:m] if m <= 8 else np.linspace(-35.0, 35.0, m)
    cams = [look_at_camera(_orbit(2.2, 17.0 + a), (0, 0, 0), W, H) for a in az]
    return Config("C3", seed, scene, cams, K=3, orbit_radius=2.2, target_kind="noisy_render")


def _c4(seed, n_voxels, res_scale, n_cams):
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_voxels or 4_000_000
    n_bg = n // 10
    n_in = n - n_bg
    root_lo, root_edge = (-8.0, -8.0, -8.0), 16.0
    # inner cube [-1,1]^3 = the 8 level-4 cells around the origin
    inner = np.array([[i, j, k] for i in (7, 8) for j in (7, 8) for k in (7, 8)], dtype=np.int64)
    shells = _Shells.random(rng, 20)
    lmax, (ijk_i, lvl_i) = _first_fit(
        lambda lm: _shell_scene(rng, shells, root_lo, root_edge, inner, 4, 8, lm, n_in, full_level=7),
        _lmax_for(n, 4_000_000, 12, 8), 12)

    # background: level 4..7 leaves wholly outside the inner cube, centre radius <= 8
    p_leaf = {4: 0.0, 5: 0.05, 6: 0.15, 7: 1.0}

    def bg_level_fn(ctr, e, L, carry):
        r = np.sqrt((ctr ** 2).sum(1))
        is_inner = np.all(np.abs(ctr) < 1.0, axis=1)
        tl = np.where(rng.random(ctr.shape[0]) < p_leaf[L], L, L + 1)
        return np.where(is_inner | (r > 8.0), -1, tl), None

    ijk_b, lvl_b, _ = _build_octree(root_lo, root_edge, _grid(4), 4, 7, bg_level_fn)
    wb = np.power(2.0, lvl_b - 7.0)
    sel = _weighted_subsample(rng, wb, n_bg)
    ijk_b, lvl_b = ijk_b[sel], lvl_b[sel]

    ijk = np.concatenate([ijk_i, ijk_b])
    lvl = np.concatenate([lvl_i, lvl_b])
    perm = rng.permutation(n)                         # storage order carries no meaning
    ijk, lvl = ijk[perm], lvl[perm]
    raw, sh = _params(rng, n, 3, -3.0, 2.0, 0.2)
    scene = Scene(np.array(root_lo, dtype=np.float32), root_edge, lmax, 3, _pack(ijk, lvl), raw, sh)
    W, H = _scaled_res(1237, 822, res_scale)
    m = n_cams or 8
    cams = [look_at_camera(_orbit(2.5, 17.0 + 360.0 * i / 8), (0, 0, 0), W, H) for i in range(m)]
    return Config("C4", seed, scene, cams, K=3, orbit_radius=2.5, target_kind="noisy_render",
                  emit_wmax_in_backward=True)


def _split_leaves(rng, ijk, lvl, raw, sh, idx):
    """1 -> 8 split of leaves `idx`: children get the parent's trilinearly interpolated corner raws
    plus N(0, 0.1) and the parent's SH (scene recipe of C5)."""
    ch_ijk = _children(ijk[idx])                                    # [8m,3], child order bx+2by+4bz
    ch_lvl = np.repeat(lvl[idx] + 1, 8)
    p = raw[idx].astype(np.float64)                                 # [m,8]
    out = np.empty((idx.shape[0], 8, 8), dtype=np.float64)          # [m, child, corner]
    for child in range(8):
        cb = np.array([child & 1, (child >> 1) & 1, (child >> 2) & 1])
        for corner in range(8):
            kb = np.array([corner & 1, (corner >> 1) & 1, (corner >> 2) & 1])
            q = (cb + kb) / 2.0                                     # position in the parent cube
            val = np.zeros(idx.shape[0])
            for c in range(8):
                b = np.array([c & 1, (c >> 1) & 1, (c >> 2) & 1])
                wgt = np.prod(np.where(b == 1, q, 1.0 - q))
                if wgt != 0.0:
                    val += wgt * p[:, c]
            out[:, child, corner] = val
    ch_raw = (out.reshape(-1, 8) + rng.normal(0, 0.1, size=(idx.shape[0] * 8, 8))).astype(np.float32)
    ch_sh = np.repeat(sh[idx], 8, axis=0)
    keep = np.ones(ijk.shape[0], dtype=bool)
    keep[idx] = False
    return (np.concatenate([ijk[keep], ch_ijk]), np.concatenate([lvl[keep], ch_lvl]),
            np.concatenate([raw[keep], ch_raw]), np.concatenate([sh[keep], ch_sh]))


def _c5(seed, n_voxels, res_scale, n_cams, sh_degree=3):
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_voxels or 12_000_000
    base_level = 9 if n >= 2_000_000 else 7
    lmax = base_level + 3
    n_base = n // 8
    n_base += (n - n_base) % 7                                      # (n - n_base) must be 7 * splits
    shells = _Shells.random(rng, 20)
    ijk, lvl = _shell_scene(rng, shells, (-1, -1, -1), 2.0, _grid(3), 3, base_level, base_level, n_base)
    raw, sh = _params(rng, n_base, sh_degree, -3.0, 2.0, 0.2)
    W, H = _scaled_res(1600, 1066, res_scale)
    m = n_cams or 16
    radii = [1.4 if i % 2 == 0 else 2.5 for i in range(m)]
    pos = [_orbit(radii[i], 17.0 + 360.0 * i / 16) for i in range(m)]
    cams = [look_at_camera(p, (0, 0, 0), W, H) for p in pos]
    P = np.stack(pos)
    while ijk.shape[0] < n:
        cand = np.flatnonzero(lvl < lmax)
        need = (n - ijk.shape[0]) // 7
        e = 2.0 / np.power(2.0, lvl[cand])
        ctr = -1.0 + (ijk[cand] + 0.5) * e[:, None]
        d = np.min(np.sqrt(((ctr[:, None, :] - P[None, :, :]) ** 2).sum(-1)), axis=1)
        d *= rng.uniform(0.8, 1.25, size=d.shape[0])
        take = min(need, max(1, cand.shape[0] // 3))
        idx = cand[np.argpartition(d, take - 1)[:take]]
        ijk, lvl, raw, sh = _split_leaves(rng, ijk, lvl, raw, sh, np.sort(idx))
    perm = rng.permutation(n)
    scene = Scene(np.array([-1, -1, -1], dtype=np.float32), 2.0, lmax, sh_degree,
                  _pack(ijk[perm], lvl[perm]), raw[perm], sh[perm])
    return Config("C5", seed, scene, cams, K=3, orbit_radius=2.5, target_kind="noisy_render",
                  workspace_budget_bytes=32 << 30)


_BUILDERS = {"C1": _c1, "C2": _c2, "C3": _c3, "C4": _c4, "C5": _c5}


def make_config(name: str, n_voxels: Optional[int] = None, res_scale: float = 1.0,
                n_cams: Optional[int] = None, seed: Optional[int] = None) -> Config:
    """Config `name` at full size, or a reduced copy (fewer voxels / smaller images / fewer cameras)
    built by the same recipe for tests the CPU oracle must finish in seconds."""
    if name not in _BUILDERS:
        raise KeyError(name)
    return _BUILDERS[name](seed if seed is not None else _SEEDS[name], n_voxels, res_scale, n_cams)


def uniform_target(cam: Camera, seed: int) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.uniform(0.0, 1.0, size=(cam.H, cam.W, 3)).astype(np.float32)


def noisy_target(render: np.ndarray, seed: int, sigma: float = 0.05) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64(seed))
    return np.clip(render + rng.normal(0, sigma, size=render.shape), 0.0, 1.0).astype(np.float32)


def random_image_grad(cam: Camera, seed: int) -> np.ndarray:
    """A fixed random linear functional G for L = sum(G * image) (finite-difference pins)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.normal(0.0, 1.0, size=(cam.H, cam.W, 3))
