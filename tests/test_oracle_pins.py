"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only, -m "not gpu").

Each test names the passage (P:n = /root/reference/PAPER.md line n) or the closed form it holds the
oracle to. None of these retypes the oracle's own formula: they are closed forms, invariants, brute force
(point marching), finite differences and hand computations.
"""
import math
import os
from dataclasses import replace

import numpy as np
import pytest

from svr_inputs import Scene, look_at_camera, make_config, tiny_scene, uniform_grid_scene
from svr_inputs.scenes import random_image_grad

Y0 = 0.5 / math.sqrt(math.pi)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def one_voxel_scene(raw_value=0.3, rgb=(0.9, 0.5, 0.1), level=0, ijk=(0, 0, 0), root_edge=2.0):
    sh = ((np.array(rgb) - 0.5) / Y0).astype(np.float32).reshape(1, 1, 3)
    return Scene(root_lo=np.array([-1, -1, -1], dtype=np.float32), root_edge=root_edge, max_level=max(level, 1),
                 sh_degree=0, ijkl=np.array([[*ijk, level]], dtype=np.uint16),
                 raw=np.full((1, 8), raw_value, dtype=np.float32), sh=sh)


# ---------------------------------------------------------------------------------------------
# alpha from density, chord lengths (BASELINE.json north_star: alpha = 1 - exp(-sigma l))
# ---------------------------------------------------------------------------------------------
def test_single_constant_voxel_axis_ray(orc):
    raw0 = 0.3
    rgb = np.array([0.9, 0.5, 0.1])
    sc = one_voxel_scene(raw0, rgb)
    cam = look_at_camera((3.0, 0.0, 0.0), (0, 0, 0), 3, 3)          # centre pixel = optical axis, d = (-1,0,0)
    out = orc.render(sc, cam, K=3)
    sigma, ell = math.exp(float(np.float32(raw0))), 2.0                                 # axis-aligned ray through the centre: l = e
    alpha = 1.0 - math.exp(-sigma * ell)
    want = alpha * np.float32((rgb - 0.5) / Y0).astype(np.float64) * Y0 + alpha * 0.5 + (1 - alpha) * cam.bg.astype(np.float64)
    np.testing.assert_allclose(out["image"][1, 1], want, rtol=0, atol=1e-14)
    assert abs(out["T_final"][1, 1] - (1 - alpha)) < 1e-15
    assert abs(out["w_max"][0] - alpha) < 1e-15
    assert abs(out["depth"][1, 1] - alpha * 3.0) < 1e-14            # t_mid = distance to the cube centre


def test_diagonal_chord_is_sqrt3_e(orc):
    sc = one_voxel_scene(-1.0)
    cam = look_at_camera((2.0, 2.0, 2.0), (0, 0, 0), 3, 3)
    d = orc.ray_dump(sc, cam, 2, 1, 1)
    assert len(d["vox"]) == 1
    assert abs((d["t_out"][0] - d["t_in"][0]) - 2.0 * math.sqrt(3.0)) < 5e-6   # float32 R: direction off by ~1e-7
    assert abs(d["tau"][0] - math.exp(-1.0) * (d["t_out"][0] - d["t_in"][0])) < 1e-14


def test_chords_match_point_marching(orc):
    """Brute force: march 2e5 points along the ray and measure the length inside each box."""
    sc = tiny_scene(7, n=8, sh_degree=0)
    cam = look_at_camera((2.3, 1.1, 0.7), (0, 0.1, 0), 8, 8)
    e = sc.root_edge / 2.0 ** sc.ijkl[:, 3].astype(np.float64)
    lo = sc.root_lo.astype(np.float64) + sc.ijkl[:, :3] * e[:, None]
    n_steps, t_far = 200_000, 6.0
    t = (np.arange(n_steps) + 0.5) * (t_far / n_steps)
    total_hits = 0
    for (x, y) in [(0, 0), (3, 4), (4, 3), (7, 7), (2, 6)]:
        o, dirv = orc.ray(cam, x, y)
        assert abs(np.linalg.norm(dirv) - 1.0) < 1e-15             # P:68 unit direction
        pts = o[None, :] + t[:, None] * dirv[None, :]
        dump = orc.ray_dump(sc, cam, 2, x, y)
        got = dict(zip(dump["vox"].tolist(), (dump["t_out"] - dump["t_in"]).tolist()))
        for v in range(sc.n):
            inside = np.all((pts >= lo[v]) & (pts < lo[v] + e[v]), axis=1)
            length = inside.sum() * (t_far / n_steps)
            assert abs(length - got.get(v, 0.0)) < 3 * t_far / n_steps
        total_hits += len(got)
        mids = 0.5 * (dump["t_in"] + dump["t_out"])
        assert np.all(np.diff(mids) > 0)                            # front-to-back
    assert total_hits > 5


def test_K_independence_for_constant_raw(orc):
    sc = uniform_grid_scene(2, 5, sh_degree=0)
    sc = replace(sc, raw=np.repeat(sc.raw[:, :1], 8, axis=1))        # constant inside each voxel
    cam = look_at_camera((2.5, 0.9, 1.2), (0, 0, 0), 9, 7)
    ref = orc.render(sc, cam, K=1)["image"]
    for K in (2, 3, 4):
        np.testing.assert_allclose(orc.render(sc, cam, K=K)["image"], ref, rtol=0, atol=1e-14)
    # with constant raws, activating before or after interpolation is the same thing (reading R5)
    np.testing.assert_allclose(orc.render(sc, cam, K=3, act_mode=1)["image"], ref, rtol=0, atol=1e-14)


def test_exponential_density_closed_form(orc):
    """raw linear along the ray: tau -> (e^{a+b l} - e^a)/b, midpoint-rule error O(K^-2)."""
    a, b = -0.4, 0.8                                                 # raw(x) = a' + b' x on [-1,1]
    sc = one_voxel_scene(0.0)
    raw = np.array([[a + b * (-1.0 if (c & 1) == 0 else 1.0) for c in range(8)]], dtype=np.float32)
    sc = replace(sc, raw=raw)
    cam = look_at_camera((3.0, 0.0, 0.0), (0, 0, 0), 3, 3)           # ray travels x = 1 -> -1
    r64 = raw.astype(np.float64)[0]
    lo_v, hi_v = r64[0], r64[1]                                      # raw at x=-1 and x=+1
    slope = (lo_v - hi_v) / 2.0                                      # d raw / dt along the ray
    exact = (math.exp(hi_v + slope * 2.0) - math.exp(hi_v)) / slope
    errs = []
    for K in (1, 2, 4, 8):
        tau = orc.ray_dump(sc, cam, K, 1, 1)["tau"][0]
        errs.append(abs(tau - exact))
    assert errs[-1] < 2e-3 * exact
    for e0, e1 in zip(errs[:-1], errs[1:]):
        assert 3.5 < e0 / e1 < 4.5                                   # second-order convergence


# ---------------------------------------------------------------------------------------------
# compositing, eqs. 2-4, eq. 5
# ---------------------------------------------------------------------------------------------
def test_empty_scene_is_background(orc):
    sc = one_voxel_scene()
    empty = replace(sc, ijkl=sc.ijkl[:0], raw=sc.raw[:0], sh=sc.sh[:0])
    cam = look_at_camera((3.0, 1.0, 0.5), (0, 0, 0), 5, 4)
    out = orc.render(empty, cam, K=2)
    np.testing.assert_array_equal(out["image"], np.broadcast_to(cam.bg.astype(np.float64), (4, 5, 3)))
    assert np.all(out["depth"] == 0) and np.all(out["T_final"] == 1) and out["w_max"].size == 0
    # a voxel wholly behind the camera is never hit either (t >= 0)
    cam_away = look_at_camera((3.0, 0.0, 0.0), (6.0, 0.0, 0.0), 5, 4)
    out = orc.render(sc, cam_away, K=2)
    assert np.all(out["T_final"] == 1) and np.all(out["w_max"] == 0)


def test_weights_and_transmittance_sum_to_one(orc):
    cfg = make_config("C1")
    cam = cfg.cameras[0]
    for (x, y) in [(0, 0), (31, 32), (10, 50), (63, 63), (20, 20)]:
        d = orc.ray_dump(cfg.scene, cam, cfg.K, x, y)
        assert abs(d["w"].sum() + d["T_final"] - 1.0) < 1e-14
    out = orc.render(cfg.scene, cam, cfg.K)
    assert out["n_hits"].max() > 8


def test_two_voxel_hand_computation(orc):
    """Two stacked voxels on the optical axis: C = a1 c1 + (1-a1) a2 c2 + (1-a1)(1-a2) bg (eqs. 2-4)."""
    c1, c2 = np.array([0.8, 0.2, 0.4]), np.array([0.1, 0.7, 0.6])
    r1, r2 = -0.2, 0.5
    sh = np.stack([(c1 - 0.5) / Y0, (c2 - 0.5) / Y0]).astype(np.float32).reshape(2, 1, 3)
    # level-1 cells of [-1,1]^3: voxel A = [0,1]^3 (nearer to the camera at x=+4), voxel B = [-1,0]x[0,1]x[0,1]
    sc = Scene(np.array([-1, -1, -1], dtype=np.float32), 2.0, 1, 0,
               np.array([[1, 1, 1, 1], [0, 1, 1, 1]], dtype=np.uint16),
               np.array([[r1] * 8, [r2] * 8], dtype=np.float32), sh)
    cam = look_at_camera((4.0, 0.5, 0.5), (0.0, 0.5, 0.5), 3, 3)
    out = orc.render(sc, cam, K=2)
    a1 = 1 - math.exp(-math.exp(float(np.float32(r1))) * 1.0)
    a2 = 1 - math.exp(-math.exp(float(np.float32(r2))) * 1.0)
    c1f = sh[0, 0].astype(np.float64) * Y0 + 0.5
    c2f = sh[1, 0].astype(np.float64) * Y0 + 0.5
    want = a1 * c1f + (1 - a1) * a2 * c2f + (1 - a1) * (1 - a2) * cam.bg.astype(np.float64)
    np.testing.assert_allclose(out["image"][1, 1], want, rtol=0, atol=1e-14)
    np.testing.assert_allclose(out["w_max"], [a1, (1 - a1) * a2], rtol=0, atol=1e-15)
    assert abs(out["depth"][1, 1] - (a1 * 3.5 + (1 - a1) * a2 * 4.5)) < 1e-13
    # storing the two voxels in the other order changes nothing
    sc2 = replace(sc, ijkl=sc.ijkl[::-1].copy(), raw=sc.raw[::-1].copy(), sh=sc.sh[::-1].copy())
    out2 = orc.render(sc2, cam, K=2)
    np.testing.assert_array_equal(out2["image"], out["image"])


def test_storage_order_invariance_and_wmax(orc):
    cfg = make_config("C1")
    sc, cam = cfg.scene, look_at_camera((2.0, 1.5, 1.0), (0, 0, 0), 12, 12)
    out = orc.render(sc, cam, cfg.K)
    perm = np.random.default_rng(3).permutation(sc.n)
    scp = replace(sc, ijkl=sc.ijkl[perm], raw=sc.raw[perm], sh=sc.sh[perm])
    outp = orc.render(scp, cam, cfg.K)
    np.testing.assert_array_equal(outp["image"], out["image"])
    np.testing.assert_array_equal(outp["depth"], out["depth"])
    np.testing.assert_array_equal(outp["w_max"], out["w_max"][perm])
    # eq. 5: w_max equals the max over rays of the dumped per-ray weights; 0 <=> never hit
    wm = np.zeros(sc.n)
    hit = np.zeros(sc.n, dtype=bool)
    for y in range(cam.H):
        for x in range(cam.W):
            d = orc.ray_dump(sc, cam, cfg.K, x, y)
            np.maximum.at(wm, d["vox"], d["w"])
            hit[d["vox"]] = True
    np.testing.assert_array_equal(out["w_max"], wm)
    assert np.all((out["w_max"] >= 0) & (out["w_max"] <= 1))
    assert np.array_equal(out["w_max"] > 0, hit)


def test_mirror_symmetry(orc):
    """Mirroring scene and camera in x mirrors the image left-right."""
    sc = tiny_scene(11, n=8, sh_degree=0)
    cam = look_at_camera((2.2, 0.8, 0.9), (0.1, 0.0, 0.0), 10, 8)
    n_side = (1 << sc.ijkl[:, 3].astype(np.int64))
    ijkl_m = sc.ijkl.copy()
    ijkl_m[:, 0] = (n_side - 1 - sc.ijkl[:, 0]).astype(np.uint16)
    swap = [c ^ 1 for c in range(8)]                                  # corner bx -> 1 - bx
    scm = replace(sc, ijkl=ijkl_m, raw=sc.raw[:, swap].copy())
    camm = look_at_camera((-2.2, 0.8, 0.9), (-0.1, 0.0, 0.0), 10, 8)
    a = orc.render(sc, cam, 3)
    b = orc.render(scm, camm, 3)
    np.testing.assert_allclose(b["image"][:, ::-1], a["image"], rtol=0, atol=1e-6)   # float32 R, t differ in rounding
    np.testing.assert_allclose(b["w_max"], a["w_max"], rtol=0, atol=1e-6)


def _n_straddlers(scene, cam):
    """voxels that cross the camera plane (some corner behind z = 1e-6, some in front): the oracle's bucketed mode sends
    them to every block"""
    e = scene.root_edge / 2.0 ** scene.ijkl[:, 3].astype(np.float64)
    lo = scene.root_lo.astype(np.float64) + scene.ijkl[:, :3] * e[:, None]
    zmin, zmax = np.full(scene.n, np.inf), np.full(scene.n, -np.inf)
    for k in range(8):
        z = (lo + e[:, None] * np.array([k & 1, (k >> 1) & 1, (k >> 2) & 1])) @ cam.R[2].astype(np.float64) + float(cam.t[2])
        zmin, zmax = np.minimum(zmin, z), np.maximum(zmax, z)
    return int(((zmin < 1e-6) & (zmax > 0)).sum())


def test_bucketed_equals_pure(orc):
    """The bucketed mode (the reference of every C3-C5 parity test) reproduces the pure mode, including on a reduced C4 whose
    camera sits among background cells that cross the camera plane (the 'zmin < 1e-6 -> every block' branch)."""
    c4 = make_config("C4", n_voxels=6000, res_scale=0.1, n_cams=1)
    assert _n_straddlers(c4.scene, c4.cameras[0]) >= 5
    for cfg in (make_config("C1"), make_config("C2", n_voxels=3000, res_scale=0.25, n_cams=1), c4):
        cam = cfg.cameras[0]
        a = orc.render(cfg.scene, cam, cfg.K, mode="pure")
        b = orc.render(cfg.scene, cam, cfg.K, mode="bucketed")
        for k in ("image", "depth", "T_final", "w_max", "n_hits"):
            np.testing.assert_array_equal(a[k], b[k])
        G = random_image_grad(cam, 5)
        ga = orc.backward(cfg.scene, cam, cfg.K, G, mode="pure")
        gb = orc.backward(cfg.scene, cam, cfg.K, G, mode="bucketed")
        np.testing.assert_allclose(ga[0], gb[0], rtol=1e-12, atol=1e-15)
        np.testing.assert_allclose(ga[1], gb[1], rtol=1e-12, atol=1e-15)


# ---------------------------------------------------------------------------------------------
# SH basis (textbook closed forms; reading R6)
# ---------------------------------------------------------------------------------------------
def test_sh_orthonormal_by_quadrature(orc):
    xs, ws = np.polynomial.legendre.leggauss(24)                      # z = cos(theta)
    n_phi = 48
    phi = (np.arange(n_phi) + 0.5) * (2 * math.pi / n_phi)
    z, p = np.meshgrid(xs, phi, indexing="ij")
    s = np.sqrt(1 - z * z)
    dirs = np.stack([s * np.cos(p), s * np.sin(p), z], -1).reshape(-1, 3)
    wq = (ws[:, None] * np.full(n_phi, 2 * math.pi / n_phi)[None, :]).reshape(-1)
    Y = orc.sh_basis(3, dirs)
    gram = (Y * wq[:, None]).T @ Y
    assert np.abs(gram - np.eye(16)).max() < 1e-12
    assert abs(Y[0, 0] - 0.5 / math.sqrt(math.pi)) < 1e-16
    for l in range(4):                                                # addition theorem
        band = (Y[:, l * l:(l + 1) * (l + 1)] ** 2).sum(1)
        assert np.abs(band - (2 * l + 1) / (4 * math.pi)).max() < 1e-14
    # lower degrees are prefixes of degree 3
    np.testing.assert_array_equal(orc.sh_basis(1, dirs[:5]), Y[:5, :4])
    # band l=1 is linear in (y, z, x): fixes the index convention i = l(l+1)+m
    d = np.array([[0.0, 1.0, 0.0], [0.0, 0.0, 1.0], [1.0, 0.0, 0.0]])
    Y1 = orc.sh_basis(1, d)[:, 1:4]
    np.testing.assert_allclose(Y1, math.sqrt(3 / (4 * math.pi)) * np.eye(3), atol=1e-16)


def test_voxel_colour_clamp_and_direction(orc):
    sc = tiny_scene(3, n=6, sh_degree=2)
    sh = sc.sh.copy()
    sh[0, 0, :] = -8.0                                               # forces a clamped (black) voxel
    sc = replace(sc, sh=sh)
    cam = look_at_camera((1.9, -1.2, 0.8), (0, 0, 0), 4, 4)
    rgb, pre = orc.voxel_rgb(sc, cam)
    assert np.all(rgb[0] == 0) and np.all(pre[0] < 0)
    o, _ = orc.ray(cam, 0, 0)
    e = sc.root_edge / 2.0 ** sc.ijkl[:, 3].astype(np.float64)
    ctr = sc.root_lo.astype(np.float64) + (sc.ijkl[:, :3] + 0.5) * e[:, None]
    dirs = ctr - o
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    want = 0.5 + np.einsum("vi,vic->vc", orc.sh_basis(2, dirs), sc.sh.astype(np.float64))
    np.testing.assert_allclose(pre, want, rtol=0, atol=1e-14)
    np.testing.assert_array_equal(rgb, np.maximum(pre, 0.0))


# ---------------------------------------------------------------------------------------------
# gradients: central finite differences on <= 8-voxel scenes (north_star), closed form for sh0
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,deg", [(21, 1), (22, 3)])
def test_gradients_match_finite_differences(orc, seed, deg):
    sc = tiny_scene(seed, n=8, sh_degree=deg)
    sh = sc.sh.copy()
    sh[1, 0, 1] = -6.0                                               # one clamped channel (zero sub-gradient)
    sc = replace(sc, sh=sh)
    cam = look_at_camera((2.1, 0.7, 1.3), (0.05, -0.1, 0.0), 11, 9)
    G = random_image_grad(cam, seed)
    raw0, sh0 = sc.raw.astype(np.float64), sc.sh.astype(np.float64)
    g_raw, g_sh = orc.backward(sc, cam, 3, G)

    def L(raw, shv):
        return float((orc.render(sc, cam, 3, raw=raw, sh=shv)["image"] * G).sum())

    h = 1e-6
    rng = np.random.default_rng(seed)
    scale = max(np.abs(g_raw).max(), np.abs(g_sh).max())
    for idx in [tuple(rng.integers(0, s) for s in raw0.shape) for _ in range(40)]:
        rp, rm = raw0.copy(), raw0.copy()
        rp[idx] += h
        rm[idx] -= h
        fd = (L(rp, sh0) - L(rm, sh0)) / (2 * h)
        assert abs(fd - g_raw[idx]) < 2e-7 * scale + 1e-9, (idx, fd, g_raw[idx])
    for idx in [tuple(rng.integers(0, s) for s in sh0.shape) for _ in range(40)] + [(1, 0, 1)]:
        sp, sm = sh0.copy(), sh0.copy()
        sp[idx] += h
        sm[idx] -= h
        fd = (L(raw0, sp) - L(raw0, sm)) / (2 * h)
        assert abs(fd - g_sh[idx]) < 2e-7 * scale + 1e-9, (idx, fd, g_sh[idx])
    assert g_sh[1, 0, 1] == 0.0
    assert np.abs(g_raw).max() > 1e-3 and np.abs(g_sh).max() > 1e-3


def test_sh0_gradient_closed_form(orc):
    """dL/dsh[v,0,ch] = Y_0 sum_rays w(v,ray) G[ray,ch] (where unclamped), from the forward dump."""
    sc = tiny_scene(31, n=8, sh_degree=0)
    cam = look_at_camera((2.4, 1.0, 0.6), (0, 0, 0), 7, 6)
    G = random_image_grad(cam, 31)
    _, g_sh = orc.backward(sc, cam, 2, G)
    want = np.zeros((sc.n, 3))
    for y in range(cam.H):
        for x in range(cam.W):
            d = orc.ray_dump(sc, cam, 2, x, y)
            for v, w in zip(d["vox"], d["w"]):
                want[v] += Y0 * w * G[y, x]
    _, pre = orc.voxel_rgb(sc, cam)
    want *= (pre > 0)
    np.testing.assert_allclose(g_sh[:, 0, :], want, rtol=1e-12, atol=1e-15)


# ---------------------------------------------------------------------------------------------
# part B: rectangles, keys, ranges
# ---------------------------------------------------------------------------------------------
def test_rect_hand_projection(orc):
    """Voxel [0,1]^3 seen from (4,.5,.5) along -x, 64x64, 60 deg hFoV: near face at Z=3 spans
    u,v = 32 +- (32/tan30)(0.5/3) = [22.76, 41.24] -> pixels 22..41."""
    sc = one_voxel_scene(level=1, ijk=(1, 1, 1))
    cam = look_at_camera((4.0, 0.5, 0.5), (0.0, 0.5, 0.5), 64, 64)
    half = (32.0 / math.tan(math.radians(30.0))) * (0.5 / 3.0)
    rects, masks, E = orc.bin_rects(sc, cam)
    assert rects[0].tolist() == [math.floor(32 - half), math.floor(32 - half), math.floor(32 + half), math.floor(32 + half)]
    assert rects[0].tolist() == [22, 22, 41, 41]
    # tiles 1..2 in x and y; the optical axis (-x direction) splits the image into 4 direction octants
    n_ent = sum(bin(int(masks[j * 4 + i])).count("1") for j in (1, 2) for i in (1, 2))
    assert E == n_ent
    # behind the camera: culled; camera inside the voxel: whole image
    cam_away = look_at_camera((4.0, 0.5, 0.5), (8.0, 0.5, 0.5), 64, 64)
    assert orc.bin_rects(sc, cam_away)[0][0].tolist() == [65535, 65535, 0, 0]
    cam_in = look_at_camera((0.4, 0.5, 0.6), (-1.0, 0.2, 0.1), 64, 48)
    assert orc.bin_rects(sc, cam_in)[0][0].tolist() == [0, 0, 63, 47]
    # beside the camera, crossing its plane but outside the frustum: culled by the side test
    sc_side = one_voxel_scene(level=2, ijk=(3, 0, 1))                 # [0.5,1]x[-1,-0.5]x[-0.5,0]
    cam_side = look_at_camera((0.9, 0.9, 0.0), (0.9, 5.0, 0.0), 64, 48)
    assert orc.bin_rects(sc_side, cam_side)[0][0].tolist() == [65535, 65535, 0, 0]


def _check_lists_against_rays(orc, cfg, cam, pixels):
    sc = cfg.scene
    lists = orc.bin_lists(sc, cam)
    tx = (cam.W + 15) // 16
    keys, vals, ranges = lists["keys"], lists["vals"], lists["ranges"]
    assert np.all(keys[1:] > keys[:-1])                               # total order: codes of disjoint leaves are unique
    n_checked = 0
    for (x, y) in pixels:
        s = orc.pixel_octant(cam, x, y)
        tile = (y >> 4) * tx + (x >> 4)
        assert (lists["tile_masks"][tile] >> s) & 1
        a, b = ranges[tile, s]
        seg = vals[a:b]
        d = orc.ray_dump(sc, cam, cfg.K, x, y)
        pos = {int(v): i for i, v in enumerate(seg)}
        where = [pos.get(int(v), -1) for v in d["vox"]]
        assert all(w >= 0 for w in where), "an fp64 hit has no list entry (binning not conservative)"
        assert all(w1 > w0 for w0, w1 in zip(where[:-1], where[1:])), "key order != t_mid order"
        n_checked += len(where)
    return n_checked


def test_key_order_equals_depth_order_C1(orc):
    cfg = make_config("C1")
    cam = cfg.cameras[0]
    pix = [(x, y) for y in range(0, cam.H, 3) for x in range(0, cam.W, 3)]
    assert _check_lists_against_rays(orc, cfg, cam, pix) > 500


def test_key_order_equals_depth_order_mixed_levels(orc):
    cfg = make_config("C2", n_voxels=4000, res_scale=0.25, n_cams=2)
    for cam in cfg.cameras:
        rng = np.random.default_rng(9)
        pix = [(int(rng.integers(0, cam.W)), int(rng.integers(0, cam.H))) for _ in range(150)]
        assert _check_lists_against_rays(orc, cfg, cam, pix) > 50
    # a camera inside the scene: several direction octants per image, straddling voxels
    cam_in = look_at_camera((0.31, 0.27, 0.13), (-0.5, 0.4, -0.1), 48, 40)
    pix = [(x, y) for y in range(1, 40, 5) for x in range(1, 48, 5)]
    assert _check_lists_against_rays(orc, cfg, cam_in, pix) > 50
    masks = orc.bin_lists(cfg.scene, cam_in)["tile_masks"]
    assert max(bin(int(m)).count("1") for m in masks) >= 2


def test_ranges_partition_the_lists(orc):
    cfg = make_config("C2", n_voxels=3000, res_scale=0.25, n_cams=1)
    cam = cfg.cameras[0]
    L = orc.bin_lists(cfg.scene, cam)
    Lm = cfg.scene.max_level
    prefix = (L["keys"] >> np.uint64(3 * Lm)).astype(np.int64)
    r = L["ranges"].reshape(-1, 2).astype(np.int64)
    covered = 0
    for p in range(r.shape[0]):
        a, b = r[p]
        if b > a:
            assert np.all(prefix[a:b] == p)
            covered += b - a
        else:
            assert a == 0 and b == 0
    assert covered == L["keys"].size
    code_mask = np.uint64((1 << (3 * Lm)) - 1)
    # voxel id is recoverable from the key's Morton part: un-flip and compare with the voxel's own code
    v = L["vals"][:50]
    assert np.all(L["rects"][v, 0] <= L["rects"][v, 2])
    assert np.all((L["keys"][:50] & code_mask) < np.uint64(1 << (3 * Lm)))


# ---------------------------------------------------------------------------------------------
# loss (eqs. 7-10)
# ---------------------------------------------------------------------------------------------
def test_gamma_schedule_eq9(orc):
    T = 20000.0
    assert orc.gamma_schedule(0.3 * T - 1, T) == 0.0
    assert orc.gamma_schedule(0.3 * T, T) == 0.0
    assert abs(orc.gamma_schedule(0.45 * T, T) - 0.3) < 1e-15
    assert orc.gamma_schedule(0.6 * T, T) == 0.6
    assert orc.gamma_schedule(T, T) == 0.6


def test_loss_reduces_to_baseline_at_gamma0(orc):
    rng = np.random.default_rng(0)
    R, I = rng.uniform(size=(9, 11, 3)), rng.uniform(size=(9, 11, 3))
    L, dL, wt = orc.lf_loss_and_grad(R, I, 0.0)
    assert np.all(wt == 1.0)                                          # P:141 "reduces exactly"
    assert abs(L - np.abs(R - I).mean()) < 1e-15
    np.testing.assert_allclose(dL, np.sign(R - I) / (3 * 99), rtol=0, atol=1e-18)


def test_loss_weights_mean_one_and_direction(orc):
    rng = np.random.default_rng(1)
    I = np.zeros((16, 20, 3))
    I[:, 10:] = 1.0                                                   # one vertical edge, flat elsewhere
    I += rng.normal(0, 1e-3, size=I.shape)
    R = I + rng.normal(0, 0.1, size=I.shape)
    L, dL, wt = orc.lf_loss_and_grad(R, I, 0.6)
    assert abs(wt.mean() - 1.0) < 1e-14                               # eq. 8
    assert wt[:, 9:11].max() < wt[:, :8].min()                        # edges down-weighted, flats amplified
    fd_L = orc.lf_loss_and_grad(R + 1e-7 * np.sign(R - I), I, 0.6)[0]
    assert abs((fd_L - L) / 1e-7 - np.abs(dL).sum()) < 1e-6
    # constant target: s = 0 everywhere, weights 1
    _, _, wc = orc.lf_loss_and_grad(R, np.full_like(I, 0.3), 0.6)
    np.testing.assert_allclose(wc, 1.0, rtol=0, atol=1e-15)


def test_sobel_of_a_ramp(orc):
    a, b = 0.01, -0.02
    yy, xx = np.meshgrid(np.arange(12.0), np.arange(15.0), indexing="ij")
    img = np.repeat((a * xx + b * yy)[:, :, None], 3, axis=2)
    m = orc.sobel_magnitude(img)
    np.testing.assert_allclose(m[1:-1, 1:-1], math.hypot(8 * a, 8 * b), rtol=1e-12)


def test_sh_quadrature_golden_fixture(orc):
    """tests/golden/sh_l1_axes.txt: band-1 value on its own axis sqrt(3/(4 pi)) and Y_0 = 1/(2 sqrt(pi)) (textbook table of the
    real SH basis, cited in the file) against the ORACLE's basis evaluated on the three axes (index i = l(l+1)+m: y, z, x)."""
    vals = [float(x) for x in open(os.path.join(GOLDEN, "sh_l1_axes.txt")).read().split("\n") if x and not x.startswith("#")]
    Y = orc.sh_basis(1, np.eye(3))                                     # rows: dir = +x, +y, +z
    np.testing.assert_allclose(Y[:, 0], vals[1], rtol=0, atol=1e-15)
    np.testing.assert_allclose([Y[1, 1], Y[2, 2], Y[0, 3]], vals[0], rtol=0, atol=1e-15)   # Y_1,-1(y), Y_1,0(z), Y_1,1(x)
    assert abs(Y[0, 1]) + abs(Y[0, 2]) + abs(Y[1, 2]) + abs(Y[1, 3]) + abs(Y[2, 1]) + abs(Y[2, 3]) < 1e-15


def test_lf_weights_closed_form_on_a_step_edge(orc):
    """eq. 7 by VALUE (w = (eps + 1 - s)^gamma, eps = 1e-3; eq. 8). A two-level target with one vertical step
    of height a has Sobel magnitude exactly 4a on the two columns beside the step and 0 elsewhere (kernel column sums 1+2+1).
    With 10 % of the pixels on the edge the 0.99-quantile is 4a, so s = 1 on the edge and 0 on the flats:
    w_edge / w_flat = (eps / (1 + eps))^gamma and w~ = w / mean(w) in closed form."""
    H, W, a, gamma, eps = 12, 20, 0.375, 0.6, 1e-3
    I = np.zeros((H, W, 3))
    I[:, 9:] = a
    m = orc.sobel_magnitude(I)
    np.testing.assert_allclose(m[:, 8:10], 4 * a, rtol=1e-15)
    assert np.count_nonzero(m) == 2 * H
    from oracle.loss import lf_weights
    wt = lf_weights(I, gamma, eps, 0.99)
    w_e, w_f = eps ** gamma, (1.0 + eps) ** gamma
    mean = (2 * H * w_e + (W - 2) * H * w_f) / (W * H)
    np.testing.assert_allclose(wt[:, 8:10], w_e / mean, rtol=1e-13)
    np.testing.assert_allclose(np.delete(wt, [8, 9], axis=1), w_f / mean, rtol=1e-13)
    np.testing.assert_allclose(wt[0, 8] / wt[0, 0], (eps / (1.0 + eps)) ** gamma, rtol=1e-13)
    # the same through the loss: L = mean over pixels of w~ |r|, r = 0.1 everywhere
    L, dL, _ = orc.lf_loss_and_grad(I + 0.1, I, gamma, eps, 0.99)
    assert abs(L - 0.1) < 1e-15                                       # mean(w~) = 1
    np.testing.assert_allclose(dL[:, 8, 0], (w_e / mean) / (3 * W * H), rtol=1e-13)


def test_lf_quantile_is_nearest_rank(orc):
    """R10: m_q = sorted[ceil(q |P|) - 1]. A 20 x 20 lattice of 25 isolated dots of height a: each dot gives 4 pixels with
    |grad| = 2a (edge neighbours: kernel weight 2), 4 with sqrt(2) a (corner neighbours: gx = gy = a) and a zero at its centre:
    100 pixels at 2a, 100 at sqrt(2) a, 200 zeros. With q = 0.75 (exact in binary), q |P| = 300: the nearest rank is sorted[299]
    = sqrt(2) a, so BOTH rings saturate (s = 1); floor(q |P|) = sorted[300] or the maximum would give 2a and s = 0.707 on the
    corner ring."""
    a, gamma, eps = 0.5, 0.6, 1e-3
    I = np.zeros((20, 20, 3))
    I[1::4, 1::4] = a
    m = orc.sobel_magnitude(I)
    vals, counts = np.unique(np.round(m.reshape(-1), 12), return_counts=True)
    np.testing.assert_allclose(vals, [0.0, math.sqrt(2) * a, 2 * a], rtol=1e-12)
    assert counts.tolist() == [200, 100, 100]
    from oracle.loss import lf_weights
    wt = lf_weights(I, gamma, eps, 0.75)
    w_ring, w_flat = eps ** gamma, (1.0 + eps) ** gamma
    mean = (200 * w_ring + 200 * w_flat) / 400
    np.testing.assert_allclose(wt[m > 0], w_ring / mean, rtol=1e-12)  # corner ring saturated too: m_q = sqrt(2) a
    np.testing.assert_allclose(wt[m == 0], w_flat / mean, rtol=1e-12)
    # one rank higher (q |P| = 301 > 300) the quantile moves to 2a and the corner ring gets s = 1/sqrt(2)
    wt2 = lf_weights(I, gamma, eps, 0.7501)
    w_corner = (eps + 1.0 - 1.0 / math.sqrt(2)) ** gamma
    mean2 = (100 * w_ring + 100 * w_corner + 200 * w_flat) / 400
    np.testing.assert_allclose(wt2[np.isclose(m, math.sqrt(2) * a)], w_corner / mean2, rtol=1e-12)


# ---------------------------------------------------------------------------------------------
# depth-aware quantile pruning (Sec. IV-C): pins of oracle/prune.py
# ---------------------------------------------------------------------------------------------
def _prune_case(n=6000, seed=5):
    from svr_inputs import make_config
    cfg = make_config("C2", n_voxels=n)
    rng = np.random.default_rng(seed)
    w = (rng.random(cfg.scene.n) ** 3).astype(np.float32)
    w[rng.random(cfg.scene.n) < 0.25] = 0.0                     # never-seen voxels
    return cfg, w


def test_prune_quantile_is_eq11_eq12():
    """tau_b = F_b^{-1}(q_b) (eq. 12) with F_b the empirical CDF of eq. 11: F_b(tau_b) >= q_b and no
    smaller sample value reaches q_b. Checked against the CDF written out per sample, not against a sort."""
    from oracle.prune import PruneOpts, bin_quantiles, depth_bins, depth_proxy
    cfg, w = _prune_case()
    opts = PruneOpts(n_bins=5, q_near=0.4, q_far=0.15)
    z, _, _ = depth_proxy(cfg.scene, cfg.cameras)
    bins, _, _ = depth_bins(z, opts.n_bins)
    tau, q = bin_quantiles(w, bins, opts)
    assert np.isclose(q[0], 0.4) and np.isclose(q[-1], 0.15) and np.all(np.diff(q) < 0)
    for b in range(opts.n_bins):
        v = w[bins == b]
        assert v.size > 0
        F = lambda t: np.count_nonzero(v <= t) / v.size          # eq. 11
        assert F(tau[b]) >= q[b] - 1e-7
        smaller = v[v < tau[b]]
        if smaller.size:
            assert F(smaller.max()) < q[b] + 1e-7


def test_prune_depth_proxy_on_axis_and_bins_monotone():
    from oracle.prune import depth_bins, depth_proxy
    from svr_inputs import look_at_camera, tiny_scene
    sc = tiny_scene(1, n=1, sh_degree=0)                         # one voxel
    x = np.asarray(sc.root_lo, dtype=np.float64) + (sc.ijkl[0, :3] + 0.5) * sc.root_edge / 2.0 ** sc.ijkl[0, 3]
    pos = x + np.array([0.0, -2.5, 0.0])
    cam = look_at_camera(tuple(pos), tuple(x), 64, 48)
    z, delta, half = depth_proxy(sc, [cam])
    assert abs(z[0] - 2.5) < 1e-5 and abs(delta[0] - 2.5 / cam.fx) < 1e-7     # on the optical axis depth = distance
    assert half[0] == np.float32(0.5 * sc.root_edge / 2.0 ** sc.ijkl[0, 3])
    behind = look_at_camera(tuple(pos), tuple(2 * pos - x), 64, 48)           # looking away: no positive depth
    assert np.isinf(depth_proxy(sc, [behind])[0][0])
    zz = np.array([0.5, 0.7, 1.01, 1.9, 2.01, 3.9, 4.0, np.inf], dtype=np.float32)
    b, lo, hi = depth_bins(zz, 3)
    assert np.all(np.diff(b) >= 0) and b[0] == 0 and b[-1] == 2 and b[-2] == 2
    assert list(b[:7]) == [0, 0, 1, 1, 2, 2, 2]                  # bit patterns are piecewise-linear in log2: octaves 0.5-1-2-4


def test_prune_hysteresis_hand_sequence():
    """Guard i on one voxel, alpha = 0.5, m_low = 0.3, m_high = 0.7, starting in with m = 1:
    x = 0,0,1,0,0,1,1 -> m = .5,.25,.625,.3125,.15625,.578125,.7890625 -> in,out,out,out,out,out,in."""
    from oracle.prune import PruneOpts, prune_step
    from svr_inputs import look_at_camera, tiny_scene
    sc = tiny_scene(2, n=2, sh_degree=0)
    cam = look_at_camera((3.0, 1.0, 0.5), (0, 0, 0), 64, 48)
    opts = PruneOpts(n_bins=1, q_near=0.5, q_far=0.5, ema_alpha=0.5, m_low=0.3, m_high=0.7, kappa=0.0, w_keep=2.0, cap_fraction=0.0)
    m, s = np.ones(2, np.float32), np.ones(2, np.uint8)
    got_m, got_s = [], []
    for x in [0, 0, 1, 0, 0, 1, 1]:
        # two voxels, q = 0.5 -> tau = the smaller w_max: voxel 0 is "inside" iff it holds the larger value
        w = np.array([0.9, 0.1], np.float32) if x else np.array([0.1, 0.9], np.float32)
        r = prune_step(sc, [cam], w, m, s, opts)
        m, s = r["ema"], r["state"]
        got_m.append(float(m[0])); got_s.append(int(s[0]))
        assert r["n_removed"] == 0                               # cap_fraction = 0: guard iii removes nothing
    assert np.allclose(got_m, [.5, .25, .625, .3125, .15625, .578125, .7890625], atol=0)
    assert got_s == [1, 0, 0, 0, 0, 0, 1]


def test_prune_guards_and_global_cut():
    from oracle.prune import PruneOpts, prune_step
    cfg, w = _prune_case()
    n = cfg.scene.n
    ones, ins = np.zeros(n, np.float32), np.zeros(n, np.uint8)   # m_{t-1} = 0, state out: every low voxel is a candidate
    # one bin, no protection, no cap: exactly the global quantile cut w_max <= tau
    o = PruneOpts(n_bins=1, q_near=0.3, q_far=0.3, ema_alpha=1.0, m_low=0.5, m_high=0.5, kappa=0.0, w_keep=2.0, cap_fraction=1.0)
    r = prune_step(cfg.scene, cfg.cameras, w, ones, ins, o)
    tau = np.sort(w)[int(np.ceil(np.float32(0.3) * np.float32(n))) - 1]
    assert r["tau"][0] == tau and np.array_equal(r["keep"], w > tau)
    # cap: at most floor(f N) leave, and they are the smallest candidates; protected voxels never leave
    o2 = PruneOpts(n_bins=4, q_near=0.5, q_far=0.3, ema_alpha=1.0, m_low=0.5, m_high=0.5, kappa=0.5, w_keep=0.6, cap_fraction=0.02)
    r2 = prune_step(cfg.scene, cfg.cameras, w, ones, ins, o2)
    removed = ~r2["keep"]
    assert r2["n_removed"] == min(r2["cap"], int(r2["candidates"].sum())) == int(np.floor(np.float32(0.02) * np.float32(n)))
    assert not np.any(removed & r2["protected"]) and np.all(r2["candidates"][removed])
    assert w[removed].max() <= w[r2["candidates"] & ~removed].min()
    assert np.all(w[r2["protected"] & (w < 0.6)] >= 0) and np.all(r2["protected"][w >= 0.6])
    # q -> 0 with all-positive w_max: tau = min, only the minimum is "outside"
    wp = np.maximum(w, 1e-3).astype(np.float32)
    o3 = PruneOpts(n_bins=1, q_near=1e-9, q_far=1e-9, ema_alpha=1.0, m_low=0.5, m_high=0.5, kappa=0.0, w_keep=2.0, cap_fraction=1.0)
    r3 = prune_step(cfg.scene, cfg.cameras, wp, ones, ins, o3)
    assert np.array_equal(~r3["keep"], wp <= wp.min())


def _cells_scene(cells):
    """Scene of the given (ix, iy, iz, level) leaves in [0,1]^3 (parameters irrelevant to the keep-halo)."""
    ijkl = np.array(cells, dtype=np.uint16)
    n = ijkl.shape[0]
    return Scene(np.zeros(3, np.float32), 1.0, 6, 0, ijkl, np.zeros((n, 8), np.float32), np.zeros((n, 1, 3), np.float32))


def _touching_brute_force(ijkl, lmax=8):
    """O(n^2) geometric definition of the face-neighbour relation in integer coordinates at level lmax: the cells touch on one
    axis and overlap with positive length on the other two."""
    size = 1 << (lmax - ijkl[:, 3].astype(np.int64))
    lo = ijkl[:, :3].astype(np.int64) * size[:, None]
    hi = lo + size[:, None]
    pairs = set()
    for a in range(ijkl.shape[0]):
        for b in range(a + 1, ijkl.shape[0]):
            for ax in range(3):
                o1, o2 = (ax + 1) % 3, (ax + 2) % 3
                touch = hi[a, ax] == lo[b, ax] or hi[b, ax] == lo[a, ax]
                over = min(hi[a, o1], hi[b, o1]) > max(lo[a, o1], lo[b, o1]) and min(hi[a, o2], hi[b, o2]) > max(lo[a, o2], lo[b, o2])
                if touch and over:
                    pairs.add((a, b))
    return pairs


def test_keep_halo_dilation():
    """Guard ii as a dilation: hand cases, then the neighbour pairs against the geometric definition."""
    from oracle.prune import face_neighbour_pairs, keep_halo
    # a row of three level-2 cells: only the middle one is a seed -> all three protected after one step
    row = _cells_scene([(0, 1, 1, 2), (1, 1, 1, 2), (2, 1, 1, 2)])
    assert keep_halo(row, [False, True, False], 1).tolist() == [True, True, True]
    assert keep_halo(row, [True, False, False], 1).tolist() == [True, True, False]      # one step reaches one cell ...
    assert keep_halo(row, [True, False, False], 2).tolist() == [True, True, True]       # ... two steps reach two
    assert keep_halo(row, [True, False, False], 0).tolist() == [True, False, False]
    # no protection across a gap of one empty cell, none across an edge or a corner
    gap = _cells_scene([(0, 1, 1, 2), (2, 1, 1, 2), (1, 2, 1, 2), (1, 2, 2, 2)])          # cell (1,1,1) is empty
    assert keep_halo(gap, [True, False, False, False], 1).tolist() == [True, False, False, False]   # (1,2,1) touches (0,1,1) by an edge only
    # a level-1 cell beside the four level-2 cells on its +x face, and four more one cell further
    fine = [(2, y, z, 2) for y in (0, 1) for z in (0, 1)] + [(3, y, z, 2) for y in (0, 1) for z in (0, 1)]
    mixed = _cells_scene([(0, 0, 0, 1)] + fine)
    assert keep_halo(mixed, [True] + [False] * 8, 1).tolist() == [True] + [True] * 4 + [False] * 4   # coarse seed: the touching four
    one = [False] * 9
    one[2] = True                                                                                     # fine seed (2,0,1): the coarse cell,
    got = keep_halo(mixed, one, 1)                                                                   # its three face neighbours
    want = [True, True, True, False, True, False, True, False, False]
    #        coarse (2,0,0) (2,0,1)s (2,1,0) (2,1,1) (3,0,0) (3,0,1) (3,1,0) (3,1,1)
    assert got.tolist() == want
    # random octree: the pairs found through ancestor look-ups are exactly the geometric ones
    cfg = make_config("C2", n_voxels=700)
    a, b = face_neighbour_pairs(cfg.scene)
    found = {(min(i, j), max(i, j)) for i, j in zip(a.tolist(), b.tolist())}
    assert found == _touching_brute_force(cfg.scene.ijkl) and len(found) > 200
    seed = np.random.default_rng(3).random(cfg.scene.n) < 0.05
    prot = keep_halo(cfg.scene, seed, 1)
    nb = np.zeros(cfg.scene.n, dtype=bool)
    for i, j in found:
        nb[i] |= seed[j]
        nb[j] |= seed[i]
    assert np.array_equal(prot, seed | nb)


def test_prune_step_with_halo_protects_neighbours():
    from oracle.prune import PruneOpts, prune_step
    cfg, w = _prune_case()
    n = cfg.scene.n
    m0, s0 = np.zeros(n, np.float32), np.zeros(n, np.uint8)
    base = dict(n_bins=4, q_near=0.5, q_far=0.3, ema_alpha=1.0, m_low=0.5, m_high=0.5, kappa=0.0, w_keep=0.8, cap_fraction=1.0)
    r0 = prune_step(cfg.scene, cfg.cameras, w, m0, s0, PruneOpts(**base, halo=0))
    r1 = prune_step(cfg.scene, cfg.cameras, w, m0, s0, PruneOpts(**base, halo=1))
    assert np.array_equal(r0["seed"], r1["seed"]) and np.array_equal(r0["protected"], r0["seed"])
    assert np.all(r1["protected"][r1["seed"]]) and r1["protected"].sum() > r0["protected"].sum()
    assert np.all(r1["keep"][r1["protected"]]) and r1["n_removed"] < r0["n_removed"]     # the halo saved some low-w_max neighbours
    saved = r1["keep"] & ~r0["keep"]
    assert saved.any() and not np.any(saved & r1["seed"])


# ---------------------------------------------------------------------------------------------
# rendered normals (NEXT-3; reading R16): pins of oracle/normals.py
# ---------------------------------------------------------------------------------------------
def test_normals_linear_field_and_shared_normal(orc):
    from oracle import normals
    sc = tiny_scene(7, n=8, sh_degree=1)
    # corner raws sampled from a linear field a + b . x: the centre gradient of the trilinear interpolant is b exactly
    b = np.array([0.7, -1.3, 0.4])
    e = sc.root_edge / 2.0 ** sc.ijkl[:, 3].astype(np.float64)
    lo = sc.root_lo.astype(np.float64) + sc.ijkl[:, :3] * e[:, None]
    corners = np.array([[c & 1, (c >> 1) & 1, (c >> 2) & 1] for c in range(8)], dtype=np.float64)
    raw = -1.0 + ((lo[:, None, :] + corners[None, :, :] * e[:, None, None]) @ b)
    np.testing.assert_allclose(normals.voxel_gradients(sc, raw), np.broadcast_to(b, (sc.n, 3)), rtol=1e-12, atol=1e-12)
    n = normals.voxel_normals(sc, raw)
    np.testing.assert_allclose(n, np.broadcast_to(-b / np.linalg.norm(b), (sc.n, 3)), rtol=1e-12)
    assert np.all(normals.voxel_normals(sc, np.full((sc.n, 8), 0.3)) == 0.0)            # constant field: no normal
    # every voxel has the same normal: N(p) = (sum_k w_k) n = (1 - T_K) n on every ray (eqs. 2-4: sum w + T_K = 1)
    cam = look_at_camera((2.3, 0.9, 1.4), (0.0, 0.1, 0.0), 24, 18)
    N, Tf = normals.render_normals(orc, sc, cam, 3, raw=raw)
    np.testing.assert_allclose(N, (1.0 - Tf)[..., None] * (-b / np.linalg.norm(b)), rtol=0, atol=1e-13)
    assert (1.0 - Tf).max() > 0.3
    # general scene: |N| <= 1 - T_K, and N equals the weighted sum over the dumped hits of one ray
    N2, Tf2 = normals.render_normals(orc, sc, cam, 3)
    assert np.all(np.linalg.norm(N2, axis=-1) <= 1.0 - Tf2 + 1e-12)
    nv = normals.voxel_normals(sc)
    for (x, y) in [(12, 9), (5, 11), (17, 6)]:
        d = orc.ray_dump(sc, cam, 3, x, y)
        np.testing.assert_allclose(N2[y, x], (d["w"][:, None] * nv[d["vox"]]).sum(0), rtol=0, atol=1e-13)


def test_normals_gradient_matches_finite_differences(orc):
    from oracle import normals
    sc = tiny_scene(11, n=8, sh_degree=0)
    cam = look_at_camera((2.2, -0.8, 1.1), (0.0, 0.0, 0.1), 16, 12)
    rng = np.random.default_rng(2)
    G = rng.normal(0, 1, size=(cam.H, cam.W, 3))
    raw0 = sc.raw.astype(np.float64)
    g = normals.backward_normals(orc, sc, cam, 2, G, raw=raw0)
    assert np.abs(g).max() > 1e-3
    L = lambda r: float((G * normals.render_normals(orc, sc, cam, 2, raw=r)[0]).sum())
    h = 1e-6
    for (v, c) in [(0, 0), (1, 5), (3, 2), (4, 7), (6, 1), (7, 3)]:
        rp, rm = raw0.copy(), raw0.copy()
        rp[v, c] += h
        rm[v, c] -= h
        fd = (L(rp) - L(rm)) / (2 * h)
        assert abs(fd - g[v, c]) <= 2e-6 * max(1.0, abs(fd)), (v, c, fd, g[v, c])


# ---------------------------------------------------------------------------------------------
# priority-driven subdivision (Sec. IV-D, eqs. 13-16): pins of oracle/subdivide.py
# ---------------------------------------------------------------------------------------------
def test_subdivide_eligibility_priority_budget():
    from oracle.prune import depth_proxy
    from oracle.subdivide import SubdivOpts, select_splits
    from svr_inputs import make_config
    cfg = make_config("C2", n_voxels=5000)
    sc = cfg.scene
    rng = np.random.default_rng(2)
    P = rng.random(sc.n).astype(np.float32)
    P[::7] = np.float32(0.5)                                     # ties
    o = SubdivOpts(kappa=0.8, beta=0.25, max_level=8, max_splits=150)
    r = select_splits(sc, cfg.cameras, P, o)
    z, delta, half = depth_proxy(sc, cfg.cameras)
    # eq. 13 typed out in float64 on the same inputs (strict inequality, not at the finest level)
    elig = np.isfinite(z) & (sc.ijkl[:, 3] < 8) & (half.astype(np.float64) > 0.8 * delta.astype(np.float64) * (1 + 1e-6))
    assert np.all(r["eligible"][elig]) and 0 < r["eligible"].sum() < sc.n
    assert not np.any(r["eligible"] & (sc.ijkl[:, 3] >= 8))
    # eqs. 14-16 with numbers
    zf = np.sort(z[np.isfinite(z)].astype(np.float64))
    p5, p95 = zf[int(np.ceil(0.05 * zf.size)) - 1], zf[int(np.ceil(0.95 * zf.size)) - 1]
    assert abs(p5 - r["z_p5"]) < 1e-6 and abs(p95 - r["z_p95"]) < 1e-6
    zt = np.clip((z.astype(np.float64) - p5) / (p95 - p5), 0, 1)
    assert np.allclose(r["priority"], P * (1 + 0.25 * zt), rtol=1e-6)
    assert np.all(r["priority"] >= P) and np.all(r["priority"] <= P * np.float32(1.25) * (1 + 1e-6))   # b in [1, 1 + beta]
    # budget: exactly max_splits eligible voxels, none of lower priority than an unsplit eligible one
    s = r["split"]
    assert s.sum() == 150 and np.all(r["eligible"][s])
    lo, hi = r["priority"][s].min(), r["priority"][r["eligible"] & ~s].max()
    assert lo >= hi
    tie = r["eligible"] & (r["priority"] == lo)
    if (tie & s).any() and (tie & ~s).any():
        assert np.flatnonzero(tie & s).max() < np.flatnonzero(tie & ~s).min()        # ties by lower index
    # given (running) percentiles instead of this step's
    r2 = select_splits(sc, cfg.cameras, P, SubdivOpts(kappa=0.8, beta=0.25, max_level=8, max_splits=150, use_current_percentiles=False,
                                                      z_p5=2.0, z_p95=2.0))
    assert np.array_equal(r2["priority"], P)                     # degenerate range: z~ = 0


def test_subdivide_carry_rows_hand_case_and_alignment_with_the_new_topology():
    """oracle/subdivide.carry_rows (reading R17): a hand case typed out, and the property that makes it usable: row j of
    the carried array belongs to voxel j of apply_splits' new voxel set (an unsplit voxel keeps its own row; a child carries its
    parent's row, identified through the child's cell index halved) - the rows of ijkl itself serve as the carried payload."""
    from oracle import subdivide
    rows = np.array([[10, 11], [20, 21], [30, 31], [40, 41]], dtype=np.float32)
    split = np.array([False, True, False, True])
    got = subdivide.carry_rows(rows, split, "copy")
    want = np.array([[10, 11], [30, 31]] + [[20, 21]] * 8 + [[40, 41]] * 8, dtype=np.float32)
    np.testing.assert_array_equal(got, want)
    got0 = subdivide.carry_rows(rows, split, "zero")
    np.testing.assert_array_equal(got0, np.array([[10, 11], [30, 31]] + [[0, 0]] * 16, dtype=np.float32))
    assert got0.dtype == rows.dtype
    np.testing.assert_array_equal(subdivide.carry_rows(rows, np.zeros(4, dtype=bool), "zero"), rows)      # no split: identity
    state = np.array([1, 0, 1, 1], dtype=np.uint8)                                                        # 1-D, one byte per voxel
    np.testing.assert_array_equal(subdivide.carry_rows(state, split, "copy"), np.array([1, 1] + [0] * 8 + [1] * 8, dtype=np.uint8))
    with pytest.raises(ValueError):
        subdivide.carry_rows(rows, split, "mean")
    # alignment with apply_splits on a mixed-level scene
    sc = tiny_scene(321, n=8, sh_degree=1)
    rng = np.random.default_rng(5)
    split = rng.random(sc.n) < 0.4
    split[0], split[1] = True, False
    ijkl_new, _, sh_new = subdivide.apply_splits(sc, split)
    carried = subdivide.carry_rows(sc.ijkl, split, "copy").astype(np.int64)
    n_keep = int((~split).sum())
    np.testing.assert_array_equal(carried[:n_keep], ijkl_new[:n_keep])
    ch = ijkl_new[n_keep:].astype(np.int64)
    np.testing.assert_array_equal(ch[:, :3] // 2, carried[n_keep:, :3])
    np.testing.assert_array_equal(ch[:, 3] - 1, carried[n_keep:, 3])
    np.testing.assert_array_equal(subdivide.carry_rows(sc.sh, split, "copy"), sh_new)      # SH is carried by copy (R12)


def test_subdivide_children_tile_parent_and_sample_its_field():
    from oracle.subdivide import apply_splits, child_raws
    from svr_inputs import tiny_scene
    sc = tiny_scene(4, n=6, sh_degree=1)
    split = np.array([True, False, True, False, False, True])
    ijkl, raw, sh = apply_splits(sc, split)
    assert ijkl.shape[0] == 3 + 24 and np.array_equal(ijkl[:3], sc.ijkl[~split])
    def box(q, root_edge):
        e = root_edge / 2.0 ** q[3]
        return q[:3] * e, (q[:3] + 1) * e
    for k, p in enumerate(np.flatnonzero(split)):
        plo, phi = box(sc.ijkl[p].astype(np.float64), sc.root_edge)
        vol = 0.0
        for o in range(8):
            c = ijkl[3 + 8 * k + o].astype(np.float64)
            clo, chi = box(c, sc.root_edge)
            assert np.all(clo >= plo) and np.all(chi <= phi) and c[3] == sc.ijkl[p, 3] + 1
            off = (clo - plo) / (chi - clo)
            assert tuple(off.astype(int)) == (o & 1, (o >> 1) & 1, o >> 2)          # child order bx + 2 by + 4 bz
            vol += np.prod(chi - clo)
        assert np.isclose(vol, np.prod(phi - plo))                                   # the 8 children tile the parent
        assert np.array_equal(sh[3 + 8 * k: 3 + 8 * k + 8], np.repeat(sc.sh[p:p + 1], 8, axis=0))
    # child raws = the parent's trilinear field (fp64 formula) at the child corners
    r = sc.raw[split].astype(np.float64)
    ch = child_raws(sc.raw[split])
    def tri(rr, x, y, z):
        w = [(1 - x) * (1 - y) * (1 - z), x * (1 - y) * (1 - z), (1 - x) * y * (1 - z), x * y * (1 - z),
             (1 - x) * (1 - y) * z, x * (1 - y) * z, (1 - x) * y * z, x * y * z]
        return sum(wi * rr[:, i] for i, wi in enumerate(w))
    for o in range(8):
        for c in range(8):
            x, y, zc = ((o & 1) + (c & 1)) / 2, (((o >> 1) & 1) + ((c >> 1) & 1)) / 2, ((o >> 2) + (c >> 2)) / 2
            assert np.allclose(ch[:, o, c], tri(r, x, y, zc), rtol=1e-6, atol=1e-6)
    # splitting a child again still samples the ORIGINAL field (trilinear restricted to a sub-cube is trilinear)
    gg = child_raws(ch[:, 5, :])                                  # child (1,0,1), then its children
    assert np.allclose(gg[:, 2, 7], tri(r, (1 + 0.5) / 2, (0 + 1) / 2, (1 + 0.5) / 2), rtol=1e-5, atol=1e-6)


# ---------------------------------------------------------------------------------------------
# NEXT-3: gradients through the depth and transmittance heads (R7: D = sum w_k t_mid,k, T_K = prod exp(-tau_k))
# ---------------------------------------------------------------------------------------------
def test_head_gradients_match_finite_differences(orc):
    """L = sum(G * image) + sum(GD * depth) + sum(GT * T_final): central differences in fp64 on an 8-voxel scene."""
    sc = tiny_scene(23, n=8, sh_degree=1)
    cam = look_at_camera((2.1, 0.7, 1.3), (0.05, -0.1, 0.0), 11, 9)
    G = random_image_grad(cam, 23)
    rng = np.random.default_rng(5)
    GD = rng.normal(0, 1.0, size=(cam.H, cam.W))
    GT = rng.normal(0, 1.0, size=(cam.H, cam.W))
    raw0, sh0 = sc.raw.astype(np.float64), sc.sh.astype(np.float64)
    g_raw, g_sh = orc.backward(sc, cam, 3, G, G_depth=GD, G_T=GT)
    g_raw_c, g_sh_c = orc.backward(sc, cam, 3, G)
    g_raw_d, g_sh_d = orc.backward(sc, cam, 3, np.zeros_like(G), G_depth=GD)
    g_raw_t, g_sh_t = orc.backward(sc, cam, 3, np.zeros_like(G), G_T=GT)
    np.testing.assert_allclose(g_raw, g_raw_c + g_raw_d + g_raw_t, rtol=1e-12, atol=1e-14)     # linear in the three heads
    assert np.abs(g_sh_d).max() == 0.0 and np.abs(g_sh_t).max() == 0.0                        # colour does not reach D or T

    def L(raw):
        r = orc.render(sc, cam, 3, raw=raw, sh=sh0)
        return float((r["image"] * G).sum() + (r["depth"] * GD).sum() + (r["T_final"] * GT).sum())

    h = 1e-6
    scale = np.abs(g_raw).max()
    for idx in [tuple(rng.integers(0, s) for s in raw0.shape) for _ in range(40)]:
        rp, rm = raw0.copy(), raw0.copy()
        rp[idx] += h
        rm[idx] -= h
        fd = (L(rp) - L(rm)) / (2 * h)
        assert abs(fd - g_raw[idx]) < 2e-7 * scale + 1e-9, (idx, fd, g_raw[idx])
    assert np.abs(g_raw_d).max() > 1e-3 and np.abs(g_raw_t).max() > 1e-3
    # closed form for the transmittance head: dT_K/dtau_k = -T_K, so one constant-density voxel on an axis ray gives
    # dL/draw_c = -GT T_K tau W_c summed over samples; with all 8 corners equal the 8 gradients sum to -GT T_K tau
    one = tiny_scene(3, n=1, sh_degree=0)
    one = replace(one, raw=np.full((1, 8), -0.3, dtype=np.float32))
    r1 = orc.render(one, cam, 3)
    gt1 = np.ones((cam.H, cam.W))
    gr, _ = orc.backward(one, cam, 3, np.zeros((cam.H, cam.W, 3)), G_T=gt1)
    tau = -np.log(np.maximum(r1["T_final"], 1e-300))
    assert np.isclose(gr.sum(), -(r1["T_final"] * tau).sum(), rtol=1e-10)


# ---------------------------------------------------------------------------------------------
# NEXT-4 (part): Adam update, pins of oracle/adam.py
# ---------------------------------------------------------------------------------------------
def test_adam_first_step_and_fp64_rederivation():
    from oracle.adam import adam_step
    rng = np.random.default_rng(8)
    th = rng.normal(0, 1, 4000).astype(np.float32)
    g = rng.normal(0, 1e-3, 4000).astype(np.float32)
    g[:5] = 0.0
    lr, b1, b2, eps = 1e-2, 0.9, 0.999, 1e-15
    t1, m1, v1 = adam_step(th, g, np.zeros_like(th), np.zeros_like(th), lr, b1, b2, eps, 1)
    # step 1: m/c1 = g, v/c2 = g^2 => every parameter moves by lr sign(g) (textbook property of the bias correction)
    np.testing.assert_allclose(th - t1, lr * np.sign(g), rtol=0, atol=2.5e-7)      # |theta| ~ 1: half an ulp of theta
    assert np.all(t1[:5] == th[:5])
    # ten steps against the same recurrences in fp64
    T, M, V = th.astype(np.float64), np.zeros(4000), np.zeros(4000)
    tt, mm, vv = th, np.zeros_like(th), np.zeros_like(th)
    for t in range(1, 11):
        gt = (g * np.float32(1 + 0.1 * t)).astype(np.float32)
        tt, mm, vv = adam_step(tt, gt, mm, vv, lr, b1, b2, 1e-8, t)
        # the float32-rounded coefficients (1 - b2 = 0.001 carries a 5e-5 relative rounding in float32), fp64 arithmetic
        B1, B2 = float(np.float32(b1)), float(np.float32(b2))
        M = B1 * M + float(np.float32(1) - np.float32(b1)) * gt
        V = B2 * V + float(np.float32(1) - np.float32(b2)) * gt.astype(np.float64) ** 2
        T = T - lr * (M / (1 - b1 ** t)) / (np.sqrt(V / (1 - b2 ** t)) + 1e-8)
    np.testing.assert_allclose(tt, T, rtol=1e-5, atol=1e-6)
    np.testing.assert_allclose(mm, M, rtol=1e-5, atol=1e-12)
    np.testing.assert_allclose(vv, V, rtol=1e-5, atol=1e-15)


# ---------------------------------------------------------------------------------------------
# L_SSIM (eq. 17; R14: Wang et al. 2004, 11-tap Gaussian window, sigma 1.5)
# ---------------------------------------------------------------------------------------------
def test_ssim_window_identity_constants_symmetry():
    from oracle import ssim
    g = ssim.gaussian_window()
    assert abs(g.sum() - 1.0) < 1e-15 and np.array_equal(g, g[::-1])
    # by hand: sum_k exp(-k^2 / 4.5), k = -5..5, = 1 + 2 (0.800737 + 0.411112 + 0.135335 + 0.028566 + 0.003866) = 3.759232
    assert abs(g[5] - 1.0 / 3.759232) < 2e-6 and abs(g[0] - 0.003866 / 3.759232) < 2e-6
    rng = np.random.default_rng(3)
    H, W = 23, 31
    a = rng.uniform(0, 1, size=(H, W, 3))
    b = np.clip(a + rng.normal(0, 0.1, size=a.shape), 0, 1)
    # identical images: SSIM = 1 everywhere (borders included), L = 0, and L is at its minimum there: zero gradient
    L, grad = ssim.ssim_loss_and_grad(a, a)
    assert abs(L) < 1e-14 and np.abs(grad).max() < 1e-15
    # two constant images, window inside the image: all (co)variances vanish and SSIM = (2ab + C1) / (a^2 + b^2 + C1)
    ca, cb = 0.3, 0.7
    S, _ = ssim.ssim_map(np.full((H, W, 1), ca), np.full((H, W, 1), cb))
    want = (2 * ca * cb + 0.01 ** 2) / (ca * ca + cb * cb + 0.01 ** 2)
    np.testing.assert_allclose(S[5:H - 5, 5:W - 5, 0], want, rtol=1e-12)
    assert abs(S[0, 0, 0] - want) > 1e-3                 # zero padding: the border windows see the padding
    # symmetric in its arguments, bounded by 1, and each channel is on its own
    Sab, _ = ssim.ssim_map(a, b)
    Sba, _ = ssim.ssim_map(b, a)
    np.testing.assert_allclose(Sab, Sba, rtol=1e-12, atol=1e-15)
    assert Sab.max() <= 1.0 + 1e-12 and Sab.mean() < 0.99
    S0, _ = ssim.ssim_map(a[:, :, :1], b[:, :, :1])
    np.testing.assert_allclose(S0[:, :, 0], Sab[:, :, 0], rtol=1e-13)


def test_ssim_moments_brute_force_and_gradient_fd():
    from oracle import ssim
    rng = np.random.default_rng(4)
    H, W = 17, 19
    R = rng.uniform(0, 1, size=(H, W, 3))
    I = np.clip(R + rng.normal(0, 0.15, size=R.shape), 0, 1)
    # the index at a few pixels from explicit weighted sums over the 11 x 11 neighbourhood (zero outside the image)
    g = ssim.gaussian_window()
    S, _ = ssim.ssim_map(R, I)
    for (y, x, ch) in [(0, 0, 0), (8, 9, 1), (16, 18, 2), (3, 17, 0)]:
        m1 = m2 = e11 = e22 = e12 = 0.0
        for dy in range(-5, 6):
            for dx in range(-5, 6):
                yy, xx = y + dy, x + dx
                if 0 <= yy < H and 0 <= xx < W:
                    wgt = g[dy + 5] * g[dx + 5]
                    r, t = R[yy, xx, ch], I[yy, xx, ch]
                    m1 += wgt * r; m2 += wgt * t; e11 += wgt * r * r; e22 += wgt * t * t; e12 += wgt * r * t
        want = ((2 * m1 * m2 + 1e-4) * (2 * (e12 - m1 * m2) + 9e-4)) / ((m1 * m1 + m2 * m2 + 1e-4) * ((e11 - m1 * m1) + (e22 - m2 * m2) + 9e-4))
        assert abs(S[y, x, ch] - want) < 1e-13
    # analytic gradient against central differences of the loss
    _, grad = ssim.ssim_loss_and_grad(R, I)
    h = 1e-6
    for (y, x, ch) in [(0, 0, 0), (8, 9, 1), (16, 18, 2), (5, 1, 1), (12, 12, 0)]:
        Rp, Rm = R.copy(), R.copy()
        Rp[y, x, ch] += h
        Rm[y, x, ch] -= h
        fd = (ssim.ssim_loss_and_grad(Rp, I)[0] - ssim.ssim_loss_and_grad(Rm, I)[0]) / (2 * h)
        assert abs(fd - grad[y, x, ch]) <= 1e-6 * max(abs(fd), 1e-4), (y, x, ch, fd, grad[y, x, ch])


# ---------------------------------------------------------------------------------------------
# L_tv (eq. 17; R15: L1 total variation over the 12 edges of every cell)
# ---------------------------------------------------------------------------------------------
def test_tv_constant_linear_scaling_fd():
    from oracle import tv
    assert len(tv.EDGES) == 12 and all(bin(a ^ b).count("1") == 1 and a < b for a, b in tv.EDGES) and len(set(tv.EDGES)) == 12
    L, g = tv.tv_loss_and_grad(np.full((5, 8), 0.7))
    assert L == 0.0 and not g.any()
    # corners of the unit cell sampled from alpha x + beta y + gamma z + d: four edges per axis, each |coefficient| long
    al, be, ga = 0.3, -1.1, 0.45
    corners = np.array([[al * (c & 1) + be * ((c >> 1) & 1) + ga * (c >> 2) + 2.0 for c in range(8)]])
    L, g = tv.tv_loss_and_grad(np.repeat(corners, 3, axis=0))
    assert abs(L - (abs(al) + abs(be) + abs(ga)) / 3.0) < 1e-15
    np.testing.assert_allclose(g.sum(axis=1), 0.0, atol=1e-16)           # a constant offset does not change the loss
    rng = np.random.default_rng(8)
    raw = rng.normal(0, 1, size=(7, 8))
    L0, g0 = tv.tv_loss_and_grad(raw)
    assert abs(tv.tv_loss_and_grad(-2.5 * raw + 4.0)[0] - 2.5 * L0) < 1e-14
    # brute force over all corner pairs at Hamming distance 1
    want = sum(abs(raw[v, a] - raw[v, b]) for v in range(7) for a in range(8) for b in range(a + 1, 8) if bin(a ^ b).count("1") == 1)
    assert abs(L0 - want / (12 * 7)) < 1e-15
    h = 1e-7
    for (v, c) in [(0, 0), (3, 5), (6, 7), (2, 2)]:
        rp, rm = raw.copy(), raw.copy()
        rp[v, c] += h
        rm[v, c] -= h
        fd = (tv.tv_loss_and_grad(rp)[0] - tv.tv_loss_and_grad(rm)[0]) / (2 * h)
        assert abs(fd - g0[v, c]) < 1e-8
