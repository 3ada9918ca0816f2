"""TEST INFRASTRUCTURE - ctypes access to oracle/svr_oracle.cpp (argument marshalling only).

`build()` compiles the C++ oracle with g++ (-O2 -fopenmp -ffp-contract=off: part B relies on
individually rounded binary32 operations). Scene parameters are promoted fp32 -> fp64 exactly before
the call unless the caller passes float64 arrays (finite-difference pins perturb in fp64).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "svr_oracle.cpp")
_SO = os.path.join(_HERE, "libsvr_oracle.so")
_lib = None


class _Scene(C.Structure):
    _fields_ = [("n", C.c_int64), ("sh_degree", C.c_int32), ("max_level", C.c_int32),
                ("root_lo", C.c_double * 3), ("root_edge", C.c_double),
                ("ijkl", C.c_void_p), ("raw", C.c_void_p), ("sh", C.c_void_p)]


class _Camera(C.Structure):
    _fields_ = [("W", C.c_int32), ("H", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("R", C.c_float * 9), ("t", C.c_float * 3),
                ("z_near", C.c_float), ("bg", C.c_float * 3)]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               _SRC, "-o", _SO]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_ray_dump.restype = C.c_int64
        _lib.orc_bin_rects.restype = C.c_int64
        _lib.orc_pixel_octant.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _ptr(a):
    return C.c_void_p(a.ctypes.data) if a is not None else C.c_void_p(0)


class _Marshalled:
    """Keeps the numpy buffers alive next to the C structs that point into them."""

    def __init__(self, scene, cam, raw=None, sh=None):
        self.ijkl = np.ascontiguousarray(scene.ijkl, dtype=np.uint16)
        self.raw = np.ascontiguousarray(scene.raw if raw is None else raw, dtype=np.float64)
        self.sh = np.ascontiguousarray(scene.sh if sh is None else sh, dtype=np.float64)
        s = _Scene()
        s.n, s.sh_degree, s.max_level = scene.n, scene.sh_degree, scene.max_level
        s.root_lo = (C.c_double * 3)(*[float(x) for x in scene.root_lo])
        s.root_edge = float(scene.root_edge)
        s.ijkl, s.raw, s.sh = self.ijkl.ctypes.data, self.raw.ctypes.data, self.sh.ctypes.data
        self.s = s
        c = _Camera()
        c.W, c.H = cam.W, cam.H
        c.fx, c.fy, c.cx, c.cy = cam.fx, cam.fy, cam.cx, cam.cy
        c.R = (C.c_float * 9)(*[float(x) for x in np.asarray(cam.R, dtype=np.float32).reshape(-1)])
        c.t = (C.c_float * 3)(*[float(x) for x in np.asarray(cam.t, dtype=np.float32)])
        c.z_near = cam.z_near
        c.bg = (C.c_float * 3)(*[float(x) for x in np.asarray(cam.bg, dtype=np.float32)])
        self.c = c


def sh_basis(degree: int, dirs: np.ndarray) -> np.ndarray:
    dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 3)
    out = np.zeros((dirs.shape[0], (degree + 1) ** 2))
    L = lib()
    for i in range(dirs.shape[0]):
        L.orc_sh_basis(C.c_int(degree), _ptr(dirs[i]), _ptr(out[i]))
    return out


def voxel_rgb(scene, cam, raw=None, sh=None):
    m = _Marshalled(scene, cam, raw, sh)
    rgb = np.zeros((scene.n, 3))
    pre = np.zeros((scene.n, 3))
    lib().orc_voxel_rgb(C.byref(m.s), C.byref(m.c), _ptr(rgb), _ptr(pre))
    return rgb, pre


def ray(cam, x: int, y: int):
    m = _Marshalled(_EmptyScene(), cam)
    o, d = np.zeros(3), np.zeros(3)
    lib().orc_ray(C.byref(m.c), C.c_int(x), C.c_int(y), _ptr(o), _ptr(d))
    return o, d


class _EmptyScene:
    n, sh_degree, max_level = 0, 0, 1
    root_lo, root_edge = np.zeros(3), 1.0
    ijkl = np.zeros((0, 4), dtype=np.uint16)
    raw = np.zeros((0, 8))
    sh = np.zeros((0, 1, 3))


def ray_dump(scene, cam, K: int, x: int, y: int, act_mode: int = 0, raw=None, sh=None):
    """Sorted hit list of one ray: dict(vox, t_in, t_out, tau, w, T_final)."""
    m = _Marshalled(scene, cam, raw, sh)
    cap = max(1, scene.n)
    vox = np.zeros(cap, dtype=np.int64)
    tin, tout, tau, w = (np.zeros(cap) for _ in range(4))
    Tf = np.zeros(1)
    k = lib().orc_ray_dump(C.byref(m.s), C.byref(m.c), C.c_int(K), C.c_int(act_mode), C.c_int(x), C.c_int(y),
                           C.c_int64(cap), _ptr(vox), _ptr(tin), _ptr(tout), _ptr(tau), _ptr(w), _ptr(Tf))
    k = int(k)
    return dict(vox=vox[:k], t_in=tin[:k], t_out=tout[:k], tau=tau[:k], w=w[:k], T_final=float(Tf[0]))


def _rays(cam, xy):
    if xy is None:
        return cam.W * cam.H, None
    xy = np.ascontiguousarray(xy, dtype=np.int32).reshape(-1, 2)
    return xy.shape[0], xy


def render(scene, cam, K: int, mode: str = "pure", xy: Optional[np.ndarray] = None, act_mode: int = 0,
           w_max: Optional[np.ndarray] = None, raw=None, sh=None):
    """Forward. Returns dict(image [H,W,3] or [n,3], depth, T_final, w_max [n], n_hits)."""
    m = _Marshalled(scene, cam, raw, sh)
    n_rays, xy_a = _rays(cam, xy)
    image = np.zeros((n_rays, 3))
    depth, Tf = np.zeros(n_rays), np.zeros(n_rays)
    nh = np.zeros(n_rays, dtype=np.int32)
    if w_max is None:
        w_max = np.zeros(scene.n)
    assert w_max.dtype == np.float64 and w_max.flags.c_contiguous
    lib().orc_render(C.byref(m.s), C.byref(m.c), C.c_int(K), C.c_int(act_mode), C.c_int(1 if mode == "bucketed" else 0),
                     C.c_int64(n_rays), _ptr(xy_a), _ptr(image), _ptr(depth), _ptr(Tf), _ptr(w_max), _ptr(nh))
    if xy is None:
        image, depth, Tf, nh = (image.reshape(cam.H, cam.W, 3), depth.reshape(cam.H, cam.W),
                                Tf.reshape(cam.H, cam.W), nh.reshape(cam.H, cam.W))
    return dict(image=image, depth=depth, T_final=Tf, w_max=w_max, n_hits=nh)


def backward(scene, cam, K: int, G: np.ndarray, mode: str = "pure", xy: Optional[np.ndarray] = None,
             act_mode: int = 0, grad_raw=None, grad_sh=None, raw=None, sh=None, G_depth=None, G_T=None):
    """Gradient of sum(G * image) [+ sum(G_depth * depth) + sum(G_T * T_final)]. Accumulates into (and returns)
    grad_raw [n,8], grad_sh [n,B,3]."""
    m = _Marshalled(scene, cam, raw, sh)
    n_rays, xy_a = _rays(cam, xy)
    G = np.ascontiguousarray(G, dtype=np.float64).reshape(n_rays, 3)
    if grad_raw is None:
        grad_raw = np.zeros((scene.n, 8))
    if grad_sh is None:
        grad_sh = np.zeros((scene.n, scene.n_basis, 3))
    if G_depth is None and G_T is None:
        lib().orc_backward(C.byref(m.s), C.byref(m.c), C.c_int(K), C.c_int(act_mode), C.c_int(1 if mode == "bucketed" else 0),
                           C.c_int64(n_rays), _ptr(xy_a), _ptr(G), _ptr(grad_raw), _ptr(grad_sh))
    else:
        gd = None if G_depth is None else np.ascontiguousarray(G_depth, dtype=np.float64).reshape(n_rays)
        gt = None if G_T is None else np.ascontiguousarray(G_T, dtype=np.float64).reshape(n_rays)
        lib().orc_backward_heads(C.byref(m.s), C.byref(m.c), C.c_int(K), C.c_int(act_mode), C.c_int(1 if mode == "bucketed" else 0),
                                 C.c_int64(n_rays), _ptr(xy_a), _ptr(G), _ptr(gd), _ptr(gt), _ptr(grad_raw), _ptr(grad_sh))
    return grad_raw, grad_sh


def bin_rects(scene, cam):
    """Part B: (rects [n,4] u16, tile_masks [n_tiles] u8, E)."""
    m = _Marshalled(scene, cam)
    tx, ty = (cam.W + 15) // 16, (cam.H + 15) // 16
    rects = np.zeros((scene.n, 4), dtype=np.uint16)
    masks = np.zeros(tx * ty, dtype=np.uint8)
    E = lib().orc_bin_rects(C.byref(m.s), C.byref(m.c), _ptr(rects), _ptr(masks))
    return rects, masks, int(E)


def bin_lists(scene, cam):
    """Part B: dict(rects, tile_masks, keys [E] u64, vals [E] u32, ranges [n_tiles,8,2] u32)."""
    m = _Marshalled(scene, cam)
    rects, masks, E = bin_rects(scene, cam)
    tx, ty = (cam.W + 15) // 16, (cam.H + 15) // 16
    keys = np.zeros(E, dtype=np.uint64)
    vals = np.zeros(E, dtype=np.uint32)
    ranges = np.zeros((tx * ty, 8, 2), dtype=np.uint32)
    lib().orc_bin_lists(C.byref(m.s), C.byref(m.c), _ptr(rects), _ptr(masks), _ptr(keys), _ptr(vals), _ptr(ranges))
    return dict(rects=rects, tile_masks=masks, keys=keys, vals=vals, ranges=ranges)


def pixel_octant(cam, x: int, y: int) -> int:
    m = _Marshalled(_EmptyScene(), cam)
    return int(lib().orc_pixel_octant(C.byref(m.c), C.c_int(x), C.c_int(y)))
