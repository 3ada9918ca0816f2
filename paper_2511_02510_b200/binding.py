"""ctypes binding of libsvr.so - argument marshalling only (include/svr.h is the contract).

PyTorch is used for device memory and streams; every step of the path runs in the library's kernels.
There is no fallback: if libsvr.so is missing or cannot be loaded, importing this module raises.
Function names mirror the C ABI (svr_create, svr_preprocess, svr_forward, svr_loss_grad, svr_backward, ...).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsvr.so")

SVR_OK, SVR_ERR_INVALID_ARG, SVR_ERR_CUDA, SVR_ERR_WORKSPACE, SVR_ERR_UNSUPPORTED = range(5)
_STATUS = {0: "SVR_OK", 1: "SVR_ERR_INVALID_ARG", 2: "SVR_ERR_CUDA", 3: "SVR_ERR_WORKSPACE", 4: "SVR_ERR_UNSUPPORTED"}

EXPORTS = ["svr_create", "svr_create_with_allocator", "svr_destroy", "svr_last_error", "svr_workspace_peak_bytes", "svr_kernel_launches",
           "svr_preprocess", "svr_frame_refresh_colors", "svr_frame_release", "svr_forward", "svr_loss_grad", "svr_loss_prepare", "svr_ssim_loss_grad", "svr_tv_loss_grad",
           "svr_ssim_loss_grad_static", "svr_ssim_static_max_pixels", "svr_static_last_error",
           "svr_backward", "svr_backward_heads", "svr_render_normals", "svr_backward_normals", "svr_train_view_host", "svr_frame_lists", "svr_frame_colors", "svr_copy_to_host", "svr_gamma_schedule",
           "svr_forward_stats", "svr_measure_peaks", "svr_set_stage_timing", "svr_num_stages", "svr_stage_name", "svr_get_stage_times", "svr_set_debug_flags",
           "svr_prune_step", "svr_compact_rows", "svr_subdivide_select", "svr_subdivide_apply", "svr_subdivide_rows", "svr_adam_step",
           "svr_gather_corners", "svr_scatter_add_corners"]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)     # SvrAllocFn
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)            # SvrFreeFn


class SvrError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class SvrVoxels(C.Structure):
    _fields_ = [("n", C.c_int64), ("sh_degree", C.c_int32), ("max_level", C.c_int32), ("root_lo", C.c_float * 3),
                ("root_edge", C.c_float), ("ijkl", C.c_void_p), ("raw_density", C.c_void_p), ("sh", C.c_void_p)]


class SvrCamera(C.Structure):
    _fields_ = [("W", C.c_int32), ("H", C.c_int32), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float),
                ("cy", C.c_float), ("R", C.c_float * 9), ("t", C.c_float * 3), ("z_near", C.c_float), ("bg", C.c_float * 3)]


class SvrRenderOpts(C.Structure):
    _fields_ = [("K", C.c_int32), ("T_min", C.c_float), ("record", C.c_int32), ("grad_overwrite", C.c_int32)]


class SvrPruneOpts(C.Structure):
    _fields_ = [("n_bins", C.c_int32), ("q_near", C.c_float), ("q_far", C.c_float), ("ema_alpha", C.c_float), ("m_low", C.c_float),
                ("m_high", C.c_float), ("kappa", C.c_float), ("w_keep", C.c_float), ("cap_fraction", C.c_float), ("halo", C.c_int32)]


class SvrSubdivOpts(C.Structure):
    _fields_ = [("kappa", C.c_float), ("beta", C.c_float), ("max_level", C.c_int32), ("max_splits", C.c_int64),
                ("use_current_percentiles", C.c_int32), ("z_p5", C.c_float), ("z_p95", C.c_float)]


class SvrLossOpts(C.Structure):
    _fields_ = [("eps", C.c_float), ("percentile", C.c_float), ("sobel_source", C.c_int32)]


def _load():
    if not os.path.exists(_SO):
        raise ImportError(f"{_SO} is missing: build it with `python -m paper_2511_02510_b200._build` "
                          "(nvcc, sm_100a). There is no CPU or PyTorch fallback.")
    lib = C.CDLL(_SO)
    lib.svr_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p, C.c_size_t]
    lib.svr_create_with_allocator.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p, ALLOC_FN, FREE_FN, C.c_void_p, C.c_size_t]
    lib.svr_destroy.argtypes = [C.c_void_p]
    lib.svr_destroy.restype = None
    lib.svr_last_error.argtypes = [C.c_void_p]
    lib.svr_last_error.restype = C.c_char_p
    lib.svr_workspace_peak_bytes.argtypes = [C.c_void_p]
    lib.svr_workspace_peak_bytes.restype = C.c_size_t
    lib.svr_kernel_launches.argtypes = [C.c_void_p]
    lib.svr_kernel_launches.restype = C.c_int64
    lib.svr_preprocess.argtypes = [C.c_void_p, C.POINTER(SvrVoxels), C.POINTER(SvrCamera), C.POINTER(C.c_void_p)]
    lib.svr_frame_refresh_colors.argtypes = [C.c_void_p, C.c_void_p]
    lib.svr_measure_peaks.argtypes = [C.c_void_p, C.c_void_p]
    lib.svr_frame_release.argtypes = [C.c_void_p, C.c_void_p]
    lib.svr_frame_release.restype = None
    lib.svr_forward.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(SvrRenderOpts)] + [C.c_void_p] * 4
    lib.svr_loss_grad.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_float,
                                  C.POINTER(SvrLossOpts), C.c_void_p, C.c_void_p]
    lib.svr_ssim_loss_grad.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_float, C.c_int32,
                                       C.c_void_p, C.c_void_p]
    lib.svr_ssim_loss_grad_static.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_float, C.c_int32,
                                              C.c_void_p, C.c_void_p]
    lib.svr_ssim_static_max_pixels.restype = C.c_int64
    lib.svr_static_last_error.restype = C.c_char_p
    lib.svr_tv_loss_grad.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_void_p, C.c_void_p]
    lib.svr_loss_prepare.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.POINTER(SvrLossOpts)]
    lib.svr_backward.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(SvrRenderOpts)] + [C.c_void_p] * 5
    lib.svr_backward_heads.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(SvrRenderOpts)] + [C.c_void_p] * 9
    lib.svr_train_view_host.argtypes = [C.c_void_p, C.POINTER(SvrVoxels), C.POINTER(SvrCamera), C.POINTER(SvrRenderOpts),
                                        C.POINTER(SvrLossOpts), C.c_float] + [C.c_void_p] * 6
    lib.svr_render_normals.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(SvrRenderOpts), C.c_void_p, C.c_void_p]
    lib.svr_backward_normals.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(SvrRenderOpts)] + [C.c_void_p] * 3
    lib.svr_frame_lists.argtypes = [C.c_void_p] + [C.POINTER(C.c_void_p)] * 2 + [C.POINTER(C.c_int64)] + [C.POINTER(C.c_void_p)] * 3
    lib.svr_frame_colors.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
    lib.svr_copy_to_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t]
    lib.svr_forward_stats.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(SvrRenderOpts), C.c_void_p, C.c_void_p]
    lib.svr_prune_step.argtypes = [C.c_void_p, C.POINTER(SvrVoxels), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                   C.POINTER(SvrPruneOpts), C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
    lib.svr_compact_rows.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_int64, C.POINTER(C.c_int64)]
    lib.svr_subdivide_select.argtypes = [C.c_void_p, C.POINTER(SvrVoxels), C.c_void_p, C.c_int32, C.c_void_p, C.POINTER(SvrSubdivOpts),
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
    lib.svr_subdivide_apply.argtypes = [C.c_void_p, C.POINTER(SvrVoxels), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]
    lib.svr_subdivide_rows.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_int64)]
    lib.svr_adam_step.argtypes = [C.c_void_p] * 5 + [C.c_int64, C.c_float, C.c_float, C.c_float, C.c_float, C.c_int32, C.c_int32]
    lib.svr_gather_corners.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
    lib.svr_scatter_add_corners.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
    lib.svr_set_stage_timing.argtypes = [C.c_void_p, C.c_int]
    lib.svr_set_stage_timing.restype = None
    lib.svr_num_stages.restype = C.c_int
    lib.svr_set_debug_flags.argtypes = [C.c_void_p, C.c_int]
    lib.svr_set_debug_flags.restype = None
    lib.svr_stage_name.argtypes = [C.c_int]
    lib.svr_stage_name.restype = C.c_char_p
    lib.svr_get_stage_times.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
    lib.svr_gamma_schedule.argtypes = [C.c_float] * 5
    lib.svr_gamma_schedule.restype = C.c_float
    return lib


_lib = _load()


def lib():
    return _lib


def _p(t: Optional[torch.Tensor]):
    return C.c_void_p(0) if t is None else C.c_void_p(t.data_ptr())


def _dev(t: torch.Tensor, dtype, name: str):
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise ValueError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")
    return t


def make_camera(cam) -> SvrCamera:
    """From any object with W,H,fx,fy,cx,cy,R,t,z_near,bg attributes (e.g. svr_inputs.Camera)."""
    c = SvrCamera()
    c.W, c.H = int(cam.W), int(cam.H)
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    c.R = (C.c_float * 9)(*[float(x) for x in np.asarray(cam.R, dtype=np.float32).reshape(-1)])
    c.t = (C.c_float * 3)(*[float(x) for x in np.asarray(cam.t, dtype=np.float32)])
    c.z_near = float(cam.z_near)
    c.bg = (C.c_float * 3)(*[float(x) for x in np.asarray(cam.bg, dtype=np.float32)])
    return c


class Voxels:
    """Device-resident voxel arrays + the C struct pointing at them."""

    def __init__(self, ijkl: torch.Tensor, raw: torch.Tensor, sh: torch.Tensor, sh_degree: int, max_level: int,
                 root_lo, root_edge: float):
        self.ijkl = _dev(ijkl, torch.int16, "ijkl")          # uint16 bit patterns
        self.raw = _dev(raw, torch.float32, "raw")
        self.sh = _dev(sh, torch.float32, "sh")
        self.n = int(ijkl.shape[0])
        self.sh_degree, self.max_level = int(sh_degree), int(max_level)
        assert raw.shape == (self.n, 8) and sh.shape == (self.n, (sh_degree + 1) ** 2, 3) and ijkl.shape == (self.n, 4)
        s = SvrVoxels()
        s.n, s.sh_degree, s.max_level = self.n, self.sh_degree, self.max_level
        s.root_lo = (C.c_float * 3)(*[float(x) for x in root_lo])
        s.root_edge = float(root_edge)
        s.ijkl, s.raw_density, s.sh = self.ijkl.data_ptr(), self.raw.data_ptr(), self.sh.data_ptr()
        self.c = s

    @staticmethod
    def from_scene(scene, device="cuda:0") -> "Voxels":
        ijkl = torch.from_numpy(np.ascontiguousarray(scene.ijkl).view(np.int16)).to(device)
        raw = torch.from_numpy(np.ascontiguousarray(scene.raw, dtype=np.float32)).to(device)
        sh = torch.from_numpy(np.ascontiguousarray(scene.sh, dtype=np.float32)).to(device)
        return Voxels(ijkl, raw, sh, scene.sh_degree, scene.max_level, scene.root_lo, scene.root_edge)


class Frame:
    def __init__(self, ctx: "Context", handle: int, vox: Voxels, cam: SvrCamera):
        self.ctx, self.handle, self.vox, self.cam = ctx, handle, vox, cam
        self.W, self.H = cam.W, cam.H

    def release(self):
        if self.handle:
            _lib.svr_frame_release(self.ctx.handle, C.c_void_p(self.handle))
            self.handle = 0

    def __del__(self):
        try:
            self.release()
        except Exception:
            pass

    def refresh_colors(self):
        """svr_frame_refresh_colors: re-capture raw_density / sh values (colours + per-voxel view records); the lists stay."""
        self.ctx._check(_lib.svr_frame_refresh_colors(self.ctx.handle, C.c_void_p(self.handle)))

    @property
    def n_entries(self) -> int:
        n = C.c_int64()
        self.ctx._check(_lib.svr_frame_lists(C.c_void_p(self.handle), None, None, C.byref(n), None, None, None))
        return int(n.value)

    def lists(self):
        """Copies of the inspection buffers as NumPy arrays (tests)."""
        keys, vals, ranges, rects, masks = (C.c_void_p() for _ in range(5))
        n = C.c_int64()
        self.ctx._check(_lib.svr_frame_lists(C.c_void_p(self.handle), C.byref(keys), C.byref(vals), C.byref(n),
                                             C.byref(ranges), C.byref(rects), C.byref(masks)))
        self.ctx.synchronize()
        E = int(n.value)
        n_tiles = ((self.W + 15) // 16) * ((self.H + 15) // 16)

        def grab(ptr, count, dtype):
            out = np.empty(count, dtype=dtype)
            if count:
                self.ctx._check(_lib.svr_copy_to_host(self.ctx.handle, out.ctypes.data, ptr, out.nbytes))
            return out
        return dict(keys=grab(keys, E, np.uint64), vals=grab(vals, E, np.uint32),
                    ranges=grab(ranges, n_tiles * 16, np.uint32).reshape(n_tiles, 8, 2),
                    rects=grab(rects, self.vox.n * 4, np.uint16).reshape(self.vox.n, 4),
                    tile_masks=grab(masks, n_tiles, np.uint8), n_entries=E)

    def colors(self) -> np.ndarray:
        p = C.c_void_p()
        self.ctx._check(_lib.svr_frame_colors(C.c_void_p(self.handle), C.byref(p)))
        self.ctx.synchronize()
        out = np.empty(self.vox.n * 4, dtype=np.float32)
        if self.vox.n:
            self.ctx._check(_lib.svr_copy_to_host(self.ctx.handle, out.ctypes.data, p, out.nbytes))
        return out.reshape(self.vox.n, 4)




class Context:
    """One library context bound to a device and a stream (default: torch's current stream)."""

    def __init__(self, device: int = 0, stream: Optional[torch.cuda.Stream] = None, workspace_budget_bytes: int = 0,
                 torch_allocator: bool = False):
        """torch_allocator: the library's workspace blocks come from PyTorch's caching allocator (svr_create_with_allocator)
        instead of the context's private CUDA memory pool."""
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2511_02510_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        torch.cuda.set_device(device)
        self.device = device
        self.stream = stream if stream is not None else torch.cuda.current_stream(device)
        h = C.c_void_p()
        if torch_allocator:
            cs = self.stream.cuda_stream
            self.alloc_calls = 0

            def _alloc(nbytes, _user):
                self.alloc_calls += 1
                try:
                    return torch.cuda.caching_allocator_alloc(int(nbytes), device, cs)
                except RuntimeError:
                    return None

            def _free(ptr, _user):
                torch.cuda.caching_allocator_delete(ptr)

            self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)       # keep the thunks alive with the context
            st = _lib.svr_create_with_allocator(C.byref(h), device, C.c_void_p(cs), self._alloc_cb, self._free_cb, None, workspace_budget_bytes)
        else:
            st = _lib.svr_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream), workspace_budget_bytes)
        if st != SVR_OK:
            raise SvrError(st, "svr_create failed")
        self.handle = h

    def close(self):
        if self.handle:
            _lib.svr_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != SVR_OK:
            raise SvrError(st, _lib.svr_last_error(self.handle).decode())

    def synchronize(self):
        self.stream.synchronize()

    @property
    def workspace_peak_bytes(self) -> int:
        return int(_lib.svr_workspace_peak_bytes(self.handle))

    @property
    def kernel_launches(self) -> int:
        return int(_lib.svr_kernel_launches(self.handle))

    # ---- measurement hooks -----------------------------------------------------------------------
    def svr_forward_stats(self, frame: "Frame", K: int, T_min: float = 1e-5) -> dict:
        image = torch.empty((frame.H, frame.W, 3), dtype=torch.float32, device=frame.vox.raw.device)
        out = (C.c_uint64 * 4)()
        o = SvrRenderOpts(K, T_min, 1)
        self._check(_lib.svr_forward_stats(self.handle, C.c_void_p(frame.handle), C.byref(o), _p(image), C.cast(out, C.c_void_p)))
        return dict(hits=int(out[0]), slab_tests=int(out[1]), warp_voxel_pairs=int(out[2]), entries_staged=int(out[3]))

    def svr_set_debug_flags(self, flags: int):
        """Measurement / test hook: bit 3 (8) selects the first list-build design (per-voxel scan + global radix sort)."""
        _lib.svr_set_debug_flags(self.handle, int(flags))

    def svr_set_stage_timing(self, enabled: bool):
        _lib.svr_set_stage_timing(self.handle, 1 if enabled else 0)

    def svr_measure_peaks(self) -> dict:
        out = (C.c_float * 4)()
        self._check(_lib.svr_measure_peaks(self.handle, C.cast(out, C.c_void_p)))
        return {"fp32_ffma_tflops": float(out[0]), "fp32_ffma2_tflops": float(out[1]), "l2_red_v4_gops": float(out[2]),
                "issue_gwarp_inst_per_s": float(out[3])}

    def svr_get_stage_times(self, reset: bool = True) -> dict:
        n = _lib.svr_num_stages()
        ms, calls = (C.c_double * n)(), (C.c_int64 * n)()
        self._check(_lib.svr_get_stage_times(self.handle, C.cast(ms, C.c_void_p), C.cast(calls, C.c_void_p), 1 if reset else 0))
        return {_lib.svr_stage_name(i).decode(): (float(ms[i]), int(calls[i])) for i in range(n)}

    # ---- the four calls of the path -------------------------------------------------------------
    def svr_preprocess(self, vox: Voxels, cam) -> Frame:
        c = cam if isinstance(cam, SvrCamera) else make_camera(cam)
        h = C.c_void_p()
        self._check(_lib.svr_preprocess(self.handle, C.byref(vox.c), C.byref(c), C.byref(h)))
        return Frame(self, h.value, vox, c)

    def svr_forward(self, frame: Frame, K: int, T_min: float = 1e-5, w_max: Optional[torch.Tensor] = None,
                    image=None, depth=None, T_final=None, want_aux: bool = True, record: bool = True):
        dev = frame.vox.raw.device
        if image is None:
            image = torch.empty((frame.H, frame.W, 3), dtype=torch.float32, device=dev)
        if want_aux:
            if depth is None:
                depth = torch.empty((frame.H, frame.W), dtype=torch.float32, device=dev)
            if T_final is None:
                T_final = torch.empty((frame.H, frame.W), dtype=torch.float32, device=dev)
        o = SvrRenderOpts(K, T_min, 1 if record else 0)
        self._check(_lib.svr_forward(self.handle, C.c_void_p(frame.handle), C.byref(o), _p(image), _p(depth), _p(T_final), _p(w_max)))
        return image, depth, T_final

    def svr_loss_prepare(self, target: torch.Tensor, eps: float = 1e-3, percentile: float = 0.99, sobel_source: int = 0):
        H, W = int(target.shape[0]), int(target.shape[1])
        _dev(target, torch.float32, "target")
        o = SvrLossOpts(eps, percentile, sobel_source)
        self._check(_lib.svr_loss_prepare(self.handle, _p(target), W, H, C.byref(o)))

    def svr_ssim_loss_grad(self, render: torch.Tensor, target: torch.Tensor, lam: float = 1.0, dL=None, loss=None,
                           accumulate: bool = False):
        """dL (+)= lam * dL_SSIM/d render; returns (dL, loss) with loss = L_SSIM on the device."""
        H, W = int(render.shape[0]), int(render.shape[1])
        _dev(render, torch.float32, "render")
        _dev(target, torch.float32, "target")
        if dL is None:
            dL = torch.zeros_like(render) if accumulate else torch.empty_like(render)
        if loss is None:
            loss = torch.empty(1, dtype=torch.float32, device=render.device)
        self._check(_lib.svr_ssim_loss_grad(self.handle, _p(render), _p(target), W, H, lam, 1 if accumulate else 0, _p(dL), _p(loss)))
        return dL, loss

    def svr_tv_loss_grad(self, raw: torch.Tensor, grad_raw: torch.Tensor, lam: float = 1.0, loss=None):
        """grad_raw += lam * dL_tv/draw; returns the device scalar L_tv."""
        _dev(raw, torch.float32, "raw")
        _dev(grad_raw, torch.float32, "grad_raw")
        if loss is None:
            loss = torch.empty(1, dtype=torch.float32, device=raw.device)
        self._check(_lib.svr_tv_loss_grad(self.handle, _p(raw), int(raw.shape[0]), lam, _p(grad_raw), _p(loss)))
        return loss

    def svr_loss_grad(self, render: torch.Tensor, target: torch.Tensor, gamma: float, eps: float = 1e-3,
                      percentile: float = 0.99, sobel_source: int = 0, dL=None, loss=None):
        H, W = int(render.shape[0]), int(render.shape[1])
        _dev(render, torch.float32, "render")
        _dev(target, torch.float32, "target")
        if dL is None:
            dL = torch.empty_like(render)
        if loss is None:
            loss = torch.empty(1, dtype=torch.float32, device=render.device)
        o = SvrLossOpts(eps, percentile, sobel_source)
        self._check(_lib.svr_loss_grad(self.handle, _p(render), _p(target), W, H, gamma, C.byref(o), _p(dL), _p(loss)))
        return dL, loss

    def svr_backward(self, frame: Frame, K: int, dL: torch.Tensor, image: torch.Tensor, grad_raw: torch.Tensor,
                     grad_sh: torch.Tensor, T_min: float = 1e-5, w_max: Optional[torch.Tensor] = None, overwrite: bool = False):
        """overwrite=False: gradients accumulate (+=); True: grad_raw / grad_sh are written for all voxels (SvrRenderOpts.grad_overwrite)."""
        _dev(dL, torch.float32, "dL")
        _dev(image, torch.float32, "image")
        _dev(grad_raw, torch.float32, "grad_raw")
        _dev(grad_sh, torch.float32, "grad_sh")
        o = SvrRenderOpts(K, T_min, 1, 1 if overwrite else 0)
        self._check(_lib.svr_backward(self.handle, C.c_void_p(frame.handle), C.byref(o), _p(dL), _p(image), _p(grad_raw),
                                      _p(grad_sh), _p(w_max)))

    def svr_backward_heads(self, frame: "Frame", K: int, dL, image, grad_raw, grad_sh, T_min: float = 1e-5, w_max=None,
                           dL_ddepth=None, dL_dT=None, depth=None, T_final=None, overwrite: bool = False):
        o = SvrRenderOpts(K, T_min, 1, 1 if overwrite else 0)
        self._check(_lib.svr_backward_heads(self.handle, C.c_void_p(frame.handle), C.byref(o), _p(dL), _p(dL_ddepth), _p(dL_dT), _p(image),
                                            _p(depth), _p(T_final), _p(grad_raw), _p(grad_sh), _p(w_max)))

    # ---- NEXT-3: rendered normals (R16) -------------------------------------------------
    def svr_render_normals(self, frame: "Frame", K: int, T_min: float = 1e-5):
        dev = frame.vox.raw.device
        normal = torch.empty((frame.H, frame.W, 3), dtype=torch.float32, device=dev)
        Tf = torch.empty((frame.H, frame.W), dtype=torch.float32, device=dev)
        o = SvrRenderOpts(K, T_min, 0)
        self._check(_lib.svr_render_normals(self.handle, C.c_void_p(frame.handle), C.byref(o), _p(normal), _p(Tf)))
        return normal, Tf

    def svr_backward_normals(self, frame: "Frame", K: int, dL_dnormal: torch.Tensor, normal: torch.Tensor, grad_raw: torch.Tensor,
                             T_min: float = 1e-5):
        o = SvrRenderOpts(K, T_min, 0)
        self._check(_lib.svr_backward_normals(self.handle, C.c_void_p(frame.handle), C.byref(o), _p(dL_dnormal), _p(normal), _p(grad_raw)))

    def svr_train_view_host(self, vox: Voxels, cam, K: int, gamma: float, target_host: torch.Tensor, grad_raw, grad_sh,
                            w_max=None, T_min: float = 1e-5, eps: float = 1e-3, percentile: float = 0.99,
                            sobel_source: int = 0, image_host: Optional[torch.Tensor] = None, overwrite: bool = False) -> float:
        c = cam if isinstance(cam, SvrCamera) else make_camera(cam)
        assert not target_host.is_cuda and target_host.dtype == torch.float32 and target_host.is_contiguous()
        ro, lo = SvrRenderOpts(K, T_min, 1, 1 if overwrite else 0), SvrLossOpts(eps, percentile, sobel_source)
        loss = C.c_float()
        self._check(_lib.svr_train_view_host(self.handle, C.byref(vox.c), C.byref(c), C.byref(ro), C.byref(lo), gamma,
                                             _p(target_host), _p(grad_raw), _p(grad_sh), _p(w_max),
                                             C.cast(C.byref(loss), C.c_void_p), _p(image_host)))
        return float(loss.value)


    # ---- NEXT-1: depth-aware quantile pruning -----------------------------------------
    def svr_prune_step(self, vox: Voxels, cams, w_max: torch.Tensor, ema: torch.Tensor, state: torch.Tensor, opts: SvrPruneOpts):
        """One adaptation step; ema / state are updated in place. Returns (keep uint8 [n], tau float32 [n_bins], n_removed)."""
        arr = (SvrCamera * len(cams))(*[c if isinstance(c, SvrCamera) else make_camera(c) for c in cams])
        keep = torch.empty(vox.n, dtype=torch.uint8, device=w_max.device)
        tau = (C.c_float * opts.n_bins)()
        n_removed = C.c_int64()
        self._check(_lib.svr_prune_step(self.handle, C.byref(vox.c), C.cast(arr, C.c_void_p), len(cams), _p(w_max), _p(ema), _p(state),
                                        C.byref(opts), _p(keep), C.cast(tau, C.c_void_p), C.byref(n_removed)))
        return keep, np.array(list(tau), dtype=np.float32), int(n_removed.value)

    def svr_compact_rows(self, keep: torch.Tensor, src: torch.Tensor) -> torch.Tensor:
        """Stable compaction of the rows of `src` (first dimension) whose keep flag is set."""
        assert src.is_contiguous() and keep.dtype == torch.uint8
        n = src.shape[0]
        row_bytes = src.element_size() * (src.numel() // max(n, 1)) if n else src.element_size()
        dst = torch.empty_like(src)
        n_out = C.c_int64()
        self._check(_lib.svr_compact_rows(self.handle, _p(keep), n, _p(src), _p(dst), row_bytes, C.byref(n_out)))
        return dst[: int(n_out.value)]


    # ---- NEXT-2: priority-driven subdivision -------------------------------------------
    def svr_subdivide_select(self, vox: Voxels, cams, usefulness: torch.Tensor, opts: SvrSubdivOpts):
        """Returns (split uint8 [n], priority float32 [n], (z_p5, z_p95) of this step, n_split)."""
        arr = (SvrCamera * len(cams))(*[c if isinstance(c, SvrCamera) else make_camera(c) for c in cams])
        split = torch.empty(vox.n, dtype=torch.uint8, device=usefulness.device)
        priority = torch.empty(vox.n, dtype=torch.float32, device=usefulness.device)
        zp = (C.c_float * 2)()
        n_split = C.c_int64()
        self._check(_lib.svr_subdivide_select(self.handle, C.byref(vox.c), C.cast(arr, C.c_void_p), len(cams), _p(usefulness), C.byref(opts),
                                              _p(split), _p(priority), C.cast(zp, C.c_void_p), C.byref(n_split)))
        return split, priority, (float(zp[0]), float(zp[1])), int(n_split.value)

    def svr_subdivide_apply(self, vox: Voxels, split: torch.Tensor, n_split: int):
        """Returns (ijkl int16 [n', 4], raw [n', 8], sh [n', B, 3]) with n' = n + 7 n_split."""
        n_new = vox.n + 7 * n_split
        ijkl = torch.empty((n_new, 4), dtype=torch.int16, device=vox.raw.device)
        raw = torch.empty((n_new, 8), dtype=torch.float32, device=vox.raw.device)
        sh = torch.empty((n_new,) + tuple(vox.sh.shape[1:]), dtype=torch.float32, device=vox.raw.device)
        n_out = C.c_int64()
        self._check(_lib.svr_subdivide_apply(self.handle, C.byref(vox.c), _p(split), _p(ijkl), _p(raw), _p(sh), C.byref(n_out)))
        assert int(n_out.value) == n_new, (int(n_out.value), n_new)
        return ijkl, raw, sh


    def svr_subdivide_rows(self, split: torch.Tensor, src: torch.Tensor, n_split: int, zero: bool = False) -> torch.Tensor:
        """A per-voxel array (first dimension = voxels) through the split `split`: unsplit rows, then 8 rows per split voxel,
        each the parent's row (zero=False) or zeros (zero=True). n_split = number of set entries of `split`."""
        _dev(split, torch.uint8, "split")
        if not (src.is_cuda and src.is_contiguous()):
            raise ValueError("src must be a contiguous CUDA tensor")
        n = int(src.shape[0])
        row_bytes = src.element_size() * (src.numel() // max(n, 1))
        dst = torch.empty((n + 7 * int(n_split),) + tuple(src.shape[1:]), dtype=src.dtype, device=src.device)
        self._check(_lib.svr_subdivide_rows(self.handle, _p(split), n, _p(src), _p(dst), row_bytes, 1 if zero else 0, None))
        return dst

    def svr_adam_step(self, theta, grad, m, v, lr: float, beta1: float, beta2: float, eps: float, step: int, zero_grad: bool = True):
        """Fused Adam over flat float32 tensors (in place)."""
        self._check(_lib.svr_adam_step(self.handle, _p(theta), _p(grad), _p(m), _p(v), theta.numel(), lr, beta1, beta2, eps, step,
                                       1 if zero_grad else 0))


    def svr_gather_corners(self, grid, corner_index, raw):
        self._check(_lib.svr_gather_corners(self.handle, _p(grid), _p(corner_index), raw.shape[0], _p(raw)))

    def svr_scatter_add_corners(self, grad_raw, corner_index, grad_grid):
        self._check(_lib.svr_scatter_add_corners(self.handle, _p(grad_raw), _p(corner_index), grad_raw.shape[0], _p(grad_grid)))


def svr_gamma_schedule(t: float, T: float, t0_frac: float = 0.3, t1_frac: float = 0.6, gamma_max: float = 0.6) -> float:
    return float(_lib.svr_gamma_schedule(t, T, t0_frac, t1_frac, gamma_max))


def svr_ssim_static_max_pixels() -> int:
    return int(_lib.svr_ssim_static_max_pixels())


def svr_ssim_loss_grad_static(render: torch.Tensor, target: torch.Tensor, dL: torch.Tensor, loss: torch.Tensor, lam: float = 1.0,
                              accumulate: bool = False, stream: Optional[torch.cuda.Stream] = None):
    """svr_ssim_loss_grad without a Context and without any allocation, for callers that cannot allocate device memory (see
    include/svr.h): the scratch is a fixed array inside libsvr.so, good for images of up to svr_ssim_static_max_pixels()
    pixels. Nothing is allocated here either, so the outputs are the caller's: dL [H,W,3] (written, or added to when
    `accumulate`) and loss [1], float32 on the inputs' device. Runs on `stream` (default: torch's current stream of that
    device). All calls on a device share the one scratch array: keep them ordered on the GPU."""
    for t, name in ((render, "render"), (target, "target"), (dL, "dL"), (loss, "loss")):
        _dev(t, torch.float32, name)
    H, W = int(render.shape[0]), int(render.shape[1])
    dev = render.device.index if render.device.index is not None else torch.cuda.current_device()
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    st = _lib.svr_ssim_loss_grad_static(dev, C.c_void_p(s.cuda_stream), _p(render), _p(target), W, H, lam, 1 if accumulate else 0,
                                        _p(dL), _p(loss))
    if st != SVR_OK:
        raise SvrError(st, _lib.svr_static_last_error().decode())
    return dL, loss
