"""B200-native differentiable sparse-voxel tile rasterizer (LiteVoxel hot path, arXiv 2511.02510).

`paper_2511_02510_b200.<name>` resolves through `binding`, which loads libsvr.so (hand-written CUDA for
sm_100a, built in-tree by `_build.py`). The load is deferred to first use only so that `_build` can be
imported before the library exists; there is no fallback path: a missing library raises ImportError, a
missing GPU raises at Context().
"""
_NAMES = ["Context", "Frame", "Voxels", "SvrCamera", "SvrError", "SvrLossOpts", "SvrPruneOpts", "SvrRenderOpts", "SvrSubdivOpts", "SvrVoxels", "EXPORTS",
          "make_camera", "svr_gamma_schedule", "svr_ssim_loss_grad_static", "svr_ssim_static_max_pixels", "lib"]
__all__ = list(_NAMES)


def __getattr__(name):
    if name in _NAMES:
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
