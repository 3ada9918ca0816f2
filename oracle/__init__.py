"""TEST INFRASTRUCTURE - the CPU oracle (see svr_oracle.cpp and loss.py headers).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this package. The product (paper_2511_02510_b200) never does.
"""
from .binding import (build, lib, num_threads, sh_basis, voxel_rgb, ray, ray_dump, render, backward,
                      bin_rects, bin_lists, pixel_octant)
from .loss import gamma_schedule, lf_loss_and_grad, sobel_magnitude
from . import adam, prune, subdivide

__all__ = ["build", "lib", "num_threads", "sh_basis", "voxel_rgb", "ray", "ray_dump", "render", "backward",
           "bin_rects", "bin_lists", "pixel_octant", "gamma_schedule", "lf_loss_and_grad", "sobel_magnitude", "adam", "prune", "subdivide"]
