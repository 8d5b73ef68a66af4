"""paper_2508_13304_b200 - B200-native differentiable cone-beam forward / back-projector (arXiv 2508.13304).

The product is `libdfp.so` (hand-written CUDA for sm_100a behind the C ABI in include/dfp.h).  This package is
the thin Python binding with the same names: argument marshalling only, every step of the path runs in the
library's kernels.  torch is used for device memory and streams.  There is no CPU fallback.
"""
from .binding import (DfpError, Geometry, backproject, backproject_host, backproject_pose_grad,
                      backproject_pose_grad_host, count_ray_steps, forward, forward_host, forward_pose_grad,
                      forward_pose_grad_host, last_kernel_ms, last_launch_count, set_kernel_timing, lib_path, status_string, version,
                      workspace_bytes, workspace_bytes_for_views, OP_FORWARD, OP_FORWARD_POSE_GRAD, OP_BACKPROJECT, OP_BACKPROJECT_POSE_GRAD,
                      OP_FORWARD_FUSED, OP_NCC, forward_fused_moments, ncc_pose_grad, ncc_pose_grad_static, NCC_STATIC_MAX_VIEWS,
                      FLAG_DW, FLAG_NO_TMA, FLAG_GRAD_INTERP, FLAG_SIDDON, FLAG_ACCUMULATE, FLAG_JOSEPH, FLAG_VIEW_FRAMES, FLAG_DD, FLAG_SF, PATH_GATHER, PATH_TMA, last_path)

__all__ = ["DfpError", "Geometry", "forward", "forward_pose_grad", "backproject", "backproject_pose_grad",
           "forward_host", "forward_pose_grad_host", "backproject_host", "backproject_pose_grad_host",
           "workspace_bytes", "workspace_bytes_for_views", "count_ray_steps", "last_launch_count", "set_kernel_timing", "last_kernel_ms", "status_string", "version", "lib_path",
           "OP_FORWARD", "OP_FORWARD_POSE_GRAD", "OP_BACKPROJECT", "OP_BACKPROJECT_POSE_GRAD", "OP_FORWARD_FUSED",
           "forward_fused_moments", "ncc_pose_grad", "ncc_pose_grad_static", "NCC_STATIC_MAX_VIEWS", "OP_NCC", "FLAG_DW", "FLAG_NO_TMA", "FLAG_GRAD_INTERP", "FLAG_SIDDON", "FLAG_ACCUMULATE", "FLAG_JOSEPH", "FLAG_VIEW_FRAMES", "FLAG_DD", "FLAG_SF", "PATH_GATHER", "PATH_TMA", "last_path"]
