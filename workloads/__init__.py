"""Seeded synthetic inputs for the dfp hot path.

This package is the ONLY code shared by the oracle side (`oracle/`, tests) and the
CUDA side (`paper_2508_13304_b200/`, bench).  It holds input generators only:
seeded random numbers, ellipsoid / Gaussian-blob phantoms, scanner numbers of the
five BASELINE.json configs, closed-form line integrals used to render target data,
the ramp filter that prepares FDK input, and the loss gradients that produce the
upstream arrays.  It holds none of the method's arithmetic (no discrete projector,
no back-projector, no pose gradient) and imports neither `oracle` nor the package.
"""
from .rng import SplitMix64, normal_field, uniform_field
from .geometry import Geometry, view_angles, circular_frame, move_frame, noncircular_orbit, FLAG_VIEW_FRAMES
from .phantom import (Ellipsoid, random_ellipsoids, voxelise_ellipsoids, voxelise_blobs,
                      ellipsoid_projection, blob_projection, rotation_zyx)
from .losses import ncc, ncc_grad, variance_grad, ssd_grad, gradient_entropy
from .ramp import ramp_filter
from .configs import CONFIGS, make_config, base_seed

__all__ = [
    "SplitMix64", "normal_field", "uniform_field", "Geometry", "view_angles", "circular_frame", "move_frame", "noncircular_orbit",
    "FLAG_VIEW_FRAMES", "Ellipsoid",
    "random_ellipsoids", "voxelise_ellipsoids", "voxelise_blobs", "ellipsoid_projection",
    "blob_projection", "rotation_zyx", "ncc", "ncc_grad", "variance_grad", "ssd_grad", "gradient_entropy",
    "ramp_filter", "CONFIGS", "make_config", "base_seed",
]
