"""Shared test helpers (small geometries, error metrics).  No method arithmetic here."""
import math

import numpy as np
import torch

import workloads as W

DEG = math.pi / 180.0


def small_geom(n=24, voxel=1.25, nu=20, nv=18, pix=2.4, sad=120.0, sdd=200.0, **kw) -> W.Geometry:
    """A toy cone-beam scanner with a wide cone (stresses the geometry more than the clinical ones)."""
    return W.Geometry(nx=n, ny=n, nz=n, vx=voxel, vy=voxel, vz=voxel, nu=nu, nv=nv, du=pix, dv=pix,
                      sad=sad, sdd=sdd, **kw).f32()


def aniso_geom(**kw) -> W.Geometry:
    """Non-cubic grid, non-square pixels, shifted principal point and volume centre."""
    d = dict(nx=22, ny=18, nz=14, vx=1.1, vy=1.4, vz=1.9, nu=21, nv=17, du=2.1, dv=2.7, sad=130.0, sdd=210.0,
             cx=1.5, cy=-2.0, cz=0.7, u0=0.8, v0=-1.3)
    d.update(kw)
    return W.Geometry(**d).f32()


def blobs(seed=3, n=3, half=10.0, sig=(2.0, 4.0), amp=(0.01, 0.04)):
    rng = W.SplitMix64(seed)
    return W.random_ellipsoids(rng, n, sig, amp, half, 3.0 * sig[1])


def random_pose(rng, t=5.0, r_deg=8.0):
    return [rng.uniform(-t, t) for _ in range(3)] + [rng.uniform(-r_deg, r_deg) * DEG for _ in range(3)]


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def cos_sim(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    return float(a @ b / (np.linalg.norm(a) * np.linalg.norm(b)))


def grad_err_u9(g, ref):
    """SURVEY.md U9 / DESIGN.md: per view, per component
    |g_k - ref_k| / max(|ref_k|, 0.01 * max_{k' in same group} |ref_k'|), groups = translations, rotations."""
    g = np.asarray(g, dtype=np.float64).reshape(-1, 6)
    ref = np.asarray(ref, dtype=np.float64).reshape(-1, 6)
    err = np.zeros_like(ref)
    for sl in (slice(0, 3), slice(3, 6)):
        floor = 0.01 * np.abs(ref[:, sl]).max(axis=1, keepdims=True)
        den = np.maximum(np.abs(ref[:, sl]), floor)
        den = np.maximum(den, 1e-300)
        err[:, sl] = np.abs(g[:, sl] - ref[:, sl]) / den
    return err


def t64(a):
    return torch.as_tensor(np.asarray(a), dtype=torch.float64)


def check_values(got, ref, tol_l2=1e-5, tol_abs=5e-5, zero_border=True):
    """Values (projections, back-projections) against the oracle: the stated metric (relative L2 <= 1e-5), backed by a
    per-element bound - max |got - ref| <= 5e-5 max|ref|, five times the L2 tolerance (an fp32
    result carries ~1e-6 of its own magnitude, so only a wrong element - a tile edge, a missed sample - can exceed it) -
    and by the zero pattern: where the oracle is exactly zero (rays / voxels that miss) the CUDA result is exactly zero
    too (`zero_border`: inputs whose outermost voxels / pixels are zero, all workloads' phantoms) or below 1e-6 of the
    largest value (white-noise inputs: a sample within fp32 rounding of the support's edge may pick up a last voxel)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape and np.all(np.isfinite(got))
    scale = np.abs(ref).max()
    if scale == 0.0:
        assert not got.any(), "oracle is all zero, the CUDA result is not"
        return 0.0
    e = rel_l2(got, ref)
    assert e <= tol_l2, e
    assert np.abs(got - ref).max() <= tol_abs * scale, (np.abs(got - ref).max() / scale)
    z = ref == 0
    if z.any():
        if zero_border:
            assert not got[z].any(), "non-zero where the oracle is exactly zero"
        else:
            assert np.abs(got[z]).max() <= 1e-6 * scale
    return e
