"""Pins for the oracle's forward pose gradient (O3, O7; Eq.3-8 :81-113, Eq.19-20 :179-191).  CPU only.

None of these re-types the oracle's formula: they use central finite differences of the oracle's own
*forward projector* (already pinned by closed forms in test_oracle_forward.py) and of the closed-form
projections, the paper's structural identity "gradient of a projection = projection of G with the same
a^ij" (:179-181) carried out literally with stored volumes, and the 12-element G_f route of Eq.6-8.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from helpers import aniso_geom, blobs, cos_sim, grad_err_u9, small_geom

POSE = [1.2, -0.8, 0.6, 0.11, -0.07, 0.19]
BETA = 0.7


def _fd_loss_grad(g, beta, pose, vol, w, eps=1e-4):
    """Central FD of L(theta) = sum_i w_i l_i(theta) through the oracle's forward projector."""
    out = np.zeros(6)
    for k in range(6):
        pp, pm = list(pose), list(pose)
        pp[k] += eps
        pm[k] -= eps
        lp = oracle.forward(g, [beta], [pp], vol)[0]
        lm = oracle.forward(g, [beta], [pm], vol)[0]
        out[k] = float(((lp - lm) * w).sum() / (2 * eps))
    return out


def _smooth_case(n=28, fine=False):
    g = small_geom(n=n, voxel=30.0 / n, nu=20, nv=18)
    if fine:
        g = g.replace(step_mm=g.vx * 0.5)
    vol = W.voxelise_blobs(g, blobs(seed=3, n=3, half=8.0, sig=(2.5, 4.0))).double().numpy()
    w = np.random.default_rng(5).standard_normal(g.det_shape).astype(np.float32)
    return g, vol, w


def test_interp_mode_is_the_derivative_of_the_discrete_projector():
    """grad_mode=INTERP must reproduce FD of the discrete projector: pins the chain rule, the lever
    arm, the axial vectors w_k, dL/dt = -R S_A and every sign, component by component."""
    g, vol, w = _smooth_case()
    fd = _fd_loss_grad(g, BETA, POSE, vol, w)
    an = oracle.forward_pose_grad(g, [BETA], [POSE], vol, w[None], grad_mode=oracle.GRAD_INTERP)[0]
    assert cos_sim(an, fd) > 0.99999
    assert grad_err_u9(an, fd).max() < 3e-2


def test_central_mode_matches_fd_at_the_papers_cosine_level():
    """The paper's own accuracy protocol (Eq.23a :215, Eq.24 :219-222): L2 loss against a projection at
    another pose, cos-sim of the analytical gradient vs central FD of the loss; the paper reports a mean
    of 0.9952 for its ray-driven projector (:278).  On smooth phantoms the method does better."""
    g, vol, _ = _smooth_case()
    target = oracle.forward(g, [BETA], [[0.0] * 6], vol)[0]
    w = (2.0 * (oracle.forward(g, [BETA], [POSE], vol)[0] - target)).astype(np.float32)   # dL/dl at POSE
    eps, fd = 1e-4, np.zeros(6)
    for k in range(6):
        pp, pm = list(POSE), list(POSE)
        pp[k] += eps
        pm[k] -= eps
        Lp = ((oracle.forward(g, [BETA], [pp], vol)[0] - target) ** 2).sum()
        Lm = ((oracle.forward(g, [BETA], [pm], vol)[0] - target) ** 2).sum()
        fd[k] = (Lp - Lm) / (2 * eps)
    an = oracle.forward_pose_grad(g, [BETA], [POSE], vol, w[None])[0]
    assert cos_sim(an, fd) > 0.995
    assert cos_sim(an[:3], fd[:3]) > 0.9995


def _central_difference_volumes(g, vol):
    """Stored per-voxel central differences of the zero-extended volume on a grid padded by one voxel."""
    p = np.pad(vol, 2)
    gx = (p[1:-1, 1:-1, 2:] - p[1:-1, 1:-1, :-2]) / (2 * g.vx)
    gy = (p[1:-1, 2:, 1:-1] - p[1:-1, :-2, 1:-1]) / (2 * g.vy)
    gz = (p[2:, 1:-1, 1:-1] - p[:-2, 1:-1, 1:-1]) / (2 * g.vz)
    gp = g.replace(nx=g.nx + 2, ny=g.ny + 2, nz=g.nz + 2)
    return gp, (gx, gy, gz)


def test_translation_gradient_equals_projection_of_stored_volume_gradient():
    """north_star invariant: dL/dt = -R * <w, A[d mu/d x']>, to round-off (not a tolerance-level check).
    Pins O3 (on-the-fly central difference == interpolated stored central-difference volume)."""
    g = aniso_geom()
    vol = np.random.default_rng(1).standard_normal(g.vol_shape)
    w = np.random.default_rng(2).standard_normal(g.det_shape).astype(np.float32)
    gp, grads = _central_difference_volumes(g, vol)
    SA = np.array([float((oracle.forward(gp, [BETA], [POSE], gv)[0] * w).sum()) for gv in grads])
    R, _ = oracle.rotation(POSE)
    an = oracle.forward_pose_grad(g, [BETA], [POSE], vol, w[None])[0]
    assert np.abs(an[:3] - (-R @ SA)).max() <= 1e-12 * np.abs(SA).max()
    # identity pose: dl_i/dt_a = -(A d_a mu)_i exactly
    an0 = oracle.forward_pose_grad(g, [BETA], [[0] * 6], vol, w[None])[0]
    SA0 = np.array([float((oracle.forward(gp, [BETA], [[0] * 6], gv)[0] * w).sum()) for gv in grads])
    assert np.abs(an0[:3] + SA0).max() <= 1e-12 * np.abs(SA0).max()


def test_six_accumulator_route_equals_the_papers_twelve_element_route():
    """Eq.6-8: G_f = [ (r-t) g^T | -R g ] contracted with dM/dtheta  ==  (-R S_A, -w_k . S_B)."""
    g = aniso_geom()
    vol = np.random.default_rng(3).standard_normal(g.vol_shape)
    w = np.random.default_rng(4).standard_normal((2,) + g.det_shape).astype(np.float32)
    angles, poses = [0.3, 2.0], [POSE, [-2.0, 1.0, 0.3, -0.2, 0.15, -0.4]]
    for mode in (oracle.GRAD_CENTRAL, oracle.GRAD_INTERP):
        a = oracle.forward_pose_grad(g, angles, poses, vol, w, grad_mode=mode, route=oracle.ROUTE_SIX)
        b = oracle.forward_pose_grad(g, angles, poses, vol, w, grad_mode=mode, route=oracle.ROUTE_TWELVE)
        assert np.abs(a - b).max() <= 1e-11 * np.abs(b).max()


def test_voxel_lever_arm_equals_literal_stored_G_algorithm():
    """PAPER.md :189-191 literally: build the twelve G_f^j volumes (central-difference gradient and lever
    arm at voxel centres), forward-project each with the same a^ij, weight by dL/dl, contract with
    dM/dtheta.  Must equal the oracle's on-the-fly VOXEL mode to round-off."""
    g = small_geom(n=12, voxel=2.0, nu=9, nv=8)
    vol = np.random.default_rng(6).standard_normal(g.vol_shape)
    w = np.random.default_rng(7).standard_normal(g.det_shape).astype(np.float32)
    gp, (gx, gy, gz) = _central_difference_volumes(g, vol)
    R, dR = oracle.rotation(POSE)
    # voxel-centre coordinates r'_j on the padded grid, and the lever arm r_j - t = R r'_j
    ax = [gp_c + (np.arange(n) - (n - 1) / 2.0) * v for gp_c, n, v in
          ((gp.cx, gp.nx, gp.vx), (gp.cy, gp.ny, gp.vy), (gp.cz, gp.nz, gp.vz))]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    rp = np.stack([X, Y, Z])                       # [3, nz, ny, nx]
    lever = np.einsum("ab,bzyx->azyx", R, rp)
    gr = np.stack([gx, gy, gz])
    Rg = np.einsum("ab,bzyx->azyx", R, gr)
    GM = np.zeros((3, 4))
    for a in range(3):
        for b in range(4):
            Gab = lever[a] * gr[b] if b < 3 else -Rg[a]
            GM[a, b] = float((oracle.forward(gp, [BETA], [POSE], np.ascontiguousarray(Gab))[0] * w).sum())
    lit = np.concatenate([GM[:, 3], [float((dR[k] * GM[:, :3]).sum()) for k in range(3)]])
    an = oracle.forward_pose_grad(g, [BETA], [POSE], vol, w[None], lever_arm=oracle.LEVER_VOXEL)[0]
    assert np.abs(an - lit).max() <= 1e-11 * np.abs(lit).max()


def test_sample_and_voxel_lever_arms_agree_closely_on_smooth_volumes():
    """Reading U2: the two lever-arm choices differ at O(h^2) only."""
    g, vol, w = _smooth_case()
    a = oracle.forward_pose_grad(g, [BETA], [POSE], vol, w[None], lever_arm=oracle.LEVER_SAMPLE)[0]
    b = oracle.forward_pose_grad(g, [BETA], [POSE], vol, w[None], lever_arm=oracle.LEVER_VOXEL)[0]
    assert cos_sim(a, b) > 0.9999
    assert np.abs(a[:3] - b[:3]).max() <= 1e-12 * np.abs(a[:3]).max()   # translations have no lever arm


def test_gradient_approaches_the_continuous_truth():
    """FD of the CLOSED-FORM Gaussian-blob projection (independent of any discretisation)."""
    bl = blobs(seed=3, n=3, half=8.0, sig=(2.5, 4.0))
    g = small_geom(n=40, voxel=0.75, nu=20, nv=18)
    vol = W.voxelise_blobs(g, bl).double().numpy()
    w = np.random.default_rng(5).standard_normal(g.det_shape).astype(np.float32)
    eps = 1e-5
    fd = np.zeros(6)
    for k in range(6):
        pp, pm = list(POSE), list(POSE)
        pp[k] += eps
        pm[k] -= eps
        fd[k] = float(((W.blob_projection(g, bl, BETA, pp) - W.blob_projection(g, bl, BETA, pm)).numpy() * w).sum()
                      / (2 * eps))
    an = oracle.forward_pose_grad(g, [BETA], [POSE], vol, w[None])[0]
    assert cos_sim(an, fd) > 0.9995
    # small components carry 10-100 % discretisation error; the dominant ones are at the few-% level
    big = np.abs(fd) > 0.1 * np.abs(fd).max()
    assert (np.abs(an - fd)[big] / np.abs(fd)[big]).max() < 5e-2


def test_gradient_of_a_missed_or_empty_volume_is_zero_and_views_are_independent():
    g = small_geom(n=10, nu=7, nv=6)
    vol = np.random.default_rng(8).standard_normal(g.vol_shape).astype(np.float32)
    w = np.random.default_rng(9).standard_normal((3,) + g.det_shape).astype(np.float32)
    angles = [0.1, 1.0, 2.0]
    poses = [POSE, [0, 0, 900.0, 0, 0, 0], [0.5, 0.2, -0.3, 0.05, 0.02, -0.04]]
    gr = oracle.forward_pose_grad(g, angles, poses, vol, w)
    assert np.all(gr[1] == 0.0) and np.all(gr[0] != 0.0)
    solo = oracle.forward_pose_grad(g, [angles[2]], [poses[2]], vol, w[2:3])[0]
    assert np.array_equal(solo, gr[2])
    assert np.all(oracle.forward_pose_grad(g, angles, poses, 0 * vol, w) == 0.0)


def test_gradient_is_linear_in_upstream_and_volume():
    g = small_geom(n=10, nu=7, nv=6)
    rng = np.random.default_rng(10)
    v1, v2 = rng.standard_normal(g.vol_shape), rng.standard_normal(g.vol_shape)
    w1 = rng.standard_normal((1,) + g.det_shape).astype(np.float32)
    f = lambda v, w: oracle.forward_pose_grad(g, [BETA], [POSE], v, w)[0]
    assert np.allclose(f(v1 + 2 * v2, w1), f(v1, w1) + 2 * f(v2, w1), rtol=0, atol=1e-11 * np.abs(f(v1, w1)).max())
    assert np.allclose(f(v1, 2 * w1), 2 * f(v1, w1), rtol=1e-12)   # x2 is exact in the float32 upstream
