"""Pins for the oracle's explicit view frames (O14: flags & 64, one (s, c, U, V) frame per view instead of a gantry
angle - SURVEY.md 8b optional extension, PAPER.md :244 non-circular orbit).  CPU only.

What fixes the result without reference to the code under test:
  * Eq.1 (:60-63): every point of the line source -> pixel centre must map to that pixel's index, w' is the depth
    from the source along the detector normal - for tilted, skewed (non-orthogonal U, V), off-centre detectors;
  * closed-form line integrals of Gaussian blobs for a general frame (the renderer builds its own rays);
  * the frame of a circular-orbit view reproduces the (separately pinned) circular path to round-off;
  * moving scanner and object together changes nothing: frame (Q F + tau) with pose (R, t) == frame F with pose
    (Q^T R, Q^T (t - tau)) - checked with Q = Rz so that the Euler angles stay explicit - and for a general rigid
    motion of the scanner against the closed form;
  * the pose gradients under a general frame against finite differences of the discrete projector / back-projector.
"""
import numpy as np

import oracle
import workloads as W
from helpers import aniso_geom, blobs, cos_sim, grad_err_u9, rel_l2, small_geom

VF = W.FLAG_VIEW_FRAMES
POSE = [1.2, -0.8, 0.9, 0.07, -0.05, 0.11]


def _general_frame(g, beta=0.6, skew=True):
    """A scanner nowhere near the circular orbit: source off the mid-plane, detector tilted about all three axes and
    shifted, pixel steps of unequal length and (skew) not orthogonal."""
    Q = W.rotation_zyx(0.12, -0.2, 0.3)
    f = W.move_frame(W.circular_frame(g, beta), Q, [4.0, -3.0, 6.0]).reshape(4, 3).clone()
    f[1] += 2.5 * f[2] - 1.5 * f[3]                # reference point away from the foot of the perpendicular
    f[0] += W.rotation_zyx(0, 0, beta) @ W.rotation_zyx(0, 0, 0)[:, 0] * 9.0 + W.rotation_zyx(0, 0, beta)[:, 1] * 5.0 - \
        W.rotation_zyx(0, 0, beta)[:, 2] * 7.0   # source moved on its own: SAD, SDD change
    if skew:
        f[3] = f[3] + 0.15 * f[2]
        f[2] = 1.1 * f[2]
    return f.reshape(-1).numpy()


def test_projection_matrix_of_a_general_frame_maps_pixel_centres_to_their_indices():
    g = aniso_geom(flags=VF)
    for skew in (False, True):
        f = _general_frame(g, skew=skew)
        s, c, U, V = f.reshape(4, 3)
        P = oracle.projection_matrix(g, f)
        cu, cv = (g.nu - 1) / 2 + g.u0, (g.nv - 1) / 2 + g.v0
        nh = np.cross(U, V)
        nh /= np.linalg.norm(nh)
        if (c - s) @ nh < 0:
            nh = -nh
        for iu, iv in ((0, 0), (g.nu - 1, 3), (7, g.nv - 1), (2.25, 5.5)):
            pix = c + (iu - cu) * U + (iv - cv) * V
            for lam in (0.3, 1.0, 1.7):
                r = s + lam * (pix - s)
                h = P @ np.append(r, 1.0)
                assert abs(h[0] / h[2] - iu) < 1e-10 and abs(h[1] / h[2] - iv) < 1e-10
                assert abs(h[2] - (r - s) @ nh) < 1e-10            # w' = depth from the source, mm
        assert abs((P @ np.append(s, 1.0))[2]) < 1e-10


def test_frame_of_a_circular_view_reproduces_the_circular_path():
    g = aniso_geom()
    gf = g.replace(flags=VF)
    vol = W.voxelise_blobs(g, blobs(seed=4, n=3, half=7.0, sig=(2.5, 4.0))).numpy()
    rng = np.random.default_rng(2)
    betas = [0.0, 0.9, -2.2]
    poses = [POSE, [0.0] * 6, [-2.0, 1.0, 0.5, -0.1, 0.2, -0.3]]
    frames = np.stack([W.circular_frame(g, b).numpy() for b in betas])
    for b, f in zip(betas, frames):
        assert np.abs(oracle.projection_matrix(gf, f) - oracle.projection_matrix(g, b)).max() < 1e-10
    p0 = oracle.forward(g, betas, poses, vol)
    p1 = oracle.forward(gf, frames, poses, vol)
    assert rel_l2(p1, p0) < 1e-13
    w = rng.standard_normal(p0.shape).astype(np.float32)
    for mode in (oracle.GRAD_CENTRAL, oracle.GRAD_INTERP):
        a0 = oracle.forward_pose_grad(g, betas, poses, vol, w, grad_mode=mode)
        a1 = oracle.forward_pose_grad(gf, frames, poses, vol, w, grad_mode=mode)
        assert np.abs(a1 - a0).max() < 1e-10 * np.abs(a0).max()
    proj = p0.astype(np.float32)
    up = rng.standard_normal(g.vol_shape).astype(np.float32)
    for bw, fl in ((0, 0), (1, 0), (1, 1)):
        ga, gb = g.replace(bp_weight=bw, flags=fl), g.replace(bp_weight=bw, flags=fl | VF)
        assert rel_l2(oracle.backproject(gb, frames, poses, proj), oracle.backproject(ga, betas, poses, proj)) < 1e-13
        b0 = oracle.backproject_pose_grad(ga, betas, poses, proj, up)
        b1 = oracle.backproject_pose_grad(gb, frames, poses, proj, up)
        assert np.abs(b1 - b0).max() < 1e-10 * np.abs(b0).max()
    assert rel_l2(oracle.forward_siddon(gf, frames, poses, vol), oracle.forward_siddon(g, betas, poses, vol)) < 1e-12
    assert rel_l2(oracle.forward_joseph(gf, frames, poses, vol), oracle.forward_joseph(g, betas, poses, vol)) < 1e-12


def test_forward_under_a_general_frame_matches_closed_form_blobs():
    bl = blobs(seed=5, n=3, half=8.0, sig=(2.5, 4.0))
    errs = []
    for k in (1, 2):
        g = aniso_geom(nx=22 * k, ny=18 * k, nz=14 * k, vx=1.1 / k, vy=1.4 / k, vz=1.9 / k, flags=VF)
        f = _general_frame(g)
        vol = W.voxelise_blobs(g, bl).double().numpy()
        p = oracle.forward(g, [f], [POSE], vol)[0]
        cf = W.blob_projection(g, bl, f, POSE).numpy()
        errs.append(rel_l2(p, cf))
    assert errs[0] < 3e-2 and errs[0] / errs[1] > 3.0          # second-order convergence to the exact integral


def test_moving_scanner_and_object_together_changes_nothing():
    """Frame Rz(d) F + tau with pose (R, t) is frame F with pose (Rz(-d) R, Rz(-d)(t - tau)); for R = Rz Ry Rx the
    left factor only shifts gamma_z, so both sides are explicit poses: values equal, dL/dgamma equal, dL/dt rotated."""
    g = small_geom(n=20, voxel=1.5, nu=16, nv=14, flags=VF)
    vol = W.voxelise_blobs(g, blobs(seed=6, n=3, half=7.0, sig=(2.5, 4.0))).numpy()
    d, tau = 0.37, np.array([3.0, -2.0, 1.5])
    Qz = W.rotation_zyx(0, 0, d).numpy()
    F = _general_frame(g, beta=0.4)
    Fm = W.move_frame(F, Qz, tau).numpy()
    pose_m = np.array(POSE)
    pose_0 = np.concatenate([Qz.T @ (pose_m[:3] - tau), [POSE[3], POSE[4], POSE[5] - d]])
    p_m = oracle.forward(g, [Fm], [pose_m], vol)
    p_0 = oracle.forward(g, [F], [pose_0], vol)
    assert rel_l2(p_m, p_0) < 1e-12
    w = np.random.default_rng(3).standard_normal(p_0.shape).astype(np.float32)
    g_m = oracle.forward_pose_grad(g, [Fm], [pose_m], vol, w)[0]
    g_0 = oracle.forward_pose_grad(g, [F], [pose_0], vol, w)[0]
    assert np.abs(g_m[:3] - Qz @ g_0[:3]).max() < 1e-10 * np.abs(g_0[:3]).max()
    assert np.abs(g_m[3:] - g_0[3:]).max() < 1e-10 * np.abs(g_0[3:]).max()
    proj = p_0.astype(np.float32)
    for bw in (0, 1):
        gb = g.replace(bp_weight=bw)
        v_m = oracle.backproject(gb, [Fm], [pose_m], proj)
        v_0 = oracle.backproject(gb, [F], [pose_0], proj)
        assert rel_l2(v_m, v_0) < 1e-12
        up = np.random.default_rng(4).standard_normal(g.vol_shape).astype(np.float32)
        b_m = oracle.backproject_pose_grad(gb, [Fm], [pose_m], proj, up)[0]
        b_0 = oracle.backproject_pose_grad(gb, [F], [pose_0], proj, up)[0]
        assert np.abs(b_m[:3] - Qz @ b_0[:3]).max() < 1e-10 * np.abs(b_0[:3]).max()
        assert np.abs(b_m[3:] - b_0[3:]).max() < 1e-10 * np.abs(b_0[3:]).max()


def test_pose_gradients_under_a_general_frame_match_finite_differences():
    g = small_geom(n=24, voxel=1.25, nu=20, nv=18, flags=VF)
    F = _general_frame(g, beta=1.1)
    vol = W.voxelise_blobs(g, blobs(seed=3, n=3, half=8.0, sig=(2.5, 4.0))).double().numpy()
    w = np.random.default_rng(5).standard_normal(g.det_shape).astype(np.float32)
    eps = 1e-6    # the discrete projector is piecewise smooth in theta: a small step keeps both FD points on one piece

    def fd(fun):
        out = np.zeros(6)
        for k in range(6):
            pp, pm = list(POSE), list(POSE)
            pp[k] += eps
            pm[k] -= eps
            out[k] = (fun(pp) - fun(pm)) / (2 * eps)
        return out

    ref = fd(lambda th: float((oracle.forward(g, [F], [th], vol)[0] * w).sum()))
    an = oracle.forward_pose_grad(g, [F], [POSE], vol, w[None], grad_mode=oracle.GRAD_INTERP)[0]
    assert cos_sim(an, ref) > 0.9999999 and grad_err_u9(an, ref).max() < 1e-4
    # the paper's own estimator (central differences) under its own protocol (Eq.23a / 24): L2 loss, cosine with FD
    target = oracle.forward(g, [F], [[0.0] * 6], vol)[0]
    w2 = (2.0 * (oracle.forward(g, [F], [POSE], vol)[0] - target)).astype(np.float32)
    ref2 = fd(lambda th: float(((oracle.forward(g, [F], [th], vol)[0] - target) ** 2).sum()))
    an_c = oracle.forward_pose_grad(g, [F], [POSE], vol, w2[None])[0]
    assert cos_sim(an_c, ref2) > 0.995

    # back-projector: smooth projections (closed-form blobs), random upstream volume
    proj = W.blob_projection(g, blobs(seed=8, n=3, half=8.0, sig=(3.0, 5.0)), F, [0.0] * 6).numpy().astype(np.float32)
    up = np.random.default_rng(6).standard_normal(g.vol_shape).astype(np.float32)
    for bw, fl in ((0, 0), (1, 1)):
        gb = g.replace(bp_weight=bw, flags=VF | fl)
        ref = fd(lambda th: float((oracle.backproject(gb, [F], [th], proj[None]) * up).sum()))
        an = oracle.backproject_pose_grad(gb, [F], [POSE], proj[None], up, grad_mode=oracle.GRAD_INTERP)[0]
        assert cos_sim(an, ref) > 0.999999 and grad_err_u9(an, ref).max() < 2e-3     # a few voxels cross a pixel edge
