"""Pins for the oracle's distance-driven projector pair and its two pose gradients (O15; SURVEY.md section 8f-3,
PAPER.md :213 [44], Tables III / IV rows DD; reading DESIGN.md U14).  CPU only.

Independent references: the textbook separable distance-driven weights written out with numpy overlap matrices for the
two axis-aligned standard views; the hand formula for uniform volumes; the explicit transpose (DD is a matched pair);
closed-form line integrals with their convergence; the paper's stored-G algorithms on BOTH sides (12 G_f volumes
projected; stored central-difference images back-projected, Eq.13, G_b contracted); finite differences.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from helpers import aniso_geom, blobs, cos_sim, rel_l2, small_geom
from test_oracle_joseph import wide_geom
from test_oracle_siddon import object_frame_rays


def overlap_matrix(lo, hi, n):
    """O[i, j] = |[lo_i, hi_i] n [j - 1/2, j + 1/2]| / (hi_i - lo_i): normalised 1-D overlaps of pixel footprints
    (in continuous voxel indices) with the n voxel cells."""
    lo, hi = np.minimum(lo, hi), np.maximum(lo, hi)
    j = np.arange(n)
    ov = np.minimum(hi[:, None], j[None, :] + 0.5) - np.maximum(lo[:, None], j[None, :] - 0.5)
    return np.clip(ov, 0.0, None) / (hi - lo)[:, None]


@pytest.mark.parametrize("beta", [0.0, math.pi / 2])
def test_standard_views_equal_the_textbook_separable_distance_driven_weights(beta):
    """Identity pose, gantry at 0 (driving axis x, u runs along y) and at 90 degrees (driving axis y, u along -x):
    the detector is parallel to the voxel planes, so a pixel's footprint on plane k is the pixel scaled by the
    magnification (source-to-plane distance over SDD) - De Man & Basu's construction.  Per plane the projection is
    O_u . slice . O_v^T with 1-D overlap matrices, times the slab length v_a / |e_a| of the pixel-centre ray."""
    g = W.Geometry(nx=10, ny=12, nz=9, vx=1.3, vy=1.1, vz=0.9, nu=11, nv=8, du=1.5, dv=1.7, sad=90.0, sdd=140.0,
                   cx=0.4, cy=-0.3, cz=0.2, u0=0.3, v0=-0.2)
    rng = np.random.default_rng(0)
    vol = rng.random(g.vol_shape)
    got = oracle.forward_dd(g, [beta], [[0] * 6], vol)[0]
    cu, cv = (g.nu - 1) / 2 + g.u0, (g.nv - 1) / 2 + g.v0
    iu, iv = np.arange(g.nu), np.arange(g.nv)
    zc = lambda v_mm: (v_mm - g.cz) / g.vz + (g.nz - 1) / 2          # mm -> continuous voxel index
    ref = np.zeros(g.det_shape)
    # unit directions of the pixel-centre rays: (-SDD n + (iu-cu) du e_u + (iv-cv) dv e_v) / |.|
    U, V = (iu - cu) * g.du, (iv - cv) * g.dv
    norm = np.sqrt(g.sdd ** 2 + U[None, :] ** 2 + V[:, None] ** 2)
    if beta == 0.0:      # source at (+SAD, 0, 0); e_u = +y; planes x = x_k; depth of plane from the source: SAD - x_k
        L = g.vx / (g.sdd / norm)
        for k in range(g.nx):
            m = (g.sad - (g.cx + (k - (g.nx - 1) / 2) * g.vx)) / g.sdd
            yc = lambda y_mm: (y_mm - g.cy) / g.vy + (g.ny - 1) / 2
            Ou = overlap_matrix(yc((iu - 0.5 - cu) * g.du * m), yc((iu + 0.5 - cu) * g.du * m), g.ny)     # [nu, ny]
            Ov = overlap_matrix(zc((iv - 0.5 - cv) * g.dv * m), zc((iv + 0.5 - cv) * g.dv * m), g.nz)     # [nv, nz]
            ref += L * (Ov @ vol[:, :, k] @ Ou.T)
    else:                # source at (0, +SAD, 0); e_u = -x; planes y = y_k
        L = g.vy / (g.sdd / norm)
        for k in range(g.ny):
            m = (g.sad - (g.cy + (k - (g.ny - 1) / 2) * g.vy)) / g.sdd
            xc = lambda x_mm: (x_mm - g.cx) / g.vx + (g.nx - 1) / 2
            Ou = overlap_matrix(xc(-(iu - 0.5 - cu) * g.du * m), xc(-(iu + 0.5 - cu) * g.du * m), g.nx)   # [nu, nx]
            Ov = overlap_matrix(zc((iv - 0.5 - cv) * g.dv * m), zc((iv + 0.5 - cv) * g.dv * m), g.nz)
            ref += L * (Ov @ vol[:, k, :] @ Ou.T)
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()


def test_uniform_volume_interior_rays_hand_formula():
    """mu = const and every footprint inside the grid: the normalised overlaps of a plane sum to 1, so
    l = mu * n_planes * v_a / |e_a| - under a general pose (in-plane rotation included)."""
    g = wide_geom()
    beta, pose = 0.05, [0.2, -0.3, 0.1, 0.12, -0.03, 0.04]           # driven along x
    p = oracle.forward_dd(g, [beta], [pose], np.full(g.vol_shape, 0.21))[0]
    _, eo = object_frame_rays(g, beta, pose)
    assert np.all(np.abs(eo[..., 0]) > np.maximum(np.abs(eo[..., 1]), np.abs(eo[..., 2])))
    ref = 0.21 * g.nx * g.vx / np.abs(eo[..., 0])
    assert np.abs(p - ref).max() < 1e-12


def test_adjointness_the_backprojector_is_the_exact_transpose():
    g = aniso_geom(nx=10, ny=8, nz=6, nu=9, nv=7)
    rng = np.random.default_rng(4)
    x = rng.standard_normal(g.vol_shape)
    y = rng.standard_normal((3, g.nv, g.nu)).astype(np.float32)
    angles, poses = [0.3, 1.9, 4.0], [[1, -1, 0.5, 0.1, -0.2, 0.3], [0] * 6, [-2, 0.5, 1, -0.15, 0.1, -0.4]]
    lhs = float((oracle.forward_dd(g, angles, poses, x) * y.astype(np.float64)).sum())
    BTy = oracle.backproject_dd(g, angles, poses, y)
    rhs = float((x * BTy).sum())
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    # slabs of the back-projection and the sum over views
    assert np.array_equal(oracle.backproject_dd(g, angles, poses, y, 2, 5), BTy[2:5])
    s = sum(oracle.backproject_dd(g, angles[v:v + 1], poses[v:v + 1], y[v:v + 1]) for v in range(3))
    assert np.abs(s - BTy).max() <= 1e-13 * np.abs(BTy).max()


def test_closed_form_gaussian_blobs_convergence_all_driving_axes():
    """Views driven along x, along y, and (pose tilted by 70 degrees about y) along z; halving h divides the error."""
    bl = blobs(seed=5, n=3, half=9.0, sig=(2.5, 4.0))
    for beta, pose in ((2.9, [1.5, -2.0, 1.0, 0.2, -0.15, 0.3]), (1.4, [0.5, 1.0, -1.0, -0.1, 0.2, 0.1]),
                       (0.1, [0.5, 0.3, 0.2, 0.05, 1.2, 0.0])):
        errs = []
        for k in (1, 2):
            g = aniso_geom(nx=22 * k, ny=18 * k, nz=14 * k, vx=1.1 / k, vy=1.4 / k, vz=1.9 / k,
                           nu=21 * k, nv=17 * k, du=2.1 / k, dv=2.7 / k, u0=0.8 * k, v0=-1.3 * k)
            vol = W.voxelise_blobs(g, bl).double().numpy()
            p = oracle.forward_dd(g, [beta], [pose], vol)[0]
            errs.append(rel_l2(p, W.blob_projection(g, bl, beta, pose).numpy()))
        assert errs[0] < 6e-2 and errs[1] < 2e-2 and errs[0] / errs[1] > 2.5, (beta, errs)


def test_closed_form_ellipsoids_config1():
    w = W.make_config(1)
    p = oracle.forward_dd(w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy())[0]
    cf = w.closed_form(w.poses)[0].numpy()
    assert rel_l2(p, cf) < 4e-2 and abs(p.sum() / cf.sum() - 1) < 3e-3


def test_missed_and_empty_inputs_give_exact_zeros():
    g = small_geom(n=8, nu=6, nv=5)
    far = [[0, 0, 500.0, 0, 0, 0]]
    up = np.ones((1,) + g.det_shape, np.float32)
    assert np.all(oracle.forward_dd(g, [0.2], far, np.ones(g.vol_shape)) == 0)
    assert np.all(oracle.backproject_dd(g, [0.2], far, up) == 0)
    assert np.all(oracle.forward_pose_grad_dd(g, [0.2], far, np.ones(g.vol_shape), up) == 0)
    assert np.all(oracle.backproject_pose_grad_dd(g, [0.2], far, up, np.ones(g.vol_shape, np.float32)) == 0)
    assert np.all(oracle.forward_pose_grad_dd(g, [0.2], [[1, 2, 3, .1, .2, .3]], np.zeros(g.vol_shape), up) == 0)


# ---------------------------------------------------------------- forward pose gradient (Eq.19-20 :179-191)
def stored_Gf_gradient(g, beta, pose, vol, up, forward=None):
    """The paper's algorithm as printed (:189-191) with DD weights: 12 volumes G_f^j = [ (R r'_j) g_j^T | -R g_j ]
    built with numpy, each projected by the (separately pinned) forward_dd, weighted, contracted with dM/dtheta."""
    forward = oracle.forward_dd if forward is None else forward
    R, dR = oracle.rotation(pose)
    pad = np.pad(vol, 1)
    gj = np.stack([(pad[1:-1, 1:-1, 2:] - pad[1:-1, 1:-1, :-2]) / (2 * g.vx),
                   (pad[1:-1, 2:, 1:-1] - pad[1:-1, :-2, 1:-1]) / (2 * g.vy),
                   (pad[2:, 1:-1, 1:-1] - pad[:-2, 1:-1, 1:-1]) / (2 * g.vz)])
    iz, iy, ix = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    rj = np.stack([g.cx + (ix - (g.nx - 1) / 2) * g.vx, g.cy + (iy - (g.ny - 1) / 2) * g.vy,
                   g.cz + (iz - (g.nz - 1) / 2) * g.vz])
    lever = np.einsum("ab,bzyx->azyx", R, rj)
    Rg = np.einsum("ab,bzyx->azyx", R, gj)
    GM = np.zeros((3, 4))
    for a in range(3):
        for b in range(3):
            GM[a, b] = float((forward(g, [beta], [pose], lever[a] * gj[b])[0] * up).sum())
        GM[a, 3] = float((forward(g, [beta], [pose], -Rg[a])[0] * up).sum())
    out = np.zeros(6)
    out[:3] = GM[:, 3]
    for k in range(3):
        out[3 + k] = float((dR[k] * GM[:, :3]).sum())
    return out


def test_forward_gradient_equals_the_projection_of_stored_Gf_volumes():
    g = aniso_geom(nx=12, ny=10, nz=8, nu=9, nv=7)
    rng = np.random.default_rng(6)
    vol = rng.standard_normal(g.vol_shape)
    up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
    for beta, pose in ((0.7, [1.0, -0.5, 0.8, 0.15, -0.1, 0.25]), (2.0, [0, 0, 0, 0, 0, 0])):
        ref = stored_Gf_gradient(g, beta, pose, vol, up)
        got = oracle.forward_pose_grad_dd(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
        assert np.abs(got - ref).max() <= 1e-10 * np.abs(ref).max(), (got, ref)


def test_forward_gradient_vs_finite_differences_of_the_continuous_projection():
    """Paper protocol (Eq.24 :219-222): cosine similarity with central finite differences; the paper reports a mean of
    0.9977 for its DD forward projector (:278)."""
    bl = blobs(seed=8, n=3, half=8.0, sig=(2.5, 4.0))
    g = small_geom(n=40, voxel=0.75, nu=24, nv=20, pix=2.0)
    vol = W.voxelise_blobs(g, bl).double().numpy()
    rng = np.random.default_rng(9)
    sims = []
    for trial in range(3):
        beta = float(rng.uniform(0, 2 * math.pi))
        pose = np.concatenate([rng.uniform(-3, 3, 3), rng.uniform(-0.15, 0.15, 3)])
        up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
        ana = oracle.forward_pose_grad_dd(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
        fd = np.zeros(6)
        for k in range(6):
            e = 1e-5
            pp, pm = pose.copy(), pose.copy()
            pp[k] += e
            pm[k] -= e
            fd[k] = float(((W.blob_projection(g, bl, beta, pp.tolist()).numpy() -
                            W.blob_projection(g, bl, beta, pm.tolist()).numpy()) * up).sum()) / (2 * e)
        sims.append(cos_sim(ana, fd))
    assert min(sims) >= 0.995, sims


# ---------------------------------------------------------------- back-projection pose gradient (Eq.22 :198-206)
@pytest.mark.parametrize("beta,pose", [(0.3, [1.2, -0.8, 0.6, 0.11, -0.07, 0.19]), (2.0, [-2.0, 1.0, 0.3, -0.2, 0.15, -0.4])])
def test_back_gradient_equals_the_papers_stored_Gb_algorithm(beta, pose):
    """PAPER.md :202-206 with DD weights: the two central-difference images of the zero-extended projection, one value
    per detector pixel, each BACK-PROJECTED with the (separately pinned) `backproject_dd`; per voxel
    q_j = B[D_u]_j J_u(r_j) + B[D_v]_j J_v(r_j) with Eq.13's Jacobian from `oracle.projection_matrix` at r_j = R r'_j + t;
    G_b^j = q_j^T (x) (x', y', z', 1) (Eq.15 / 17) summed with the upstream weights and contracted with dM/dtheta.
    Dyadic projection values keep the stored difference images exact in float32."""
    g = aniso_geom()
    rng = np.random.default_rng(23)
    proj = (rng.integers(-64, 65, size=(1,) + g.det_shape) / 64.0).astype(np.float32)
    w = rng.standard_normal(g.vol_shape).astype(np.float32)
    expect = stored_Gb_gradient(g, beta, pose, proj, w, backproject=oracle.backproject_dd)
    got = oracle.backproject_pose_grad_dd(g, [beta], [pose], proj, w)[0]
    assert np.abs(got - expect).max() <= 1e-11 * np.abs(expect).max(), (got, expect)


def stored_Gb_gradient(g, beta, pose, proj, w, backproject):
    """The paper's stored-G_b algorithm (:202-206) for a matched projector pair given by its `backproject`."""
    lp = np.pad(proj[0].astype(np.float64), 1)
    Du = 0.5 * (lp[1:-1, 2:] - lp[1:-1, :-2])
    Dv = 0.5 * (lp[2:, 1:-1] - lp[:-2, 1:-1])
    assert np.array_equal(Du.astype(np.float32), Du) and np.array_equal(Dv.astype(np.float32), Dv)
    Bu = backproject(g, [beta], [pose], Du[None].astype(np.float32))
    Bv = backproject(g, [beta], [pose], Dv[None].astype(np.float32))
    iz, iy, ix = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    rp = np.stack([g.cx + (ix - (g.nx - 1) / 2) * g.vx, g.cy + (iy - (g.ny - 1) / 2) * g.vy,
                   g.cz + (iz - (g.nz - 1) / 2) * g.vz], axis=-1)
    hom = np.concatenate([rp, np.ones(rp.shape[:-1] + (1,))], axis=-1)
    P = oracle.projection_matrix(g, beta)
    R, dR = oracle.rotation(pose)
    r = rp @ R.T + np.asarray(pose[:3])
    up_, vp_, wp_ = (r @ P[k, :3] + P[k, 3] for k in range(3))
    Ju = (P[0, :3] * wp_[..., None] - P[2, :3] * up_[..., None]) / wp_[..., None] ** 2
    Jv = (P[1, :3] * wp_[..., None] - P[2, :3] * vp_[..., None]) / wp_[..., None] ** 2
    q = Bu[..., None] * Ju + Bv[..., None] * Jv
    GM = np.einsum("zyx,zyxa,zyxb->ab", w.astype(np.float64), q, hom)
    return np.concatenate([GM[:, 3], [(dR[k] * GM[:, :3]).sum() for k in range(3)]])


def test_back_gradient_vs_finite_differences_of_the_discrete_dd_backprojector():
    """Paper protocol (Eq.23b :217, Eq.24): L = sum_j w_j mu_j(theta) through the DD back-projector of smooth
    (Gaussian-spot) projections; cosine similarity of the analytical 6-vector with central finite differences of L."""
    # clinical cone (SAD 785): the transpose's weights carry the magnification (sum_i a^ij ~ 1 / m(r_j)^2), a factor the
    # paper's formula treats as part of a^ij, like the FDK weight (U8) - on a toy cone (SAD 120) its neglected
    # derivative alone pulls the cosine down to 0.86-0.96
    g = small_geom(n=14, voxel=2.0, nu=44, nv=40, pix=1.8, sad=785.0, sdd=1200.0)
    bl = blobs(seed=4, n=4, half=8.0, sig=(2.5, 4.5))
    sims = []
    rng = np.random.default_rng(31)
    for beta, pose in ((0.2, [1.2, -0.8, 0.6, 0.11, -0.07, 0.19]), (1.77, [-0.5, 0.4, 0.9, -0.08, 0.05, 0.12])):
        proj = W.blob_projection(g, bl, beta, [0.3, -0.2, 0.1, 0.02, 0.01, -0.03]).numpy()[None].astype(np.float32)
        w = oracle.backproject_dd(g, [beta], [pose], proj)[0:g.nz]            # a smooth, one-signed upstream
        w = (w / np.abs(w).max()).astype(np.float32)
        ana = oracle.backproject_pose_grad_dd(g, [beta], [pose], proj, w)[0]
        fd, eps = np.zeros(6), 1e-4
        for k in range(6):
            pp, pm = np.array(pose, float), np.array(pose, float)
            pp[k] += eps
            pm[k] -= eps
            fd[k] = float(((oracle.backproject_dd(g, [beta], [pp], proj) -
                            oracle.backproject_dd(g, [beta], [pm], proj)) * w).sum()) / (2 * eps)
        sims.append(cos_sim(ana, fd))
    assert min(sims) >= 0.99, sims
