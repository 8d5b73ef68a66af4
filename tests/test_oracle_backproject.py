"""Pins for the oracle's voxel-driven back-projector and its pose gradient (O8, O9, O10;
PAPER.md Eq.2b :71-75, Eq.21 :193-196, Eq.9-17 :115-168, Eq.22 :198-206).  CPU only.

Independent references used: plain ray geometry (a voxel placed on the source->pixel line must pick up
exactly that pixel), the textbook FDK reconstruction formula (back-projecting ramp-filtered closed-form
projections must give the object back), an explicit-transpose adjointness check, finite differences of
the (pinned) back-projector itself, and the paper's 12-element G_b route of Eq.15/17.
"""
import math

import numpy as np
import pytest
import torch

import oracle
import workloads as W
from helpers import aniso_geom, blobs, cos_sim, grad_err_u9, small_geom

POSE = [1.2, -0.8, 0.6, 0.11, -0.07, 0.19]


def _scanner_vectors(g, beta):
    n = np.array([math.cos(beta), math.sin(beta), 0.0])
    eu = np.array([-math.sin(beta), math.cos(beta), 0.0])
    ev = np.array([0.0, 0.0, 1.0])
    cu, cv = (g.nu - 1) / 2 + g.u0, (g.nv - 1) / 2 + g.v0
    return n, eu, ev, cu, cv


# ---------------------------------------------------------------- O8 values
@pytest.mark.parametrize("bp_weight", [0, 1])
def test_single_voxel_on_a_pixel_ray_picks_up_that_pixel(bp_weight):
    """A 1-voxel volume whose centre lies on the line source -> pixel (iu,iv) receives exactly that pixel
    (times (SAD/w')^2 for the FDK weight, w' = SAD - r.n = depth from the source); half a pixel off in u it
    receives the mean of the two neighbours (bilinear hat); behind the source it receives nothing."""
    beta, iu, iv, lam = 0.9, 5, 11, 0.55
    g0 = aniso_geom(nx=1, ny=1, nz=1, bp_weight=bp_weight)
    n, eu, ev, cu, cv = _scanner_vectors(g0, beta)
    s = g0.sad * n
    proj = np.random.default_rng(0).standard_normal((1,) + g0.det_shape).astype(np.float32)
    for du_off, expect in ((0.0, proj[0, iv, iu]), (0.5, 0.5 * (float(proj[0, iv, iu]) + float(proj[0, iv, iu + 1])))):
        pix = -(g0.sdd - g0.sad) * n + (iu + du_off - cu) * g0.du * eu + (iv - cv) * g0.dv * ev
        r = s + lam * (pix - s)
        g = g0.replace(cx=float(r[0]), cy=float(r[1]), cz=float(r[2]))
        mu = oracle.backproject(g, [beta], [[0] * 6], proj)[0, 0, 0]
        Wt = (g.sad / (g.sad - r @ n)) ** 2 if bp_weight else 1.0
        assert abs(mu - Wt * expect) < 1e-9
    # the same voxel reached through a pose: r = R r' + t  ->  put r' so that R r' + t is the same world point
    R, _ = oracle.rotation(POSE)
    rp = R.T @ (r - np.array(POSE[:3]))
    g = g0.replace(cx=float(rp[0]), cy=float(rp[1]), cz=float(rp[2]))
    mu2 = oracle.backproject(g, [beta], [POSE], proj)[0, 0, 0]
    assert abs(mu2 - mu) < 1e-9
    # a voxel behind the source (w' <= 0) contributes nothing
    r = s + 5.0 * n
    g = g0.replace(cx=float(r[0]), cy=float(r[1]), cz=float(r[2]))
    assert oracle.backproject(g, [beta], [[0] * 6], proj)[0, 0, 0] == 0.0


def test_fdk_reconstruction_of_a_moved_gaussian_blob():
    """Textbook FDK (Feldkamp-Davis-Kress): f = (dbeta/2) sum_beta (SAD/w')^2 [ramp * (cos-weighted p)] at iso
    pitch.  Data: closed-form projections of a blob that sits at a rigid pose; back-projecting with that same
    pose must return the blob in its own frame.  Pins geometry, pose direction, bilinear sampling, the FDK
    weight and workloads.ramp_filter's normalisation in one go."""
    n_views = 96
    g = W.Geometry(nx=28, ny=28, nz=20, vx=1.0, vy=1.0, vz=1.0, nu=72, nv=40, du=1.0, dv=1.2, sad=400.0, sdd=600.0,
                   bp_weight=1)
    bl = [W.Ellipsoid([1.5, -2.0, 1.0], [3.0, 3.6, 2.8], [0.3, -0.2, 0.5], 0.03)]
    angles = W.view_angles(n_views).numpy()
    poses = np.tile(np.array(POSE), (n_views, 1))
    n, eu, ev, cu, cv = _scanner_vectors(g, 0.0)
    U = (np.arange(g.nu) - cu) * g.du
    V = (np.arange(g.nv) - cv) * g.dv
    cosw = g.sdd / np.sqrt(g.sdd ** 2 + U[None, :] ** 2 + V[:, None] ** 2)
    du_iso = g.du * g.sad / g.sdd
    q = np.empty((n_views,) + g.det_shape, np.float32)
    for v in range(n_views):
        p = W.blob_projection(g, bl, float(angles[v]), POSE)
        q[v] = W.ramp_filter(p * torch.from_numpy(cosw), du_iso).numpy().astype(np.float32)
    rec = oracle.backproject(g, angles, poses, q) * (2 * math.pi / n_views) / 2.0
    truth = W.voxelise_blobs(g, bl).double().numpy()
    err = np.abs(rec - truth).max() / truth.max()
    assert err < 0.03, err
    # without the pose the blob lands elsewhere: the check is sensitive to the pose handling
    rec0 = oracle.backproject(g, angles, np.zeros_like(poses), q) * (2 * math.pi / n_views) / 2.0
    assert np.abs(rec0 - truth).max() / truth.max() > 0.2


def test_backprojection_adjointness_with_explicit_transpose():
    for bw in (0, 1):
        g = aniso_geom(bp_weight=bw)
        rng = np.random.default_rng(1)
        angles = [0.4, 2.2]
        poses = [POSE, [0, 1, -1, -0.2, 0.05, 0.4]]
        y = rng.standard_normal((2,) + g.det_shape).astype(np.float32)
        x = rng.standard_normal(g.vol_shape)
        By = oracle.backproject(g, angles, poses, y)
        BTx = oracle.backproject_T(g, angles, poses, x)
        lhs, rhs = float((By * x).sum()), float((y.astype(np.float64) * BTx).sum())
        assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs))


def test_backprojection_slab_range_views_and_off_detector_voxels():
    g = aniso_geom()
    rng = np.random.default_rng(2)
    y = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    angles, poses = [0.1, 1.3, 4.0], [POSE, [0] * 6, [2, 2, 2, 0.1, 0.1, 0.1]]
    full = oracle.backproject(g, angles, poses, y)
    part = oracle.backproject(g, angles, poses, y, iz0=3, iz1=7)
    assert np.array_equal(part, full[3:7])
    # sum over views = sum of single-view back-projections
    s = sum(oracle.backproject(g, angles[v:v + 1], poses[v:v + 1], y[v:v + 1]) for v in range(3))
    assert np.abs(s - full).max() <= 1e-13 * np.abs(full).max()
    # object pushed out of the cone along z: every voxel projects off the detector -> exact zeros
    far = oracle.backproject(g, [0.1], [[0, 0, 400.0, 0, 0, 0]], y[:1])
    assert np.all(far == 0.0)


# ---------------------------------------------------------------- O9 gradient
def _smooth_projections(g, n_views, seed=4):
    """Smooth (Gaussian-spot) projections: closed-form blob projections at slightly different poses."""
    bl = blobs(seed=seed, n=4, half=8.0, sig=(2.5, 4.5))
    angles = W.view_angles(n_views).numpy() + 0.2
    proj = np.stack([W.blob_projection(g, bl, float(a), [0.3, -0.2, 0.1, 0.02, 0.01, -0.03]).numpy() for a in angles])
    return angles, proj.astype(np.float32)


def _fd_backproject_grad(g, angles, poses, proj, w, eps=1e-7):
    """Central FD of L = sum_j w_j mu_j(theta) with respect to every view's six parameters.  eps is tiny
    because the bilinear interpolant has slope kinks at pixel centres: a voxel whose projection crosses one
    inside [-eps, eps] makes FD average two slopes; the chance of that is proportional to eps."""
    V = len(angles)
    out = np.zeros((V, 6))
    for v in range(V):       # mu is a sum over views: only view v's term depends on theta_v
        for k in range(6):
            pp, pm = np.array(poses[v], float), np.array(poses[v], float)
            pp[k] += eps
            pm[k] -= eps
            mp = oracle.backproject(g, angles[v:v + 1], [pp], proj[v:v + 1])
            mm = oracle.backproject(g, angles[v:v + 1], [pm], proj[v:v + 1])
            out[v, k] = float(((mp - mm) * w).sum() / (2 * eps))
    return out


@pytest.mark.parametrize("bp_weight,flags", [(0, 0), (1, 1)])
def test_backproject_grad_interp_mode_is_the_derivative_of_the_discrete_backprojector(bp_weight, flags):
    """INTERP + (for the FDK weight) the dW/dtheta term reproduce FD of the discrete back-projector:
    pins Eq.13's Jacobian, the chain through r = R r' + t, the axial vectors a_k and all signs (U11: plus)."""
    g = small_geom(n=14, voxel=2.0, nu=24, nv=20, bp_weight=bp_weight, flags=flags)
    angles, proj = _smooth_projections(g, 2)
    poses = [POSE, [-0.5, 0.4, 0.9, -0.08, 0.05, 0.12]]
    w = np.random.default_rng(6).standard_normal(g.vol_shape).astype(np.float32)
    fd = _fd_backproject_grad(g, angles, poses, proj, w)
    an = oracle.backproject_pose_grad(g, angles, poses, proj, w, grad_mode=oracle.GRAD_INTERP)
    for v in range(2):
        assert cos_sim(an[v], fd[v]) > 0.999999
    assert grad_err_u9(an, fd).max() < 2e-3


def test_backproject_grad_central_mode_matches_fd_at_the_papers_cosine_level():
    """Paper protocol (Eq.23b :217, Eq.24 :219-222): L2 loss |B(theta) l - mu_ref|^2 with mu_ref the
    back-projection at another pose; cos-sim of the analytical gradient vs central FD of that loss.  The paper
    reports a mean of 0.9984 for its voxel-driven back-projector (:278)."""
    g = small_geom(n=14, voxel=2.0, nu=44, nv=40, pix=1.2)
    angles, proj = _smooth_projections(g, 2)
    poses = [POSE, [-0.5, 0.4, 0.9, -0.08, 0.05, 0.12]]
    ref = oracle.backproject(g, angles, [[0] * 6] * 2, proj)
    w = (2.0 * (oracle.backproject(g, angles, poses, proj) - ref)).astype(np.float32)      # dL/dmu at `poses`
    eps, fd = 1e-5, np.zeros((2, 6))
    for v in range(2):
        for k in range(6):
            pp, pm = np.array(poses, float), np.array(poses, float)
            pp[v, k] += eps
            pm[v, k] -= eps
            Lp = ((oracle.backproject(g, angles, pp, proj) - ref) ** 2).sum()
            Lm = ((oracle.backproject(g, angles, pm, proj) - ref) ** 2).sum()
            fd[v, k] = (Lp - Lm) / (2 * eps)
    an = oracle.backproject_pose_grad(g, angles, poses, proj, w)
    for v in range(2):
        assert cos_sim(an[v], fd[v]) > 0.998


def test_fdk_weight_without_the_dW_term_is_the_papers_approximation():
    """Reading U8: with W inside a^ij and no dW/dtheta term the result is close to, but not, the FD gradient;
    adding the term (flags bit0) closes the gap."""
    g = small_geom(n=14, voxel=2.0, nu=24, nv=20, bp_weight=1)
    angles, proj = _smooth_projections(g, 1)
    w = np.random.default_rng(6).standard_normal(g.vol_shape).astype(np.float32)
    fd = _fd_backproject_grad(g, angles, [POSE], proj, w)
    a0 = oracle.backproject_pose_grad(g, angles, [POSE], proj, w, grad_mode=oracle.GRAD_INTERP)
    a1 = oracle.backproject_pose_grad(g.replace(flags=1), angles, [POSE], proj, w, grad_mode=oracle.GRAD_INTERP)
    assert 0.9 < cos_sim(a0, fd) < cos_sim(a1, fd)
    assert cos_sim(a1, fd) > 0.999999


def test_backproject_grad_six_accumulators_equal_the_papers_twelve_element_route():
    """Eq.15/17: G_b = q^T (x) (x', y', z', 1) contracted with dM/dtheta == (S_q, a_k . S_c)."""
    for bw, fl in ((0, 0), (1, 0), (1, 1)):
        g = aniso_geom(bp_weight=bw, flags=fl)
        rng = np.random.default_rng(7)
        proj = rng.standard_normal((2,) + g.det_shape).astype(np.float32)
        w = rng.standard_normal(g.vol_shape).astype(np.float32)
        angles, poses = [0.3, 2.0], [POSE, [-2.0, 1.0, 0.3, -0.2, 0.15, -0.4]]
        for mode in (oracle.GRAD_CENTRAL, oracle.GRAD_INTERP):
            a = oracle.backproject_pose_grad(g, angles, poses, proj, w, grad_mode=mode, route=oracle.ROUTE_SIX)
            b = oracle.backproject_pose_grad(g, angles, poses, proj, w, grad_mode=mode, route=oracle.ROUTE_TWELVE)
            assert np.abs(a - b).max() <= 1e-11 * np.abs(b).max()


def test_backproject_grad_of_one_voxel_on_the_central_ray_by_hand():
    """One voxel on the central ray of a view at beta=0, identity pose: J_u = (SDD/du)/w' e_y, J_v = (SDD/dv)/w' e_z
    (Eq.13 :143-146), the central differences are those of the pixel the voxel hits (a pixel CENTRE - the general,
    non-integer (u,v) case is pinned by the stored-G_b test below), rotations move the voxel at (x0,0,0) by hand."""
    g0 = W.Geometry(nx=1, ny=1, nz=1, vx=1, vy=1, vz=1, nu=9, nv=7, du=1.5, dv=2.0, sad=100.0, sdd=160.0)
    proj = np.random.default_rng(8).standard_normal((1,) + g0.det_shape).astype(np.float32)
    x0 = 12.0                                        # voxel on the central axis, 12 mm towards the source
    g = g0.replace(cx=x0)
    w = np.ones(g.vol_shape, np.float32)
    an = oracle.backproject_pose_grad(g, [0.0], [[0] * 6], proj, w)[0]
    cu, cv = 4, 3
    dlu = 0.5 * (float(proj[0, cv, cu + 1]) - float(proj[0, cv, cu - 1]))
    dlv = 0.5 * (float(proj[0, cv + 1, cu]) - float(proj[0, cv - 1, cu]))
    wp = g.sad - x0
    expect_t = np.array([0.0, dlu * (g.sdd / g.du) / wp, dlv * (g.sdd / g.dv) / wp])
    assert np.abs(an[:3] - expect_t).max() < 1e-12
    # rotations about the origin move the voxel at (x0,0,0): d r/d gz = (0,x0,0), d r/d gy = (0,0,-x0), d r/d gx = 0
    expect_r = np.array([0.0, -x0 * expect_t[2], x0 * expect_t[1]])
    assert np.abs(an[3:] - expect_r).max() < 1e-12


def _dyadic(rng, shape, bits=6, span=64):
    """Random values k / 2^bits, |k| <= span: sums, differences and halves of a few of them are exact in float32."""
    return (rng.integers(-span, span + 1, size=shape) / float(1 << bits)).astype(np.float32)


@pytest.mark.parametrize("bp_weight", [0, 1])
def test_backproject_grad_central_mode_equals_the_papers_stored_Gb_algorithm(bp_weight):
    """The paper's algorithm taken literally (PAPER.md :202-206, Eq.22 :200): "the gradient of the projection is
    computed with central finite difference", "compute matrix G_b^i for each detector pixel", "backproject each
    element of G_b", "accumulate" - here with STORED images instead of on-the-fly values:
      1. the two central-difference images D_u[iv][iu] = (l[iv][iu+1] - l[iv][iu-1]) / 2, D_v likewise, of the
         zero-extended projection, stored on the detector padded by one pixel per side (beyond it both neighbours
         are outside the detector); shifting by exactly one pixel keeps the bilinear weights, so the interpolated
         central difference of b~ IS the bilinear interpolation of these images;
      2. each image back-projected with `oracle.backproject` (O8, pinned above) on a general anisotropic grid, pose
         and view -> B[D_u]_j, B[D_v]_j (the weight W of a^ij included);
      3. q_j = B[D_u]_j J_u(j) + B[D_v]_j J_v(j), J from Eq.13 (:143-146) built here in numpy from
         `oracle.projection_matrix` (Eq.1, pinned by hand values) at r_j = R r'_j + t;
      4. the 12-element G_b^j = q_j^T (x) (x', y', z', 1) (Eq.15 / 17 :155-168) summed with the upstream weights and
         contracted with dM/dtheta (`oracle.rotation`: R, dR/dgamma_k, pinned by finite differences).
    The projection values are dyadic rationals so that the stored difference images are exact in float32.
    This pins `backproject_grad_impl` CENTRAL at NON-INTEGER (u, v): replacing its two difference lines
    (0.5 * (b~(u+1,v) - b~(u-1,v)), same in v) by the half-pixel form b~(u+1/2,v) - b~(u-1/2,v) - which coincides
    with it at pixel centres and passed every other pin - fails this test at the 1e-2 level (checked by mutation
    when the test was written)."""
    g = aniso_geom(bp_weight=bp_weight)
    rng = np.random.default_rng(21)
    angles = [0.3, 2.0]
    poses = [POSE, [-2.0, 1.0, 0.3, -0.2, 0.15, -0.4]]
    proj = _dyadic(rng, (2,) + g.det_shape)
    w = rng.standard_normal(g.vol_shape).astype(np.float32)
    # 1. stored difference images on the padded detector: index iu' = iu + 1; c_u' = c_u + 1 needs u0' = u0
    gp = g.replace(nu=g.nu + 2, nv=g.nv + 2)
    lp = np.zeros((2, g.nv + 4, g.nu + 4))                       # zero extension by two pixels per side
    lp[:, 2:-2, 2:-2] = proj
    Du = 0.5 * (lp[:, 1:-1, 2:] - lp[:, 1:-1, :-2])
    Dv = 0.5 * (lp[:, 2:, 1:-1] - lp[:, :-2, 1:-1])
    assert np.array_equal(Du.astype(np.float32), Du) and np.array_equal(Dv.astype(np.float32), Dv)
    # voxel centres r'_j (O1)
    iz, iy, ix = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    rp = np.stack([g.cx + (ix - (g.nx - 1) / 2) * g.vx, g.cy + (iy - (g.ny - 1) / 2) * g.vy,
                   g.cz + (iz - (g.nz - 1) / 2) * g.vz], axis=-1)                            # [nz,ny,nx,3]
    hom = np.concatenate([rp, np.ones(rp.shape[:-1] + (1,))], axis=-1)
    expect = np.zeros((2, 6))
    for v in range(2):
        # 2. back-project each stored image
        Bu = oracle.backproject(gp, angles[v:v + 1], poses[v:v + 1], Du[v:v + 1].astype(np.float32))
        Bv = oracle.backproject(gp, angles[v:v + 1], poses[v:v + 1], Dv[v:v + 1].astype(np.float32))
        # 3. Jacobian of Eq.13 at r_j = R r'_j + t
        P = oracle.projection_matrix(g, angles[v])
        R, dR = oracle.rotation(poses[v])
        r = rp @ R.T + np.asarray(poses[v][:3])
        up_ = r @ P[0, :3] + P[0, 3]
        vp_ = r @ P[1, :3] + P[1, 3]
        wp_ = r @ P[2, :3] + P[2, 3]
        assert (wp_ > 0).all()
        Ju = (P[0, :3][None, None, None, :] * wp_[..., None] - P[2, :3][None, None, None, :] * up_[..., None]) / wp_[..., None] ** 2
        Jv = (P[1, :3][None, None, None, :] * wp_[..., None] - P[2, :3][None, None, None, :] * vp_[..., None]) / wp_[..., None] ** 2
        q = Bu[..., None] * Ju + Bv[..., None] * Jv                                           # [nz,ny,nx,3]
        # 4. grad_M L = sum_j w_j q_j^T (x) (x',y',z',1);  dL/dtheta_k = <dM/dtheta_k, grad_M L>
        GM = np.einsum("zyx,zyxa,zyxb->ab", w.astype(np.float64), q, hom)                     # [3,4]
        expect[v, :3] = GM[:, 3]                                                              # dM/dt_k = [0 | e_k]
        for k in range(3):
            expect[v, 3 + k] = (dR[k] * GM[:, :3]).sum()                                      # dM/dgamma_k = [dR_k | 0]
    for route in (oracle.ROUTE_SIX, oracle.ROUTE_TWELVE):
        an = oracle.backproject_pose_grad(g, angles, poses, proj, w, grad_mode=oracle.GRAD_CENTRAL, route=route)
        assert np.abs(an - expect).max() <= 1e-11 * np.abs(expect).max(), (an, expect)
    # the voxels do not sit on pixel centres: the identity is exercised at general fractional (u, v)
    frac = np.abs((up_ / wp_) - np.rint(up_ / wp_))
    assert np.median(frac) > 0.1


def test_backproject_grad_zero_cases_and_linearity():
    g = aniso_geom()
    rng = np.random.default_rng(9)
    proj = rng.standard_normal((2,) + g.det_shape).astype(np.float32)
    w = rng.standard_normal(g.vol_shape).astype(np.float32)
    angles, poses = [0.3, 2.0], [POSE, [0, 0, 400.0, 0, 0, 0]]
    a = oracle.backproject_pose_grad(g, angles, poses, proj, w)
    assert np.all(a[1] == 0.0) and np.all(a[0] != 0.0)
    assert np.all(oracle.backproject_pose_grad(g, angles, poses, 0 * proj, w) == 0.0)
    b = oracle.backproject_pose_grad(g, angles, poses, 2 * proj, 2 * w)
    assert np.allclose(b, 4 * a, rtol=1e-12)
