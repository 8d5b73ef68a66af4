"""Pins for the oracle's Joseph projector and its pose gradient (O13).  CPU only.

Joseph's method steps the ray from voxel-centre plane to voxel-centre plane along its driving axis and interpolates
bilinearly in each plane.  Pins: hand formulas for volumes that bilinear interpolation reproduces exactly (constants,
functions linear in the two in-plane coordinates), the explicit transpose, closed-form line integrals with their
convergence order, the paper's stored-G algorithm, finite differences of closed-form projections.
"""
import math

import numpy as np

import oracle
import workloads as W
from helpers import aniso_geom, blobs, cos_sim, rel_l2, small_geom
from test_oracle_siddon import object_frame_rays


def wide_geom():
    """A grid much wider (y, z) than the fan: every plane intersection keeps its 4 bilinear neighbours inside."""
    return W.Geometry(nx=9, ny=41, nz=37, vx=1.3, vy=1.1, vz=0.9, nu=7, nv=5, du=1.5, dv=1.7, sad=150.0, sdd=230.0,
                      cx=0.4, cy=-0.3, cz=0.2, u0=0.3, v0=-0.2)


def test_uniform_volume_interior_rays_hand_formula():
    """mu = const and all bilinear supports inside the grid: l = mu * n_planes * v_a / |e_a| (weights sum to 1)."""
    g = wide_geom()
    beta, pose = 0.05, [0.2, -0.3, 0.1, 0.02, -0.03, 0.04]           # rays driven along x
    p = oracle.forward_joseph(g, [beta], [pose], np.full(g.vol_shape, 0.21))[0]
    _, eo = object_frame_rays(g, beta, pose)
    assert np.all(np.abs(eo[..., 0]) > np.maximum(np.abs(eo[..., 1]), np.abs(eo[..., 2])))
    ref = 0.21 * g.nx * g.vx / np.abs(eo[..., 0])
    assert np.abs(p - ref).max() < 1e-12
    # an exactly axis-parallel ray: the plain chord n * v
    g1 = small_geom(n=8, nu=5, nv=5)
    assert abs(oracle.forward_joseph(g1, [0.0], [[0] * 6], np.ones(g1.vol_shape))[0][2, 2] - 8 * 1.25) < 1e-12


def test_volume_linear_in_the_plane_coordinates_hand_formula():
    """f = a + b y + c z: bilinear interpolation is exact for it, so l = (vx/|ex|) sum_k f(y(t_k), z(t_k)) with the
    ray's own intersection points - evaluated here from the ray equation, no interpolation involved."""
    g = wide_geom()
    beta, pose = -0.04, [0.1, 0.2, -0.2, -0.03, 0.02, 0.05]
    iz, iy, ix = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    y = g.cy + (iy - (g.ny - 1) / 2) * g.vy
    z = g.cz + (iz - (g.nz - 1) / 2) * g.vz
    a, b, c = 0.7, 0.031, -0.017
    p = oracle.forward_joseph(g, [beta], [pose], a + b * y + c * z)[0]
    so, eo = object_frame_rays(g, beta, pose)
    xk = g.cx + (np.arange(g.nx) - (g.nx - 1) / 2) * g.vx
    ref = np.zeros(g.det_shape)
    for iv in range(g.nv):
        for iu in range(g.nu):
            e = eo[iv, iu]
            t = (xk - so[0]) / e[0]
            ref[iv, iu] = g.vx / abs(e[0]) * np.sum(a + b * (so[1] + t * e[1]) + c * (so[2] + t * e[2]))
    assert np.abs(p - ref).max() < 1e-11


def test_adjointness_with_the_explicit_transpose():
    g = aniso_geom(nx=10, ny=8, nz=6, nu=9, nv=7)
    rng = np.random.default_rng(4)
    x = rng.standard_normal(g.vol_shape)
    y = rng.standard_normal((3, g.nv, g.nu))
    angles, poses = [0.3, 1.9, 4.0], [[1, -1, 0.5, 0.1, -0.2, 0.3], [0] * 6, [-2, 0.5, 1, -0.15, 0.1, -0.4]]
    lhs = float((oracle.forward_joseph(g, angles, poses, x) * y).sum())
    rhs = float((x * oracle.forward_joseph_T(g, angles, poses, y)).sum())
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_closed_form_gaussian_blobs_second_order_convergence_all_driving_axes():
    """Views driven along x, along y, and (pose tilted by 70 degrees about y) along z."""
    bl = blobs(seed=5, n=3, half=9.0, sig=(2.5, 4.0))
    for beta, pose in ((2.9, [1.5, -2.0, 1.0, 0.2, -0.15, 0.3]), (1.4, [0.5, 1.0, -1.0, -0.1, 0.2, 0.1]),
                       (0.1, [0.5, 0.3, 0.2, 0.05, 1.2, 0.0])):
        errs = []
        for k in (1, 2):
            g = aniso_geom(nx=22 * k, ny=18 * k, nz=14 * k, vx=1.1 / k, vy=1.4 / k, vz=1.9 / k)
            vol = W.voxelise_blobs(g, bl).double().numpy()
            p = oracle.forward_joseph(g, [beta], [pose], vol)[0]
            errs.append(rel_l2(p, W.blob_projection(g, bl, beta, pose).numpy()))
        assert errs[0] < 4e-2 and errs[1] < 1.2e-2 and errs[0] / errs[1] > 2.5, (beta, errs)


def test_closed_form_ellipsoids_config1():
    w = W.make_config(1)
    p = oracle.forward_joseph(w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy())[0]
    cf = w.closed_form(w.poses)[0].numpy()
    assert rel_l2(p, cf) < 3e-2 and abs(p.sum() / cf.sum() - 1) < 2e-3


def test_missed_and_empty_volumes_give_exact_zeros():
    g = small_geom(n=8, nu=6, nv=5)
    assert np.all(oracle.forward_joseph(g, [0.2], [[0, 0, 500.0, 0, 0, 0]], np.ones(g.vol_shape)) == 0)
    up = np.ones((1,) + g.det_shape, np.float32)
    assert np.all(oracle.forward_pose_grad_joseph(g, [0.2], [[0, 0, 500.0, 0, 0, 0]], np.ones(g.vol_shape), up) == 0)
    assert np.all(oracle.forward_pose_grad_joseph(g, [0.2], [[1, 2, 3, .1, .2, .3]], np.zeros(g.vol_shape), up) == 0)


# ---------------------------------------------------------------- pose gradient (Eq.19-20 :179-191)
def stored_G_gradient(g, beta, pose, vol, up):
    """The paper's algorithm as printed (:189-191) with Joseph weights: 12 volumes G_f^j = [ (R r'_j) g_j^T | -R g_j ]
    built with numpy, each projected by the (separately pinned) forward_joseph, weighted, contracted with dM/dtheta."""
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
            GM[a, b] = float((oracle.forward_joseph(g, [beta], [pose], lever[a] * gj[b])[0] * up).sum())
        GM[a, 3] = float((oracle.forward_joseph(g, [beta], [pose], -Rg[a])[0] * up).sum())
    out = np.zeros(6)
    out[:3] = GM[:, 3]
    for k in range(3):
        out[3 + k] = float((dR[k] * GM[:, :3]).sum())
    return out


def test_gradient_equals_the_projection_of_stored_G_volumes():
    g = aniso_geom(nx=12, ny=10, nz=8, nu=9, nv=7)
    rng = np.random.default_rng(6)
    vol = rng.standard_normal(g.vol_shape)
    up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
    for beta, pose in ((0.7, [1.0, -0.5, 0.8, 0.15, -0.1, 0.25]), (2.0, [0, 0, 0, 0, 0, 0])):
        ref = stored_G_gradient(g, beta, pose, vol, up)
        got = oracle.forward_pose_grad_joseph(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
        assert np.abs(got - ref).max() <= 1e-10 * np.abs(ref).max(), (got, ref)


def test_gradient_vs_finite_differences_of_the_continuous_projection():
    bl = blobs(seed=8, n=3, half=8.0, sig=(2.5, 4.0))
    g = small_geom(n=40, voxel=0.75, nu=24, nv=20, pix=2.0)
    vol = W.voxelise_blobs(g, bl).double().numpy()
    rng = np.random.default_rng(9)
    sims = []
    for trial in range(3):
        beta = float(rng.uniform(0, 2 * math.pi))
        pose = np.concatenate([rng.uniform(-3, 3, 3), rng.uniform(-0.15, 0.15, 3)])
        up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
        ana = oracle.forward_pose_grad_joseph(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
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
