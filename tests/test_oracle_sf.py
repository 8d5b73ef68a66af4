"""Pins for the oracle's separable-footprint projector pair SF-TR and its two pose gradients (O16; SURVEY.md section
8f-3, PAPER.md :213 [29], Tables III / IV rows SF; reading DESIGN.md U16).  CPU only.

Independent references: the mass of a voxel's footprint against the brute-force integral of its exact chord image; the
textbook SF-TR weights for the two axis-aligned standard views, written from the scanner's numbers with numpy (the
reading linearises the footprint, so the agreement is 1 %, not round-off); the explicit transpose; closed-form line integrals with their convergence; the paper's stored-G
algorithms on both sides; finite differences.
"""
import math

import numpy as np
import pytest

import oracle
import workloads as W
from helpers import aniso_geom, blobs, cos_sim, rel_l2, small_geom


def pixel_integral_of_trapezoid(tau, lo, hi):
    """int_lo^hi of the unit-height trapezoid with sorted vertices tau[0..3]: trapezoidal rule on the union of the
    interval's ends and the vertices inside it (exact: the integrand is linear between those points)."""
    xs = np.unique(np.clip(np.concatenate([[lo, hi], tau]), lo, hi))
    ys = np.interp(xs, tau + np.array([0, 0, 0, 0]), [0.0, 1.0, 1.0, 0.0], left=0.0, right=0.0)
    if tau[0] == tau[1]:
        ys = np.where(xs == tau[0], 1.0 if tau[2] > tau[0] else ys, ys)
    return float(np.trapezoid(ys, xs))


@pytest.mark.parametrize("beta", [0.0, math.pi / 2])
def test_standard_views_agree_with_the_textbook_sf_tr_weights(beta):
    """Identity pose, gantry at 0 (rays along -x: transaxial plane (x, y), u along +y) and at 90 degrees (rays along -y,
    u along -x), v along z: SF-TR as in Long, Fessler & Balter - per voxel the trapezoid from the four (x, y) corners
    under the fan-beam map u = c_u + (SDD/du) y' / (SAD - x'), the rectangle from z -+ vz/2 at the voxel centre's depth,
    the amplitude v_a |e| / |e_a| of the ray to the voxel centre.  The oracle's reading (U16) linearises the footprint about
    the voxel centre and uses trapezoids along both axes, so the two agree to the order of (voxel size / depth): the
    projections of a random volume within 1 %, their sums within 0.1 %."""
    g = W.Geometry(nx=7, ny=8, nz=6, vx=1.3, vy=1.1, vz=0.9, nu=13, nv=9, du=1.5, dv=1.7, sad=90.0, sdd=140.0,
                   cx=0.4, cy=-0.3, cz=0.2, u0=0.3, v0=-0.2)
    rng = np.random.default_rng(0)
    vol = rng.random(g.vol_shape)
    got = oracle.forward_sf(g, [beta], [[0] * 6], vol)[0]
    cu, cv = (g.nu - 1) / 2 + g.u0, (g.nv - 1) / 2 + g.v0
    ref = np.zeros(g.det_shape)
    for iz in range(g.nz):
        for iy in range(g.ny):
            for ix in range(g.nx):
                x = g.cx + (ix - (g.nx - 1) / 2) * g.vx
                y = g.cy + (iy - (g.ny - 1) / 2) * g.vy
                z = g.cz + (iz - (g.nz - 1) / 2) * g.vz
                if beta == 0.0:           # source (SAD, 0, 0): depth SAD - x, lateral +y
                    depth = lambda xx, yy: g.sad - xx
                    lat = lambda xx, yy: yy
                    va = g.vx
                else:                     # source (0, SAD, 0): depth SAD - y, lateral -x
                    depth = lambda xx, yy: g.sad - yy
                    lat = lambda xx, yy: -xx
                    va = g.vy
                tau = np.sort([cu + (g.sdd / g.du) * lat(x + sx * g.vx / 2, y + sy * g.vy / 2) /
                               depth(x + sx * g.vx / 2, y + sy * g.vy / 2) for sx in (-1, 1) for sy in (-1, 1)])
                d0 = depth(x, y)
                t = np.sort([cv + (g.sdd / g.dv) * (z + sz * g.vz / 2) / d0 for sz in (-1, 1)])
                e = np.array([d0, lat(x, y), z])                      # source -> voxel centre: (depth, lateral, axial)
                L = va * np.linalg.norm(e) / abs(e[0])
                for iv in range(g.nv):
                    fv = min(t[1], iv + 0.5) - max(t[0], iv - 0.5)
                    if fv <= 0:
                        continue
                    for iu in range(g.nu):
                        if iu + 0.5 <= tau[0] or iu - 0.5 >= tau[3]:
                            continue
                        ref[iv, iu] += L * pixel_integral_of_trapezoid(tau, iu - 0.5, iu + 0.5) * fv * vol[iz, iy, ix]
    assert rel_l2(got, ref) <= 1e-2 and abs(got.sum() / ref.sum() - 1) <= 1e-3, (rel_l2(got, ref), got.sum() / ref.sum())


def box_chord(so, e, half):
    """Length of the line so + t e (t real) inside the box [-half, half] (slab method), vectorised over rays."""
    with np.errstate(divide="ignore", invalid="ignore"):
        t0 = (-half - so) / e
        t1 = (half - so) / e
    lo = np.minimum(t0, t1).max(axis=-1)
    hi = np.maximum(t0, t1).min(axis=-1)
    return np.clip(hi - lo, 0.0, None)


@pytest.mark.parametrize("beta,pose,centre", [(0.3, [1.2, -0.8, 0.6, 0.11, -0.07, 0.19], [3.0, -2.0, 1.5]),
                                              (1.9, [-2.0, 1.0, 0.3, -0.2, 0.35, -0.4], [-4.0, 2.5, -3.0]),
                                              (0.1, [0.5, 0.3, 0.2, 0.05, 1.2, 0.0], [1.0, 1.0, -2.0])])
def test_mass_of_a_voxel_footprint_equals_the_integral_of_its_exact_chord_image(beta, pose, centre):
    """sum_i a^ij - obtained by back-projecting an image of ones onto a one-voxel volume - against the integral over the
    detector (pixel units) of the EXACT chord length of the voxel's box along each ray, computed by brute force: rays
    from the source through an 8 x 8 sub-grid of every pixel, slab-method chord in the object frame.  Pins the
    amplitude (the area magnification sqrt(det J J^T) of Eq.13's Jacobian, the voxel volume), under in-plane rotation and
    on all three driving axes; the footprint's linearisation costs < 0.3 %."""
    g = W.Geometry(nx=1, ny=1, nz=1, vx=1.1, vy=1.4, vz=0.9, nu=40, nv=36, du=0.5, dv=0.6, sad=300.0, sdd=480.0,
                   cx=centre[0], cy=centre[1], cz=centre[2])
    ones = np.ones((1,) + g.det_shape, np.float32)
    mass = oracle.backproject_sf(g, [beta], [pose], ones)[0, 0, 0]
    R, _ = oracle.rotation(pose)
    t = np.asarray(pose[:3], float)
    n = np.array([math.cos(beta), math.sin(beta), 0.0])
    eu, ev = np.array([-math.sin(beta), math.cos(beta), 0.0]), np.array([0.0, 0.0, 1.0])
    src = g.sad * n
    sub = 8
    off = (np.arange(sub) + 0.5) / sub - 0.5
    uu = (np.arange(g.nu)[:, None] + off[None, :]).ravel() - (g.nu - 1) / 2
    vv = (np.arange(g.nv)[:, None] + off[None, :]).ravel() - (g.nv - 1) / 2
    pts = -(g.sdd - g.sad) * n + uu[None, :, None] * g.du * eu + vv[:, None, None] * g.dv * ev     # [nv*sub, nu*sub, 3]
    d = pts - src
    d /= np.linalg.norm(d, axis=-1, keepdims=True)
    so = R.T @ (src - t) - np.asarray(centre)                       # object frame, relative to the voxel centre
    eo = d @ R                                                       # R^T d
    chord = box_chord(so, eo, 0.5 * np.array([g.vx, g.vy, g.vz]))
    brute = chord.sum() / sub ** 2                                   # integral in pixel units
    assert chord[0].max() == 0 and chord[-1].max() == 0 and chord[:, 0].max() == 0 and chord[:, -1].max() == 0
    assert abs(mass / brute - 1) < 3e-3, (mass, brute)


def test_adjointness_the_backprojector_is_the_exact_transpose():
    g = aniso_geom(nx=10, ny=8, nz=6, nu=9, nv=7)
    rng = np.random.default_rng(4)
    x = rng.standard_normal(g.vol_shape)
    y = rng.standard_normal((3, g.nv, g.nu)).astype(np.float32)
    angles, poses = [0.3, 1.9, 4.0], [[1, -1, 0.5, 0.1, -0.2, 0.3], [0] * 6, [-2, 0.5, 1, -0.15, 0.1, -0.4]]
    lhs = float((oracle.forward_sf(g, angles, poses, x) * y.astype(np.float64)).sum())
    BTy = oracle.backproject_sf(g, angles, poses, y)
    rhs = float((x * BTy).sum())
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    assert np.array_equal(oracle.backproject_sf(g, angles, poses, y, 2, 5), BTy[2:5])
    s = sum(oracle.backproject_sf(g, angles[v:v + 1], poses[v:v + 1], y[v:v + 1]) for v in range(3))
    assert np.abs(s - BTy).max() <= 1e-13 * np.abs(BTy).max()


def test_closed_form_gaussian_blobs_convergence_all_driving_axes():
    bl = blobs(seed=5, n=3, half=9.0, sig=(2.5, 4.0))
    for beta, pose in ((2.9, [1.5, -2.0, 1.0, 0.2, -0.15, 0.3]), (1.4, [0.5, 1.0, -1.0, -0.1, 0.2, 0.1]),
                       (0.1, [0.5, 0.3, 0.2, 0.05, 1.2, 0.0])):
        errs = []
        for k in (1, 2):
            g = aniso_geom(nx=22 * k, ny=18 * k, nz=14 * k, vx=1.1 / k, vy=1.4 / k, vz=1.9 / k,
                           nu=21 * k, nv=17 * k, du=2.1 / k, dv=2.7 / k, u0=0.8 * k, v0=-1.3 * k)
            vol = W.voxelise_blobs(g, bl).double().numpy()
            p = oracle.forward_sf(g, [beta], [pose], vol)[0]
            errs.append(rel_l2(p, W.blob_projection(g, bl, beta, pose).numpy()))
        assert errs[0] < 6e-2 and errs[1] < 2.5e-2 and errs[0] / errs[1] > 2.0, (beta, errs)


def test_closed_form_ellipsoids_config1_and_zeros():
    w = W.make_config(1)
    p = oracle.forward_sf(w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy())[0]
    cf = w.closed_form(w.poses)[0].numpy()
    assert rel_l2(p, cf) < 4e-2 and abs(p.sum() / cf.sum() - 1) < 3e-3
    g = small_geom(n=8, nu=6, nv=5)
    far = [[0, 0, 500.0, 0, 0, 0]]
    up = np.ones((1,) + g.det_shape, np.float32)
    assert np.all(oracle.forward_sf(g, [0.2], far, np.ones(g.vol_shape)) == 0)
    assert np.all(oracle.backproject_sf(g, [0.2], far, up) == 0)
    assert np.all(oracle.forward_pose_grad_sf(g, [0.2], far, np.ones(g.vol_shape), up) == 0)
    assert np.all(oracle.backproject_pose_grad_sf(g, [0.2], far, up, np.ones(g.vol_shape, np.float32)) == 0)


# ---------------------------------------------------------------- pose gradients (Eq.19-20, Eq.22)
def test_forward_gradient_equals_the_projection_of_stored_Gf_volumes():
    from test_oracle_dd import stored_Gf_gradient
    g = aniso_geom(nx=12, ny=10, nz=8, nu=9, nv=7)
    rng = np.random.default_rng(6)
    vol = rng.standard_normal(g.vol_shape)
    up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
    for beta, pose in ((0.7, [1.0, -0.5, 0.8, 0.15, -0.1, 0.25]), (2.0, [0, 0, 0, 0, 0, 0])):
        ref = stored_Gf_gradient(g, beta, pose, vol, up, forward=oracle.forward_sf)
        got = oracle.forward_pose_grad_sf(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
        assert np.abs(got - ref).max() <= 1e-10 * np.abs(ref).max(), (got, ref)


def test_forward_gradient_vs_finite_differences_of_the_continuous_projection():
    """Eq.24; the paper reports a mean of 0.9978 for its SF forward projector (:278)."""
    bl = blobs(seed=8, n=3, half=8.0, sig=(2.5, 4.0))
    g = small_geom(n=40, voxel=0.75, nu=24, nv=20, pix=2.0)
    vol = W.voxelise_blobs(g, bl).double().numpy()
    rng = np.random.default_rng(9)
    sims = []
    for trial in range(3):
        beta = float(rng.uniform(0, 2 * math.pi))
        pose = np.concatenate([rng.uniform(-3, 3, 3), rng.uniform(-0.15, 0.15, 3)])
        up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
        ana = oracle.forward_pose_grad_sf(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
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


@pytest.mark.parametrize("beta,pose", [(0.3, [1.2, -0.8, 0.6, 0.11, -0.07, 0.19]), (2.0, [-2.0, 1.0, 0.3, -0.2, 0.15, -0.4])])
def test_back_gradient_equals_the_papers_stored_Gb_algorithm(beta, pose):
    from test_oracle_dd import stored_Gb_gradient
    g = aniso_geom()
    rng = np.random.default_rng(23)
    proj = (rng.integers(-64, 65, size=(1,) + g.det_shape) / 64.0).astype(np.float32)
    w = rng.standard_normal(g.vol_shape).astype(np.float32)
    expect = stored_Gb_gradient(g, beta, pose, proj, w, backproject=oracle.backproject_sf)
    got = oracle.backproject_pose_grad_sf(g, [beta], [pose], proj, w)[0]
    assert np.abs(got - expect).max() <= 1e-11 * np.abs(expect).max(), (got, expect)


def test_back_gradient_vs_finite_differences_of_the_discrete_sf_backprojector():
    g = small_geom(n=14, voxel=2.0, nu=44, nv=40, pix=1.8, sad=785.0, sdd=1200.0)
    bl = blobs(seed=4, n=4, half=8.0, sig=(2.5, 4.5))
    sims = []
    for beta, pose in ((0.2, [1.2, -0.8, 0.6, 0.11, -0.07, 0.19]), (1.77, [-0.5, 0.4, 0.9, -0.08, 0.05, 0.12])):
        proj = W.blob_projection(g, bl, beta, [0.3, -0.2, 0.1, 0.02, 0.01, -0.03]).numpy()[None].astype(np.float32)
        w = oracle.backproject_sf(g, [beta], [pose], proj)
        w = (w / np.abs(w).max()).astype(np.float32)
        ana = oracle.backproject_pose_grad_sf(g, [beta], [pose], proj, w)[0]
        fd, eps = np.zeros(6), 1e-4
        for k in range(6):
            pp, pm = np.array(pose, float), np.array(pose, float)
            pp[k] += eps
            pm[k] -= eps
            fd[k] = float(((oracle.backproject_sf(g, [beta], [pp], proj) -
                            oracle.backproject_sf(g, [beta], [pm], proj)) * w).sum()) / (2 * eps)
        sims.append(cos_sim(ana, fd))
    assert min(sims) >= 0.99, sims
