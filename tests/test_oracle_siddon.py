"""Pins for the oracle's Siddon projector and its pose gradient (O12).  CPU only.

Siddon's exact radiological path (PAPER.md :213, ref [28] :395) is the weight model of the paper's own ray-driven
projector: a^ij = length of ray i inside voxel j.  Each test checks the oracle against something other than itself:
the chord of a box (closed form), brute-force clipping of the ray against every voxel's own box, the explicit
transpose, closed-form line integrals, the paper's literal stored-G algorithm, finite differences of closed forms.
"""
import math

import numpy as np

import oracle
import workloads as W
from helpers import aniso_geom, blobs, cos_sim, rel_l2, small_geom


def object_frame_rays(g, beta, pose):
    """Source s' and unit directions e'[iv][iu] in the object frame, built here from DESIGN.md O4/O5 with numpy."""
    R = W.rotation_zyx(*pose[3:]).numpy()
    t = np.asarray(pose[:3], float)
    n = np.array([math.cos(beta), math.sin(beta), 0.0])
    eu = np.array([-math.sin(beta), math.cos(beta), 0.0])
    ev = np.array([0.0, 0.0, 1.0])
    s = g.sad * n
    cu, cv = (g.nu - 1) / 2 + g.u0, (g.nv - 1) / 2 + g.v0
    iu, iv = np.meshgrid(np.arange(g.nu), np.arange(g.nv), indexing="xy")
    pix = (-(g.sdd - g.sad) * n)[None, None] + ((iu - cu) * g.du)[..., None] * eu + ((iv - cv) * g.dv)[..., None] * ev
    d = pix - s
    d /= np.linalg.norm(d, axis=-1, keepdims=True)
    return R.T @ (s - t), d @ R          # R^T (s - t),  R^T e  (row vectors)


def box_chord(lo, hi, o, d):
    """Length of the half-line o + t d (t >= 0) inside the box [lo, hi]: the slab method, by hand."""
    t0, t1 = 0.0, np.inf
    for a in range(3):
        if abs(d[a]) < 1e-300:
            if not (lo[a] < o[a] < hi[a]):
                return 0.0
            continue
        ta, tb = (lo[a] - o[a]) / d[a], (hi[a] - o[a]) / d[a]
        t0, t1 = max(t0, min(ta, tb)), min(t1, max(ta, tb))
    return max(t1 - t0, 0.0)


def grid_box(g):
    c = np.array([g.cx, g.cy, g.cz])
    half = 0.5 * np.array([g.nx * g.vx, g.ny * g.vy, g.nz * g.vz])
    return c - half, c + half


def test_uniform_volume_gives_the_chord_of_the_grid_box():
    """mu = const: sum_j a^ij = geometric path length through the grid (closed form), to round-off."""
    g = aniso_geom(nx=11, ny=9, nz=7, nu=13, nv=10)
    beta, pose = 0.8, [1.0, -2.0, 0.5, 0.12, -0.2, 0.3]
    p = oracle.forward_siddon(g, [beta], [pose], np.full(g.vol_shape, 0.37))[0]
    so, eo = object_frame_rays(g, beta, pose)
    lo, hi = grid_box(g)
    ref = np.array([[0.37 * box_chord(lo, hi, so, eo[iv, iu]) for iu in range(g.nu)] for iv in range(g.nv)])
    assert (ref > 0).mean() > 0.3 and (ref == 0).any()           # some rays hit, some miss
    assert np.abs(p - ref).max() < 1e-12
    assert np.array_equal(p == 0, ref == 0)


def test_matches_brute_force_clipping_against_every_voxel():
    """a^ij by clipping the ray against voxel j's own box, voxel by voxel (no traversal, no sorting)."""
    g = aniso_geom(nx=6, ny=5, nz=4, nu=7, nv=5)
    rng = np.random.default_rng(3)
    vol = rng.standard_normal(g.vol_shape)
    for beta, pose in ((0.4, [0.5, 1.0, -0.7, 0.2, 0.1, -0.3]), (math.pi / 2, [0] * 6), (3.9, [-2, 1, 0.5, -0.3, 0.25, 0.6])):
        p = oracle.forward_siddon(g, [beta], [pose], vol)[0]
        so, eo = object_frame_rays(g, beta, pose)
        lo, _ = grid_box(g)
        v = np.array([g.vx, g.vy, g.vz])
        ref = np.zeros((g.nv, g.nu))
        for iv in range(g.nv):
            for iu in range(g.nu):
                acc = 0.0
                for iz in range(g.nz):
                    for iy in range(g.ny):
                        for ix in range(g.nx):
                            vlo = lo + np.array([ix, iy, iz]) * v
                            acc += box_chord(vlo, vlo + v, so, eo[iv, iu]) * vol[iz, iy, ix]
                ref[iv, iu] = acc
        assert np.abs(p - ref).max() < 1e-11


def test_adjointness_with_the_explicit_transpose():
    g = aniso_geom(nx=10, ny=8, nz=6, nu=9, nv=7)
    rng = np.random.default_rng(4)
    x = rng.standard_normal(g.vol_shape)
    y = rng.standard_normal((3, g.nv, g.nu))
    angles, poses = [0.3, 1.9, 4.0], [[1, -1, 0.5, 0.1, -0.2, 0.3], [0] * 6, [-2, 0.5, 1, -0.15, 0.1, -0.4]]
    lhs = float((oracle.forward_siddon(g, angles, poses, x) * y).sum())
    rhs = float((x * oracle.forward_siddon_T(g, angles, poses, y)).sum())
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)


def test_closed_form_ellipsoids_config1_and_convergence():
    """Config 1's phantom against the exact ellipsoid line integrals; halving the voxels must shrink the error."""
    errs = []
    for scale in (1.0, 2.0):
        w = W.make_config(1, scale=scale)
        g = w.geom
        p = oracle.forward_siddon(g, w.angles.numpy(), w.poses.numpy(), w.volume().numpy())[0]
        cf = w.closed_form(w.poses)[0].numpy()
        errs.append(rel_l2(p, cf))
        assert abs(p.sum() / cf.sum() - 1) < 5e-3
    assert errs[0] < 3e-2 and errs[1] < errs[0] / 1.5, errs


def test_closed_form_gaussian_blobs_general_pose():
    bl = blobs(seed=5, n=3, half=9.0, sig=(2.5, 4.0))
    errs = []
    for k in (1, 2):
        g = aniso_geom(nx=22 * k, ny=18 * k, nz=14 * k, vx=1.1 / k, vy=1.4 / k, vz=1.9 / k)
        vol = W.voxelise_blobs(g, bl).double().numpy()
        beta, pose = 2.1, [1.5, -2.0, 1.0, 0.2, -0.15, 0.3]
        p = oracle.forward_siddon(g, [beta], [pose], vol)[0]
        errs.append(rel_l2(p, W.blob_projection(g, bl, beta, pose).numpy()))
    assert errs[0] < 4e-2 and errs[1] < 1.2e-2 and errs[0] / errs[1] > 2.5, errs


def test_missed_and_empty_volumes_give_exact_zeros():
    g = small_geom(n=8, nu=6, nv=5)
    assert np.all(oracle.forward_siddon(g, [0.2], [[0, 0, 500.0, 0, 0, 0]], np.ones(g.vol_shape)) == 0)
    assert np.all(oracle.forward_siddon(g, [0.2], [[1, 2, 3, 0.1, 0.2, 0.3]], np.zeros(g.vol_shape)) == 0)
    up = np.ones((1,) + g.det_shape, np.float32)
    assert np.all(oracle.forward_pose_grad_siddon(g, [0.2], [[0, 0, 500.0, 0, 0, 0]], np.ones(g.vol_shape), up) == 0)


# ---------------------------------------------------------------- pose gradient (Eq.19-20 :179-191)
def stored_G_gradient(g, beta, pose, vol, up):
    """The paper's algorithm as printed (:189-191): build the 12 volumes G_f^j = [ (R r'_j) g_j^T | -R g_j ] with
    numpy (central differences of the zero-extended voxel values, lever arm at the voxel centre), project EACH with
    the (separately pinned) Siddon projector, weight by the upstream gradient, contract with dM/dtheta."""
    R, dR = oracle.rotation(pose)
    pad = np.pad(vol, 1)
    gx = (pad[1:-1, 1:-1, 2:] - pad[1:-1, 1:-1, :-2]) / (2 * g.vx)
    gy = (pad[1:-1, 2:, 1:-1] - pad[1:-1, :-2, 1:-1]) / (2 * g.vy)
    gz = (pad[2:, 1:-1, 1:-1] - pad[:-2, 1:-1, 1:-1]) / (2 * g.vz)
    gj = np.stack([gx, gy, gz])                                                  # [3, nz, ny, nx]
    iz, iy, ix = np.meshgrid(np.arange(g.nz), np.arange(g.ny), np.arange(g.nx), indexing="ij")
    rj = np.stack([g.cx + (ix - (g.nx - 1) / 2) * g.vx, g.cy + (iy - (g.ny - 1) / 2) * g.vy,
                   g.cz + (iz - (g.nz - 1) / 2) * g.vz])
    lever = np.einsum("ab,bzyx->azyx", R, rj)
    Rg = np.einsum("ab,bzyx->azyx", R, gj)
    GM = np.zeros((3, 4))
    for a in range(3):
        for b in range(3):
            GM[a, b] = float((oracle.forward_siddon(g, [beta], [pose], lever[a] * gj[b])[0] * up).sum())
        GM[a, 3] = float((oracle.forward_siddon(g, [beta], [pose], -Rg[a])[0] * up).sum())
    out = np.zeros(6)
    out[:3] = GM[:, 3]
    for k in range(3):
        out[3 + k] = float((dR[k] * GM[:, :3]).sum())
    return out


def test_gradient_equals_the_projection_of_stored_G_volumes():
    g = aniso_geom(nx=12, ny=10, nz=8, nu=9, nv=7)
    rng = np.random.default_rng(6)
    vol = rng.standard_normal(g.vol_shape)
    up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)     # the oracle takes fp32 upstream
    for beta, pose in ((0.7, [1.0, -0.5, 0.8, 0.15, -0.1, 0.25]), (2.6, [0, 0, 0, 0, 0, 0])):
        ref = stored_G_gradient(g, beta, pose, vol, up)
        for route in (oracle.ROUTE_SIX, oracle.ROUTE_TWELVE):
            got = oracle.forward_pose_grad_siddon(g, [beta], [pose], vol, up[None].astype(np.float32), route=route)[0]
            assert np.abs(got - ref).max() <= 1e-10 * np.abs(ref).max(), (route, got, ref)


def test_translation_gradient_is_minus_R_times_the_projection_of_the_difference_volumes():
    """dL/dt = -R <w, A[grad mu]> with A the Siddon projector applied to the stored central-difference volumes."""
    g = small_geom(n=10, nu=8, nv=7)
    rng = np.random.default_rng(7)
    vol = rng.standard_normal(g.vol_shape)
    up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
    beta, pose = 1.1, [0.5, 0.7, -0.3, 0.2, -0.25, 0.1]
    pad = np.pad(vol, 1)
    dvol = [(pad[1:-1, 1:-1, 2:] - pad[1:-1, 1:-1, :-2]) / (2 * g.vx), (pad[1:-1, 2:, 1:-1] - pad[1:-1, :-2, 1:-1]) / (2 * g.vy),
            (pad[2:, 1:-1, 1:-1] - pad[:-2, 1:-1, 1:-1]) / (2 * g.vz)]
    SA = np.array([float((oracle.forward_siddon(g, [beta], [pose], d)[0] * up).sum()) for d in dvol])
    R, _ = oracle.rotation(pose)
    got = oracle.forward_pose_grad_siddon(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
    assert np.abs(got[:3] + R @ SA).max() <= 1e-11 * np.abs(SA).max()


def test_gradient_vs_finite_differences_of_the_continuous_projection():
    """The paper's accuracy metric (Eq.24 :219-222): cosine similarity with central finite differences - here of the
    CLOSED-FORM blob projections, i.e. the continuous truth the discretised gradient approximates."""
    bl = blobs(seed=8, n=3, half=8.0, sig=(2.5, 4.0))
    g = small_geom(n=40, voxel=0.75, nu=24, nv=20, pix=2.0)
    vol = W.voxelise_blobs(g, bl).double().numpy()
    rng = np.random.default_rng(9)
    sims = []
    for trial in range(3):
        beta = float(rng.uniform(0, 2 * math.pi))
        pose = np.concatenate([rng.uniform(-3, 3, 3), rng.uniform(-0.15, 0.15, 3)])
        up = rng.standard_normal(g.det_shape).astype(np.float32).astype(np.float64)
        ana = oracle.forward_pose_grad_siddon(g, [beta], [pose], vol, up[None].astype(np.float32))[0]
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


def test_gradient_is_linear_in_the_upstream_and_in_the_volume():
    g = small_geom(n=8, nu=6, nv=5)
    rng = np.random.default_rng(10)
    v1, v2 = rng.standard_normal(g.vol_shape), rng.standard_normal(g.vol_shape)
    u1 = rng.standard_normal((1,) + g.det_shape).astype(np.float32)
    u2 = rng.standard_normal((1,) + g.det_shape).astype(np.float32)
    a, p = [0.9], [[0.3, -0.2, 0.5, 0.1, 0.2, -0.1]]
    f = lambda v, u: oracle.forward_pose_grad_siddon(g, a, p, v, u)[0]
    assert np.allclose(f(v1, u1 + u2), f(v1, u1) + f(v1, u2), rtol=0, atol=1e-6 * np.abs(f(v1, u1)).max())
    assert np.allclose(f(v1 + 2 * v2, u1), f(v1, u1) + 2 * f(v2, u1), rtol=0, atol=1e-11 * np.abs(f(v1, u1)).max())
