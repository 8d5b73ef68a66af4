"""GPU-vs-oracle parity with explicit per-view frames (`DFP_FLAG_VIEW_FRAMES`, include/dfp.h; oracle O14) - `-m gpu`.

The frame arrays are rounded to fp32 first and the SAME values go to the oracle.  Tolerances as in
test_gpu_parity.py: relative L2 <= 1e-5 on values, <= 1e-3 (U9) on every pose-gradient component.
"""
import math

import numpy as np
import pytest
import torch

import oracle
import workloads as W
from helpers import check_values, aniso_geom, grad_err_u9, rel_l2, small_geom
from test_gpu_parity import POSES3, check_back, check_forward, f32, run_back_case, run_forward_case
from test_oracle_view_frames import _general_frame

pytestmark = pytest.mark.gpu
VF = W.FLAG_VIEW_FRAMES


@pytest.fixture(scope="module")
def dfp():
    import paper_2508_13304_b200 as m
    return m


def _frames3(g):
    return f32(np.stack([_general_frame(g, beta=0.4), _general_frame(g, beta=1.9, skew=False),
                         W.circular_frame(g, 4.1).numpy()]))


def test_general_frames_ragged_anisotropic_gather_paths(dfp):
    """Tilted / skewed / shifted detectors, source off the orbit, odd grid sizes (gather kernels)."""
    g = aniso_geom(flags=VF)
    F = _frames3(g)
    rng = np.random.default_rng(1)
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    check_forward(run_forward_case(dfp, g, F, POSES3, vol, up))
    assert dfp.last_path() == dfp.PATH_GATHER
    proj = rng.random((3,) + g.det_shape).astype(np.float32)
    upv = rng.standard_normal(g.vol_shape).astype(np.float32)
    for bw, fl in ((0, 0), (1, 0), (1, 1)):
        check_back(run_back_case(dfp, g.replace(bp_weight=bw, flags=VF | fl), F, POSES3, proj, upv))


def test_general_frames_tma_paths_and_other_modes(dfp):
    """Grid / detector sizes the TMA-staged kernels take; Siddon, Joseph and fused modes."""
    g = small_geom(n=48, voxel=0.8, nu=72, nv=56, pix=1.1, sad=300.0, sdd=460.0, flags=VF)
    F = _frames3(g)
    rng = np.random.default_rng(2)
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    res = run_forward_case(dfp, g, F, POSES3, vol, up)
    assert dfp.last_path() == dfp.PATH_TMA
    check_forward(res)
    res_g = run_forward_case(dfp, g.replace(flags=VF | dfp.FLAG_NO_TMA), F, POSES3, vol, up)
    assert dfp.last_path() == dfp.PATH_GATHER
    assert rel_l2(res[0], res_g[0]) <= 2e-6                        # same arithmetic per sample, positions re-based elsewhere
    # band-limited projections (line integrals are smooth at the pixel scale): with white-noise pixels the central
    # differences are noise too, and a cancelling component then measures the fp32 resolution of (u, v) - 2e-6 pixel -
    # rather than the kernel (conditioning)
    iv_, iu_ = np.meshgrid(np.arange(g.nv), np.arange(g.nu), indexing="ij")
    proj = np.stack([np.sin(0.21 * iu_ + 0.13 * iv_ + k) + 0.5 * np.cos(0.07 * iu_ - 0.19 * iv_ + 2 * k)
                     for k in range(3)]).astype(np.float32)
    upv = rng.standard_normal(g.vol_shape).astype(np.float32)
    for bw, fl in ((0, 0), (1, 1)):
        res = run_back_case(dfp, g.replace(bp_weight=bw, flags=VF | fl), F, POSES3, proj, upv)
        assert dfp.last_path() == dfp.PATH_TMA
        check_back(res)
    dev = torch.device("cuda:0")
    a, p = F, f32(POSES3)
    vol_d, up_d = torch.as_tensor(vol, device=dev), torch.as_tensor(up, device=dev)
    for flag, fo, go in ((dfp.FLAG_SIDDON, oracle.forward_siddon, oracle.forward_pose_grad_siddon),
                         (dfp.FLAG_JOSEPH, oracle.forward_joseph, oracle.forward_pose_grad_joseph)):
        gm = g.replace(flags=VF | flag)
        assert rel_l2(dfp.forward(gm, a, p, vol_d).cpu().numpy(), fo(g, a, p, vol)) <= 1e-5
        e = grad_err_u9(dfp.forward_pose_grad(gm, a, p, vol_d, up_d).cpu().numpy(), go(g, a, p, vol, up))
        assert e.max() <= 1e-3, e
    proj_f, mom = dfp.forward_fused_moments(g, a, p, vol_d, up_d)
    o_proj = oracle.forward(g, a, p, vol)
    assert rel_l2(proj_f.cpu().numpy(), o_proj) <= 1e-5
    for j, wgt in enumerate((np.ones_like(up), o_proj.astype(np.float32), up)):
        e = grad_err_u9(mom[:, j].cpu().numpy(), oracle.forward_pose_grad(g, a, p, vol, wgt))
        assert e.max() <= 1e-3, (j, e)
    assert dfp.count_ray_steps(g, a, p) > 0


@pytest.mark.parametrize("index,scale,views", [(2, 0.25, 4), (4, 0.125, 6), (5, 0.125, 4)])
def test_noncircular_orbit_forward_configs_reduced(dfp, index, scale, views):
    """The registration / calibration / sweep workloads on a seeded saddle orbit with detector wobble."""
    w = W.make_config(index, scale=scale, n_views=views)
    g = w.geom.replace(flags=w.geom.flags | VF)
    F = f32(W.noncircular_orbit(w.geom, w.angles, w.seed + 17).numpy())
    check_forward(run_forward_case(dfp, g, F, w.poses.numpy(), w.volume("cpu").numpy(), w.fwd_upstream("cpu").numpy()))


def test_noncircular_orbit_exact_interpolant_gradient_mode(dfp):
    """DFP_FLAG_GRAD_INTERP on the saddle orbit; workload and bounds of test_grad_interp_mode_forward / _backproject."""
    dev = torch.device("cuda:0")
    w = W.make_config(2, scale=0.25, n_views=4)
    F = f32(W.noncircular_orbit(w.geom, w.angles, w.seed + 17).numpy())
    p = f32(w.poses.numpy())
    vol, up = w.volume(dev), w.fwd_upstream(dev)
    o = oracle.forward_pose_grad(w.geom.replace(flags=VF), F, p, vol.cpu().numpy(), up.cpu().numpy(),
                                 grad_mode=oracle.GRAD_INTERP)
    e = grad_err_u9(dfp.forward_pose_grad(w.geom.replace(flags=VF | dfp.FLAG_GRAD_INTERP), F, p, vol, up).cpu().numpy(), o)
    assert e.max() <= 1e-3, e
    w = W.make_config(3, scale=0.25, n_views=6)
    F = f32(W.noncircular_orbit(w.geom, w.angles, w.seed + 17).numpy())
    p = f32(w.poses.numpy())
    proj, upv = w.projections(dev), w.bp_upstream(dev)
    o = oracle.backproject_pose_grad(w.geom.replace(flags=VF), F, p, proj.cpu().numpy(), upv.cpu().numpy(),
                                     grad_mode=oracle.GRAD_INTERP)
    e = grad_err_u9(dfp.backproject_pose_grad(w.geom.replace(flags=VF | dfp.FLAG_GRAD_INTERP), F, p, proj, upv).cpu().numpy(), o)
    assert e.max() <= 1e-3, e


@pytest.mark.parametrize("index,scale,views", [(3, 0.25, 12), (5, 0.125, 6)])
def test_noncircular_orbit_back_configs_reduced(dfp, index, scale, views):
    w = W.make_config(index, scale=scale, n_views=views)
    g = w.geom.replace(flags=w.geom.flags | VF)
    F = f32(W.noncircular_orbit(w.geom, w.angles, w.seed + 17).numpy())
    check_back(run_back_case(dfp, g, F, w.poses.numpy(), w.projections("cpu").numpy(), w.bp_upstream("cpu").numpy()))


def test_circular_frames_agree_with_gantry_angles(dfp):
    """The frame of a circular view (rounded to fp32: the geometry moves by ~1e-5 mm) gives the angle-mode result."""
    w = W.make_config(2, scale=0.25, n_views=3)
    dev = torch.device("cuda:0")
    a, p = w.angles.float().numpy(), w.poses.float().numpy()
    F = f32(np.stack([W.circular_frame(w.geom, float(b)).numpy() for b in a]))
    vol, up = w.volume(dev), w.fwd_upstream(dev)
    gf = w.geom.replace(flags=VF)
    assert rel_l2(dfp.forward(gf, F, p, vol).cpu().numpy(), dfp.forward(w.geom, a, p, vol).cpu().numpy()) < 2e-6
    e = grad_err_u9(dfp.forward_pose_grad(gf, F, p, vol, up).cpu().numpy(),
                    dfp.forward_pose_grad(w.geom, a, p, vol, up).cpu().numpy())
    assert e.max() < 1e-3


def test_host_calls_slice_the_frame_array_by_views(dfp):
    """The host-buffer calls chunk their views: chunk c must read frames [12 v0, ...), not [v0, ...)."""
    w = W.make_config(5, scale=0.125, n_views=12)
    g = w.geom.replace(flags=VF)
    F = f32(W.noncircular_orbit(w.geom, w.angles, w.seed + 17).numpy())
    p = w.poses.float().numpy()
    dev = torch.device("cuda:0")
    vol = w.volume(dev)
    ref = dfp.forward(g, F, p, vol).cpu()
    got = dfp.forward_host(g, F, p, vol.cpu())
    assert torch.equal(got, ref)
    up = w.bp_upstream(dev)
    refg = dfp.backproject_pose_grad(g, F, p, ref.to(dev), up).cpu()
    gotg = dfp.backproject_pose_grad_host(g, F, p, ref, up.cpu())
    assert torch.allclose(gotg, refg, rtol=1e-5, atol=1e-6 * float(refg.abs().max()))
    refv = dfp.backproject(g, F, p, ref.to(dev)).cpu()
    gotv = dfp.backproject_host(g, F, p, ref)
    assert rel_l2(gotv.numpy(), refv.numpy()) < 1e-6


def test_degenerate_frames_are_rejected(dfp):
    g = small_geom(flags=VF)
    F = np.array([[120, 0, 0, -80, 0, 0, 0, 2.5, 0, 0, 0, 2.5]], np.float32)       # exactly representable numbers
    assert torch.isfinite(dfp.forward(g, F, [[0.0] * 6], torch.ones(g.vol_shape, device="cuda:0"))).all()
    dev = torch.device("cuda:0")
    vol = torch.zeros(g.vol_shape, device=dev)
    bad = F.copy()
    bad[0, 9:12] = 2.0 * bad[0, 6:9]                                 # V parallel to U
    with pytest.raises(dfp.DfpError) as e:
        dfp.forward(g, bad, [[0.0] * 6], vol)
    assert e.value.status == -2
    bad = F.copy()
    bad[0, 0:3] = [-80, 7.5, -5]                                     # source in the detector plane
    with pytest.raises(dfp.DfpError) as e:
        dfp.forward(g, bad, [[0.0] * 6], vol)
    assert e.value.status == -2


def test_c4_calibration_full_size_noncircular_orbit(dfp):
    """Full-size calibration workload (512^3, 768^2 detector) on the saddle orbit: 16 of its views through the
    kernels bench.py times; the oracle recomputes a band of rows of two views and one full 6-vector."""
    from test_gpu_full_size import pick, row_band
    dev = torch.device("cuda:0")
    w = W.make_config(4)
    sel = pick(w.seed + 911, w.n_views, 16)
    g = w.geom.replace(flags=VF)
    F = f32(W.noncircular_orbit(w.geom, w.angles, w.seed + 17).numpy())[sel]
    p = w.poses.float().numpy()[sel]
    vol = w.volume(dev)
    up = w.fwd_upstream(dev, views=sel)
    proj = dfp.forward(g, F, p, vol)
    assert dfp.last_path() == dfp.PATH_TMA
    grad = dfp.forward_pose_grad(g, F, p, vol, up).cpu().numpy()
    assert dfp.last_path() == dfp.PATH_TMA
    assert torch.isfinite(proj).all() and np.isfinite(grad).all()
    vol_c = vol.cpu().numpy()
    for v in (3, 11):
        r0 = pick(w.seed + 5 + v, g.nv - 32 + 1, 1)[0]
        o = oracle.forward(row_band(g, r0, 32), F[v:v + 1], p[v:v + 1], vol_c)[0]
        assert np.linalg.norm(o) > 0 and rel_l2(proj[v, r0:r0 + 32].cpu().numpy(), o) <= 1e-5
    o = oracle.forward_pose_grad(g, F[3:4], p[3:4], vol_c, up[3:4].cpu().numpy())
    assert grad_err_u9(grad[3:4], o).max() <= 1e-3


def _random_frame(rng, g, wild):
    """A circular view, then: the whole scanner turned about a random axis (up to 30 degrees), the detector tilted about
    its own u and v axes (up to 20 degrees), spun about its normal (any angle), sheared and rescaled, shifted by up to
    20 pixels, the source moved by up to 30 mm (wild); or a quarter of those amplitudes (a calibrated C-arm)."""
    q = 1.0 if wild else 0.25
    def rot(axis, ang):
        k = np.asarray(axis, dtype=np.float64)
        k = k / np.linalg.norm(k)
        K = np.array([[0, -k[2], k[1]], [k[2], 0, -k[0]], [-k[1], k[0], 0]])
        return np.eye(3) + math.sin(ang) * K + (1 - math.cos(ang)) * (K @ K)
    f = W.circular_frame(g, rng.uniform(0, 2 * math.pi)).numpy().reshape(4, 3)
    Q = rot(rng.standard_normal(3), rng.uniform(-0.5, 0.5))
    s, c, U, V = Q @ f[0], Q @ f[1], Q @ f[2], Q @ f[3]
    T = rot(U, q * rng.uniform(-0.35, 0.35)) @ rot(V, q * rng.uniform(-0.35, 0.35)) @ \
        rot(np.cross(U, V), (math.pi if wild else 0.1) * rng.uniform(-1, 1))
    U, V = T @ U, T @ V
    U, V = (1 + q * rng.uniform(-0.2, 0.2)) * U + q * rng.uniform(-0.2, 0.2) * V, (1 + q * rng.uniform(-0.2, 0.2)) * V
    c = c + q * rng.uniform(-20, 20) * U + q * rng.uniform(-20, 20) * V
    s = s + q * rng.uniform(-30, 30, 3)
    return np.concatenate([s, c, U, V])


def test_random_frames_both_paths_agree_and_never_nan(dfp):
    """30 seeded random scanners with arbitrary view frames.  Whatever path the host picks from the frame, the result
    must be finite (NaN = a staged box / patch did not hold its tile: host bound wrong) and agree with the gather
    path; every third case is also checked against the oracle at the 1e-5 / 1e-3 of BASELINE.json (white-noise volume and
    upstream: the worst case for cancellation)."""

    def check_grad(got, ref, case):
        e = grad_err_u9(got, ref)
        assert np.all(np.isfinite(got)) and e.max() <= 1e-3, (case, e)

    rng = np.random.default_rng(1330464)
    dev = torch.device("cuda:0")
    n_tma = 0
    for case in range(30):
        nx, ny, nz = (int(4 * rng.integers(5, 15)) for _ in range(3))
        nu, nv = int(4 * rng.integers(6, 30)), int(rng.integers(9, 70))
        vox = rng.uniform(0.6, 1.6, 3)
        sad = rng.uniform(250.0, 900.0)
        sdd = sad * rng.uniform(1.3, 2.0)
        du, dv = (vox.mean() * sdd / sad * rng.uniform(0.3, 1.5) for _ in range(2))
        g = W.Geometry(nx=nx, ny=ny, nz=nz, vx=vox[0], vy=vox[1], vz=vox[2], nu=nu, nv=nv, du=du, dv=dv, sad=sad,
                       sdd=sdd, cx=rng.uniform(-3, 3), cy=rng.uniform(-3, 3), cz=rng.uniform(-3, 3),
                       u0=rng.uniform(-2, 2), v0=rng.uniform(-2, 2), bp_weight=int((case // 2) % 2), flags=VF).f32()
        V = int(rng.integers(1, 6))
        F = f32(np.stack([_random_frame(rng, g, wild=case % 2 == 1) for _ in range(V)]))
        poses = f32(np.concatenate([rng.uniform(-8, 8, (V, 3)), rng.uniform(-0.35, 0.35, (V, 3))], axis=1))
        vol = torch.as_tensor(rng.random(g.vol_shape).astype(np.float32), device=dev)
        up = torch.as_tensor(rng.standard_normal((V,) + g.det_shape).astype(np.float32), device=dev)
        bup = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
        iv_, iu_ = np.meshgrid(np.arange(g.nv), np.arange(g.nu), indexing="ij")
        pin_np = np.stack([np.sin(0.21 * iu_ + 0.13 * iv_ + k) + 0.5 * np.cos(0.07 * iu_ - 0.19 * iv_ + 2 * k)
                           for k in range(V)]).astype(np.float32)
        pin = torch.as_tensor(pin_np, device=dev)
        gn = g.replace(flags=VF | dfp.FLAG_NO_TMA)
        proj = dfp.forward(g, F, poses, vol)
        n_tma += dfp.last_path()
        grad = dfp.forward_pose_grad(g, F, poses, vol, up)
        n_tma += dfp.last_path()
        bp = dfp.backproject(g, F, poses, pin)
        n_tma += dfp.last_path()
        bgrad = dfp.backproject_pose_grad(g, F, poses, pin, bup)
        n_tma += dfp.last_path()
        for t in (proj, grad, bp, bgrad):
            assert torch.isfinite(t).all(), (case, g)
        assert rel_l2(proj.cpu().numpy(), dfp.forward(gn, F, poses, vol).cpu().numpy()) <= 2e-6, case
        assert grad_err_u9(grad.cpu().numpy(),
                           dfp.forward_pose_grad(gn, F, poses, vol, up).cpu().numpy()).max() <= 2e-3, case      # each path within 1e-3 of the truth
        assert rel_l2(bp.cpu().numpy(), dfp.backproject(gn, F, poses, pin).cpu().numpy()) <= 1e-5, case
        assert grad_err_u9(bgrad.cpu().numpy(),
                           dfp.backproject_pose_grad(gn, F, poses, pin, bup).cpu().numpy()).max() <= 2e-3, case   # each path within 1e-3 of the truth
        if case % 3 == 0:
            o_proj, o_bp = oracle.forward(g, F, poses, vol.cpu().numpy()), oracle.backproject(g, F, poses, pin_np)
            check_values(proj.cpu().numpy(), o_proj, 1e-5, zero_border=False)    # all-zero oracle => all-zero result
            check_values(bp.cpu().numpy(), o_bp, 1e-5, zero_border=False)
            check_grad(grad.cpu().numpy(), oracle.forward_pose_grad(g, F, poses, vol.cpu().numpy(), up.cpu().numpy()), case)
            check_grad(bgrad.cpu().numpy(), oracle.backproject_pose_grad(g, F, poses, pin_np, bup.cpu().numpy()), case)
    print("TMA calls", n_tma)
    assert 30 <= n_tma <= 115, n_tma      # a mix of TMA and fallback calls (4 calls per case)
