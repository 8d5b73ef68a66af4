"""GPU-vs-oracle parity through the C ABI (`-m gpu`).  Same seeded inputs, element by element.

Tolerances (BASELINE.json north_star): relative L2 <= 1e-5 on projections and
back-projections, <= 1e-3 on every pose-gradient component with the floored denominator of reading U9.
Angles and poses are rounded to fp32 first (the C ABI takes fp32) and the SAME values go to the oracle.
"""
import math

import numpy as np
import pytest
import torch

import oracle
import workloads as W
from helpers import aniso_geom, check_values, grad_err_u9, rel_l2, small_geom

pytestmark = pytest.mark.gpu

TOL_VAL = 1e-5
TOL_GRAD = 1e-3


@pytest.fixture(scope="module")
def dfp():
    import paper_2508_13304_b200 as m
    return m


def f32(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32)


def run_forward_case(dfp, g, angles, poses, vol, up):
    dev = torch.device("cuda:0")
    angles, poses = f32(angles), f32(poses).reshape(-1, 6)
    vol_d = torch.as_tensor(vol, dtype=torch.float32, device=dev).contiguous()
    up_d = torch.as_tensor(up, dtype=torch.float32, device=dev).contiguous()
    proj = dfp.forward(g, angles, poses, vol_d).cpu().numpy()
    grad = dfp.forward_pose_grad(g, angles, poses, vol_d, up_d).cpu().numpy()
    o_proj = oracle.forward(g, angles, poses, vol_d.cpu().numpy())
    o_grad = oracle.forward_pose_grad(g, angles, poses, vol_d.cpu().numpy(), up_d.cpu().numpy())
    return proj, grad, o_proj, o_grad


def run_back_case(dfp, g, angles, poses, proj, up):
    dev = torch.device("cuda:0")
    angles, poses = f32(angles), f32(poses).reshape(-1, 6)
    proj_d = torch.as_tensor(proj, dtype=torch.float32, device=dev).contiguous()
    up_d = torch.as_tensor(up, dtype=torch.float32, device=dev).contiguous()
    vol = dfp.backproject(g, angles, poses, proj_d).cpu().numpy()
    grad = dfp.backproject_pose_grad(g, angles, poses, proj_d, up_d).cpu().numpy()
    o_vol = oracle.backproject(g, angles, poses, proj_d.cpu().numpy())
    o_grad = oracle.backproject_pose_grad(g, angles, poses, proj_d.cpu().numpy(), up_d.cpu().numpy())
    return vol, grad, o_vol, o_grad


def check_forward(res, zero_border=False):
    proj, grad, o_proj, o_grad = res
    assert np.all(np.isfinite(proj)) and np.all(np.isfinite(grad))
    check_values(proj, o_proj, TOL_VAL, zero_border=zero_border)
    e = grad_err_u9(grad, o_grad)
    assert e.max() <= TOL_GRAD, e


def check_back(res, zero_border=False):
    vol, grad, o_vol, o_grad = res
    assert np.all(np.isfinite(vol)) and np.all(np.isfinite(grad))
    check_values(vol, o_vol, TOL_VAL, zero_border=zero_border)
    e = grad_err_u9(grad, o_grad)
    assert e.max() <= TOL_GRAD, e


POSES3 = [[1.2, -0.8, 0.6, 0.11, -0.07, 0.19], [0, 0, 0, 0, 0, 0], [-3.0, 2.0, 1.5, -0.2, 0.15, -0.4]]
ANGLES3 = [0.4, math.pi / 2, 4.1]


# ------------------------------------------------------------------ ragged small cases (several tiles + tails)
def test_forward_ragged_anisotropic(dfp):
    g = aniso_geom(nx=37, ny=29, nz=23, nu=45, nv=21)
    rng = np.random.default_rng(0)
    vol = rng.standard_normal(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    check_forward(run_forward_case(dfp, g, ANGLES3, POSES3, vol, up))


def test_forward_odd_and_even_grids_and_fine_step(dfp):
    for n, step in ((16, 0.0), (17, 0.0), (21, 0.4)):
        g = small_geom(n=n, nu=33, nv=9, step_mm=step)
        rng = np.random.default_rng(n)
        vol = rng.random(g.vol_shape).astype(np.float32)
        up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
        check_forward(run_forward_case(dfp, g, ANGLES3, POSES3, vol, up))


def test_back_ragged_anisotropic(dfp):
    for bw, fl in ((0, 0), (1, 0), (1, 1)):
        g = aniso_geom(nx=37, ny=29, nz=23, nu=45, nv=21, bp_weight=bw, flags=fl)
        rng = np.random.default_rng(1)
        proj = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
        up = rng.standard_normal(g.vol_shape).astype(np.float32)
        check_back(run_back_case(dfp, g, ANGLES3, POSES3, proj, up))


def test_back_volume_larger_than_field_of_view(dfp):
    """Voxels that project outside the detector (zero extension of b~) and a tall z range (several z chunks)."""
    g = small_geom(n=40, voxel=3.0, nu=20, nv=12, pix=2.0)
    g = g.replace(nz=70)
    rng = np.random.default_rng(2)
    proj = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    up = rng.standard_normal(g.vol_shape).astype(np.float32)
    res = run_back_case(dfp, g, ANGLES3, POSES3, proj, up)
    check_back(res)
    assert (res[2] == 0).mean() > 0.2 and np.array_equal(res[0] == 0, res[2] == 0)


# ------------------------------------------------------------------ degenerate cases
def test_missed_and_empty_inputs_give_exact_zeros(dfp):
    g = small_geom(n=12, nu=10, nv=7)
    vol = np.ones(g.vol_shape, np.float32)
    up = np.ones((1,) + g.det_shape, np.float32)
    far = [[0, 0, 700.0, 0, 0, 0]]
    proj, grad, _, _ = run_forward_case(dfp, g, [0.3], far, vol, up)
    assert np.all(proj == 0) and np.all(grad == 0)
    proj, grad, _, _ = run_forward_case(dfp, g, [0.3], [POSES3[0]], 0 * vol, up)
    assert np.all(proj == 0) and np.all(grad == 0)
    pr = np.ones((1,) + g.det_shape, np.float32)
    uv = np.ones(g.vol_shape, np.float32)
    bvol, bgrad, _, _ = run_back_case(dfp, g, [0.3], far, pr, uv)
    assert np.all(bvol == 0) and np.all(bgrad == 0)


def test_single_voxel_and_single_pixel(dfp):
    g = small_geom(n=1, voxel=4.0, nu=1, nv=1, pix=3.0)
    vol = np.full(g.vol_shape, 0.7, np.float32)
    up = np.ones((1,) + g.det_shape, np.float32)
    check_forward(run_forward_case(dfp, g, [0.0], [[0.3, 0.2, -0.1, 0.01, 0.02, 0.03]], vol, up))
    check_back(run_back_case(dfp, g, [0.0], [[0.3, 0.2, -0.1, 0.01, 0.02, 0.03]], np.ones((1, 1, 1), np.float32),
                             np.ones(g.vol_shape, np.float32)))


def test_host_buffer_entry_points_match_device_ones(dfp):
    g = aniso_geom()
    rng = np.random.default_rng(3)
    vol = rng.standard_normal(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    a, p = f32(ANGLES3), f32(POSES3)
    dev = torch.device("cuda:0")
    vd, ud = torch.as_tensor(vol, device=dev), torch.as_tensor(up, device=dev)
    proj = dfp.forward(g, a, p, vd)
    assert torch.equal(dfp.forward_host(g, a, p, vol), proj.cpu())
    assert torch.equal(dfp.forward_pose_grad_host(g, a, p, vol, up), dfp.forward_pose_grad(g, a, p, vd, ud).cpu())
    pj = proj.cpu().numpy()
    wv = rng.standard_normal(g.vol_shape).astype(np.float32)
    assert torch.equal(dfp.backproject_host(g, a, p, pj), dfp.backproject(g, a, p, proj).cpu())
    assert torch.equal(dfp.backproject_pose_grad_host(g, a, p, pj, wv),
                       dfp.backproject_pose_grad(g, a, p, proj, torch.as_tensor(wv, device=dev)).cpu())


def test_results_are_deterministic(dfp):
    g = aniso_geom(nx=37, ny=29, nz=23, nu=45, nv=21)
    rng = np.random.default_rng(4)
    dev = torch.device("cuda:0")
    vol = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
    up = torch.as_tensor(rng.standard_normal((3,) + g.det_shape).astype(np.float32), device=dev)
    a, p = f32(ANGLES3), f32(POSES3)
    g1 = dfp.forward_pose_grad(g, a, p, vol, up)
    g2 = dfp.forward_pose_grad(g, a, p, vol, up)
    assert torch.equal(g1, g2)
    b1 = dfp.backproject_pose_grad(g, a, p, up, vol)
    b2 = dfp.backproject_pose_grad(g, a, p, up, vol)
    assert torch.equal(b1, b2)


@pytest.mark.parametrize("index,scale,views", [(1, 1.0, None), (2, 0.25, 5), (4, 0.125, 6), (5, 0.125, 6)])
def test_ray_step_count_matches_oracle(dfp, index, scale, views):
    """The metric's unit is defined by the ORACLE's clip - samples inside the 2-voxel-padded box;
    dfp_count_ray_steps counts the same set (both in fp64: they may differ only on samples within rounding of the
    box faces)."""
    w = W.make_config(index, scale=scale, n_views=views)
    a, p = f32(w.angles), f32(w.poses)
    n_gpu = dfp.count_ray_steps(w.geom, a, p)
    _, n_ora = oracle.forward(w.geom, a, p, w.volume().numpy(), return_steps=True)
    assert n_ora > 0 and abs(n_gpu - n_ora) <= max(2, 1e-6 * n_ora), (n_gpu, n_ora)


# ------------------------------------------------------------------ the five configs, reduced so the oracle takes seconds
@pytest.mark.parametrize("index,scale,views", [(1, 1.0, None), (2, 0.25, 3), (4, 0.125, 4), (5, 0.125, 3)])
def test_forward_configs_reduced(dfp, index, scale, views):
    w = W.make_config(index, scale=scale, n_views=views)
    check_forward(run_forward_case(dfp, w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy(),
                                   w.fwd_upstream().numpy()), zero_border=True)


@pytest.mark.parametrize("index,scale,views", [(3, 0.25, 12), (5, 0.125, 6)])
def test_back_configs_reduced(dfp, index, scale, views):
    w = W.make_config(index, scale=scale, n_views=views)
    check_back(run_back_case(dfp, w.geom, w.angles.numpy(), w.poses.numpy(), w.projections().numpy(),
                             w.bp_upstream().numpy()))


# ------------------------------------------------------------------ the two forward kernel paths (gather / TMA-staged)
def _both_paths(dfp, g, angles, poses, vol, up):
    dev = torch.device("cuda:0")
    a, p = f32(angles), f32(poses).reshape(-1, 6)
    vd = torch.as_tensor(vol, dtype=torch.float32, device=dev).contiguous()
    ud = torch.as_tensor(up, dtype=torch.float32, device=dev).contiguous()
    out = {}
    for name, gg in (("tma", g), ("gather", g.replace(flags=g.flags | dfp.FLAG_NO_TMA))):
        proj = dfp.forward(gg, a, p, vd)
        path_f = dfp.last_path()
        grad = dfp.forward_pose_grad(gg, a, p, vd, ud)
        out[name] = (proj.cpu(), grad.cpu(), path_f, dfp.last_path())
    return out


def _same(o):
    """The two forward paths do the same arithmetic per sample on positions re-based at different places (per chunk of
    the block / per 16 samples of the ray) with the fraction taken as q - floor(q) (TMA) or (q' - rint(q')) + 1/2
    (gather), and the TMA gradient kernels split a ray's samples between lanes: the results agree to fp32 rounding
    (measured on these cases: 1e-7 on the projections, <= 3.5e-5 of U9 on a gradient component of a white-noise volume;
    each path is held to the oracle at 1e-5 / 1e-3 by the parity tests)."""
    pt, pg = o["tma"][0].numpy(), o["gather"][0].numpy()
    return (rel_l2(pt, pg) <= 2e-6 and np.array_equal(pt == 0, pg == 0) and
            grad_err_u9(o["tma"][1].numpy(), o["gather"][1].numpy()).max() <= 1e-4)


def test_tma_path_is_taken_and_matches_gather_path(dfp):
    """nx % 4 == 0 and clinical magnification: the TMA-staged kernels run; same arithmetic per sample."""
    w = W.make_config(2, scale=0.25, n_views=3)
    o = _both_paths(dfp, w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy(), w.fwd_upstream().numpy())
    assert o["tma"][2] == dfp.PATH_TMA and o["tma"][3] == dfp.PATH_TMA
    assert o["gather"][2] == dfp.PATH_GATHER and o["gather"][3] == dfp.PATH_GATHER
    assert _same(o)
    w = W.make_config(4, scale=0.125, n_views=5)          # views around the circle: oblique frusta, short chunks
    o = _both_paths(dfp, w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy(), w.fwd_upstream().numpy())
    assert o["tma"][2] == dfp.PATH_TMA and o["tma"][3] == dfp.PATH_TMA
    assert _same(o)


def test_tma_path_ragged_detector_and_partial_misses(dfp):
    """Detector not a multiple of the 16x16 tile, volume partly outside the fan (zero fill by the TMA unit)."""
    g = aniso_geom(nx=40, ny=29, nz=23, nu=45, nv=21, vx=0.9, vy=1.0, vz=1.1, du=0.8, dv=0.7, sad=400.0, sdd=600.0)
    rng = np.random.default_rng(11)
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    o = _both_paths(dfp, g, ANGLES3, POSES3, vol, up)
    assert o["tma"][2] == dfp.PATH_TMA and o["tma"][3] == dfp.PATH_TMA
    assert _same(o)
    check_forward(run_forward_case(dfp, g, ANGLES3, POSES3, vol, up))


def test_tma_path_odd_row_length_and_fallback(dfp):
    """nx % 4 != 0: a tensor map needs 16-byte-aligned rows, so the TMA kernels read a row-padded copy of the volume (1x,
    in the workspace) - same results, TMA path.  Coarse pixels on fine voxels (a tile's frustum exceeds every staging
    box): the gather kernels."""
    rng = np.random.default_rng(12)
    dev = torch.device("cuda:0")
    cases = ((aniso_geom(nx=37, ny=29, nz=23, nu=44, nv=36, du=1.0, dv=1.2), dfp.PATH_TMA),
             (aniso_geom(nx=38, ny=30, nz=22, nu=40, nv=32, du=1.0, dv=1.2), dfp.PATH_TMA),
             (small_geom(n=64, voxel=0.25, nu=20, nv=18, pix=2.4), dfp.PATH_GATHER))
    for g, path in cases:
        vol = rng.random(g.vol_shape).astype(np.float32)
        up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
        o = _both_paths(dfp, g, ANGLES3, POSES3, vol, up)
        assert o["tma"][2] == path and o["tma"][3] == path, (g.nx, o["tma"][2:])
        assert o["gather"][2] == dfp.PATH_GATHER and _same(o)
        check_forward(run_forward_case(dfp, g, ANGLES3, POSES3, vol, up))


# ------------------------------------------------------------------ the two back-projection kernel paths
def _both_bp_paths(dfp, g, angles, poses, proj, up):
    dev = torch.device("cuda:0")
    a, p = f32(angles), f32(poses).reshape(-1, 6)
    pd = torch.as_tensor(proj, dtype=torch.float32, device=dev).contiguous()
    ud = torch.as_tensor(up, dtype=torch.float32, device=dev).contiguous()
    out = {}
    for name, gg in (("tma", g), ("gather", g.replace(flags=g.flags | dfp.FLAG_NO_TMA))):
        vol = dfp.backproject(gg, a, p, pd)
        path_b = dfp.last_path()
        grad = dfp.backproject_pose_grad(gg, a, p, pd, ud)
        out[name] = (vol.cpu().numpy(), grad.cpu().numpy(), path_b, dfp.last_path())
    return out


@pytest.mark.parametrize("bw,fl", [(0, 0), (1, 0), (1, 1)])
def test_bp_tma_path_is_taken_and_agrees_with_gather_path(dfp, bw, fl):
    """nu % 4 == 0, every voxel in front of the source: detector patches staged by TMA.  Same per-voxel formulae;
    the TMA kernels need no clamp of (u, v), so the compiler fuses u'/w' into the floor / fraction FMAs (one rounding
    less), and the per-view partial sums of the gradient are grouped by different voxel tiles: agreement to a few
    1e-6 (ramp-filtered data: sign-cancelling sums), both within 1e-5 of the oracle (the config tests)."""
    w = W.make_config(3, scale=0.25, n_views=12)
    g = w.geom.replace(bp_weight=bw, flags=fl)
    o = _both_bp_paths(dfp, g, w.angles.numpy(), w.poses.numpy(), w.projections().numpy(), w.bp_upstream().numpy())
    assert o["tma"][2] == dfp.PATH_TMA and o["tma"][3] == dfp.PATH_TMA
    assert o["gather"][2] == dfp.PATH_GATHER and o["gather"][3] == dfp.PATH_GATHER
    assert rel_l2(o["tma"][0], o["gather"][0]) <= 1e-5
    assert np.array_equal(o["tma"][0] == 0, o["gather"][0] == 0)
    # the gather kernels keep (u, v) in detector-wide fp32 coordinates (~3e-5 pixel), the TMA kernels in patch-local ones
    assert grad_err_u9(o["tma"][1], o["gather"][1]).max() <= 3e-4


def test_bp_tma_path_ragged_volume_off_detector_voxels_and_many_views(dfp):
    """Volume not a multiple of the 16x16x16 tile, wider than the fan (zero fill by the TMA unit), and more views
    than pipeline stages and reduction groups (17 = 2 groups of 8 + 1)."""
    g = aniso_geom(nx=37, ny=29, nz=23, nu=44, nv=21, vx=2.2, vy=2.0, vz=1.9, du=1.1, dv=1.3, sad=400.0, sdd=600.0)
    rng = np.random.default_rng(21)
    V = 17
    angles = rng.uniform(0, 2 * math.pi, V)
    poses = np.concatenate([rng.uniform(-3, 3, (V, 3)), rng.uniform(-0.15, 0.15, (V, 3))], axis=1)
    proj = rng.standard_normal((V,) + g.det_shape).astype(np.float32)
    up = rng.standard_normal(g.vol_shape).astype(np.float32)
    for bw in (0, 1):
        gg = g.replace(bp_weight=bw)
        o = _both_bp_paths(dfp, gg, angles, poses, proj, up)
        assert o["tma"][2] == dfp.PATH_TMA and o["tma"][3] == dfp.PATH_TMA
        assert rel_l2(o["tma"][0], o["gather"][0]) <= 1e-5
        assert (o["tma"][0] == 0).mean() > 0.05 and np.array_equal(o["tma"][0] == 0, o["gather"][0] == 0)
        assert grad_err_u9(o["tma"][1], o["gather"][1]).max() <= 3e-4
        check_back(run_back_case(dfp, gg, angles, poses, proj, up))


def test_bp_tma_path_odd_row_length_and_fallback(dfp):
    """nu % 4 != 0: the TMA kernels read a row-padded copy of the projections (tensor maps need 16-byte-aligned rows) -
    TMA path, same results.  A magnification so large that a tile's footprint exceeds the patch menu: the gather kernels."""
    rng = np.random.default_rng(22)
    for g, path in ((aniso_geom(nu=21, nv=17), 1), (aniso_geom(nu=22, nv=19), 1),
                    (small_geom(n=24, voxel=4.0, nu=400, nv=40, pix=0.1, sad=300.0, sdd=900.0), 0)):
        # smooth projections: at 120 pixels per voxel, white noise would measure the fp32 resolution of u (|u| <= 200
        # pixels -> 2e-5 pixel) rather than the kernel
        iv, iu = np.meshgrid(np.arange(g.nv), np.arange(g.nu), indexing="ij")
        proj = np.stack([np.sin(0.05 * iu + 0.07 * iv + k) + 0.3 * np.cos(0.11 * iu - 0.02 * iv) for k in range(2)])
        proj = proj.astype(np.float32)
        up = rng.standard_normal(g.vol_shape).astype(np.float32)
        o = _both_bp_paths(dfp, g, ANGLES3[:2], POSES3[:2], proj, up)
        want = dfp.PATH_TMA if path else dfp.PATH_GATHER
        assert o["tma"][2] == want and o["tma"][3] == want, (g.nu, o["tma"][2:])
        assert rel_l2(o["tma"][0], o["gather"][0]) <= 1e-5 and grad_err_u9(o["tma"][1], o["gather"][1]).max() <= 2e-3
        check_back(run_back_case(dfp, g, ANGLES3[:2], POSES3[:2], proj, up))


# ------------------------------------------------------------------ DFP_FLAG_GRAD_INTERP
def test_grad_interp_mode_forward(dfp):
    """Exact derivative of the trilinear interpolant (what autodiff of the discrete projector gives): the oracle's
    GRAD_INTERP mode, itself pinned against finite differences of the discrete projector.  TMA and gather paths."""
    dev = torch.device("cuda:0")
    cases = [W.make_config(2, scale=0.25, n_views=3), W.make_config(4, scale=0.125, n_views=4), W.make_config(1)]
    for w in cases:
        a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
        vol, up = w.volume(dev), w.fwd_upstream(dev)
        o = oracle.forward_pose_grad(w.geom, a, p, vol.cpu().numpy(), up.cpu().numpy(), grad_mode=oracle.GRAD_INTERP)
        o_central = oracle.forward_pose_grad(w.geom, a, p, vol.cpu().numpy(), up.cpu().numpy())
        assert grad_err_u9(o, o_central).max() > 1e-2            # the two modes are different estimators
        for fl in (dfp.FLAG_GRAD_INTERP, dfp.FLAG_GRAD_INTERP | dfp.FLAG_NO_TMA):
            g = dfp.forward_pose_grad(w.geom.replace(flags=fl), a, p, vol, up).cpu().numpy()
            assert np.all(np.isfinite(g))
            e = grad_err_u9(g, o)
            # the integrand is piecewise constant in the sample position: both sides take the cell of a sample in fp64
            # (the kernels re-derive cell and fractions in fp64 for samples within fp32 rounding of a cell face)
            assert e.max() <= TOL_GRAD, (w.name, fl, e)


@pytest.mark.parametrize("bw,fl", [(0, 0), (1, 0), (1, 1)])
def test_grad_interp_mode_backproject(dfp, bw, fl):
    dev = torch.device("cuda:0")
    w = W.make_config(3, scale=0.25, n_views=10)
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    proj, up = w.projections(dev), w.bp_upstream(dev)
    g0 = w.geom.replace(bp_weight=bw, flags=fl)
    o = oracle.backproject_pose_grad(g0, a, p, proj.cpu().numpy(), up.cpu().numpy(), grad_mode=oracle.GRAD_INTERP)
    for extra in (dfp.FLAG_GRAD_INTERP, dfp.FLAG_GRAD_INTERP | dfp.FLAG_NO_TMA):
        g = dfp.backproject_pose_grad(g0.replace(flags=fl | extra), a, p, proj, up).cpu().numpy()
        assert np.all(np.isfinite(g))
        e = grad_err_u9(g, o)
        # the derivative of the bilinear interpolant is piecewise constant in (u, v): a voxel that projects within fp32
        # rounding of a pixel boundary takes its cell from the fp64 rows, as the oracle does
        assert e.max() <= TOL_GRAD, (bw, fl, extra, e)


# ------------------------------------------------------------------ dfp_forward_fused_moments
def _fused_case(dfp, w, flags=0):
    dev = torch.device("cuda:0")
    g = w.geom.replace(flags=flags)
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    vol = w.volume(dev)
    target = w.closed_form(w.data_poses, dev).to(torch.float32).contiguous()      # b: projections at the data poses
    proj, mom = dfp.forward_fused_moments(g, a, p, vol, target)
    path = dfp.last_path()
    vol_c, tgt_c = vol.cpu().numpy(), target.cpu().numpy()
    o_proj = oracle.forward(g, a, p, vol_c)
    ones = np.ones_like(tgt_c)
    o_m = np.stack([oracle.forward_pose_grad(g, a, p, vol_c, ones),
                    oracle.forward_pose_grad(g, a, p, vol_c, o_proj.astype(np.float32)),
                    oracle.forward_pose_grad(g, a, p, vol_c, tgt_c)], axis=1)      # [V,3,6]
    return proj.cpu().numpy(), mom.cpu().numpy(), o_proj, o_m, path, (g, a, p, vol, target)


@pytest.mark.parametrize("index,scale,views,tma", [(2, 0.25, 3, True), (4, 0.125, 4, True), (1, 1.0, None, True),
                                                   (2, 0.25, 2, False)])
def test_fused_moments_match_oracle(dfp, index, scale, views, tma):
    """One traversal = projection + the pose-gradient 6-vectors for upstream 1, l and b; expected values from the
    pinned oracle functions (forward, and forward_pose_grad with those three upstreams).  tma=False: the gather
    fallback, which composes the call from the projection kernel and three gradient passes."""
    w = W.make_config(index, scale=scale, n_views=views)
    proj, mom, o_proj, o_m, path, _ = _fused_case(dfp, w, 0 if tma else dfp.FLAG_NO_TMA)
    assert path == (dfp.PATH_TMA if tma else dfp.PATH_GATHER)
    assert np.all(np.isfinite(proj)) and np.all(np.isfinite(mom))
    assert rel_l2(proj, o_proj) <= TOL_VAL
    for k in range(3):
        e = grad_err_u9(mom[:, k], o_m[:, k])
        assert e.max() <= TOL_GRAD, (index, k, e)


def test_fused_moments_give_the_ssd_and_ncc_gradients(dfp):
    """dL/dtheta from the moments == dfp_forward_pose_grad with the loss's upstream gradient (SSD: 2(l - b); NCC: the
    affine form of workloads.losses.ncc_grad), for both kernel paths."""
    w = W.make_config(2, scale=0.25, n_views=3)
    for flags in (0, dfp.FLAG_NO_TMA):
        proj, mom, _, _, _, (g, a, p, vol, target) = _fused_case(dfp, w, flags)
        l = torch.as_tensor(proj, device=vol.device)
        # SSD: dL/dl = 2 (l - b)
        ref = dfp.forward_pose_grad(g, a, p, vol, (2.0 * (l - target)).contiguous()).cpu().numpy()
        got = 2.0 * (mom[:, 1] - mom[:, 2])
        assert grad_err_u9(got, ref).max() <= 1e-4
        # NCC(l, b) per view: dNCC/dl = (b - mean b)/(sa sb) - NCC (l - mean l)/sa^2, sa = |l - mean l|, sb likewise
        got_n, up_n = [], []
        for v in range(l.shape[0]):
            lv, bv = l[v].double(), target[v].double()
            la, ba = lv - lv.mean(), bv - bv.mean()
            sa, sb = la.norm(), ba.norm()
            ncc = (la * ba).sum() / (sa * sb)
            up_n.append((ba / (sa * sb) - ncc * la / sa ** 2).float())
            gam, bet = 1.0 / (sa * sb), -ncc / sa ** 2
            alp = -gam * bv.mean() - bet * lv.mean()
            got_n.append(float(alp) * mom[v, 0] + float(bet) * mom[v, 1] + float(gam) * mom[v, 2])
        ref_n = dfp.forward_pose_grad(g, a, p, vol, torch.stack(up_n).contiguous()).cpu().numpy()
        assert grad_err_u9(np.stack(got_n), ref_n).max() <= 2e-3      # alpha, beta, gamma cancel heavily for NCC


def test_fused_moments_reject_interp_mode_and_bad_arguments(dfp):
    w = W.make_config(1)
    dev = torch.device("cuda:0")
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    vol = w.volume(dev)
    tgt = torch.zeros((1,) + w.geom.det_shape, device=dev)
    with pytest.raises(dfp.DfpError):
        dfp.forward_fused_moments(w.geom.replace(flags=dfp.FLAG_GRAD_INTERP), a, p, vol, tgt)


# ------------------------------------------------------------------ randomised geometry sweep: TMA vs gather paths
def test_random_geometries_both_paths_agree_and_never_nan(dfp):
    """40 seeded random scanners / grids / poses (cone angles up to ~25 degrees, anisotropic voxels and pixels,
    shifted principal points, views all around, rotations up to 20 degrees).  Whatever path the host picks, the result
    must be finite (a NaN is the kernels' signal that a staged box / patch did not hold its tile: the host-side bound
    would be wrong) and agree with the gather path; every third case is also checked against the oracle."""
    rng = np.random.default_rng(2508_13304)
    dev = torch.device("cuda:0")
    n_tma = 0
    for case in range(40):
        nx, ny, nz = (int(4 * rng.integers(5, 15)) for _ in range(3))
        nu, nv = int(4 * rng.integers(6, 30)), int(rng.integers(9, 70))
        vox = rng.uniform(0.6, 1.6, 3)
        sad = rng.uniform(250.0, 900.0)
        sdd = sad * rng.uniform(1.3, 2.0)
        # pixel pitch from 0.3 to 2 voxels at the isocentre: both the TMA paths and their fallbacks get exercised
        du, dv = (vox.mean() * sdd / sad * rng.uniform(0.3, 2.0) for _ in range(2))
        g = W.Geometry(nx=nx, ny=ny, nz=nz, vx=vox[0], vy=vox[1], vz=vox[2], nu=nu, nv=nv, du=du, dv=dv, sad=sad,
                       sdd=sdd, cx=rng.uniform(-3, 3), cy=rng.uniform(-3, 3), cz=rng.uniform(-3, 3),
                       u0=rng.uniform(-2, 2), v0=rng.uniform(-2, 2), bp_weight=int(case % 2)).f32()
        V = int(rng.integers(1, 6))
        angles = f32(rng.uniform(0, 2 * math.pi, V))
        poses = f32(np.concatenate([rng.uniform(-8, 8, (V, 3)), rng.uniform(-0.35, 0.35, (V, 3))], axis=1))
        vol = torch.as_tensor(rng.random(g.vol_shape).astype(np.float32), device=dev)
        up = torch.as_tensor(rng.standard_normal((V,) + g.det_shape).astype(np.float32), device=dev)
        bup = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
        # back-projection input: seeded smooth images (no oracle input ever comes from the CUDA path)
        iv_, iu_ = np.meshgrid(np.arange(g.nv), np.arange(g.nu), indexing="ij")
        pin_np = np.stack([np.sin(0.21 * iu_ + 0.13 * iv_ + k) + 0.5 * np.cos(0.07 * iu_ - 0.19 * iv_ + 2 * k)
                           for k in range(V)]).astype(np.float32)
        pin = torch.as_tensor(pin_np, device=dev)
        gn = g.replace(flags=dfp.FLAG_NO_TMA)
        proj = dfp.forward(g, angles, poses, vol)
        n_tma += dfp.last_path()
        grad = dfp.forward_pose_grad(g, angles, poses, vol, up)
        n_tma += dfp.last_path()
        bp = dfp.backproject(g, angles, poses, pin)
        n_tma += dfp.last_path()
        bgrad = dfp.backproject_pose_grad(g, angles, poses, pin, bup)
        n_tma += dfp.last_path()
        for t in (proj, grad, bp, bgrad):
            assert torch.isfinite(t).all(), (case, g)
        assert rel_l2(proj.cpu().numpy(), dfp.forward(gn, angles, poses, vol).cpu().numpy()) <= 2e-6, case
        assert grad_err_u9(grad.cpu().numpy(),
                           dfp.forward_pose_grad(gn, angles, poses, vol, up).cpu().numpy()).max() <= 2e-3, case      # each path within 1e-3 of the truth
        assert rel_l2(bp.cpu().numpy(), dfp.backproject(gn, angles, poses, pin).cpu().numpy()) <= 1e-5, case
        assert grad_err_u9(bgrad.cpu().numpy(),
                           dfp.backproject_pose_grad(gn, angles, poses, pin, bup).cpu().numpy()).max() <= 2e-3, case   # each path within 1e-3 of the truth
        if case % 3 == 0:
            check_forward((proj.cpu().numpy(), grad.cpu().numpy(), oracle.forward(g, angles, poses, vol.cpu().numpy()),
                           oracle.forward_pose_grad(g, angles, poses, vol.cpu().numpy(), up.cpu().numpy())))
            check_back((bp.cpu().numpy(), bgrad.cpu().numpy(), oracle.backproject(g, angles, poses, pin_np),
                        oracle.backproject_pose_grad(g, angles, poses, pin_np, bup.cpu().numpy())))
    assert 40 <= n_tma <= 150, n_tma      # a healthy mix of TMA and fallback calls (4 calls per case)


def test_host_buffer_entry_points_chunked_views(dfp):
    """>= 8 views: the host-buffer calls move per-view arrays in 4 chunks on a second stream, overlapped with the
    kernels (a9, view chunking); 9 views give uneven chunks (2, 2, 2, 3).  Same results as the device-pointer calls
    on the whole batch (per-view outputs do not depend on how the views are grouped)."""
    w = W.make_config(2, scale=0.25, n_views=9)
    g = w.geom
    dev = torch.device("cuda:0")
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    vol, up = w.volume(), w.fwd_upstream()
    vd, ud = vol.to(dev), up.to(dev)
    proj = dfp.forward(g, a, p, vd)
    assert torch.equal(dfp.forward_host(g, a, p, vol.numpy()), proj.cpu())
    assert torch.equal(dfp.forward_pose_grad_host(g, a, p, vol.numpy(), up.numpy()),
                       dfp.forward_pose_grad(g, a, p, vd, ud).cpu())
    pj = proj.cpu().numpy()
    wv = np.random.default_rng(5).standard_normal(g.vol_shape).astype(np.float32)
    # the back-projection sums its 4 view chunks with DFP_FLAG_ACCUMULATE: same terms, another fp32 summation order
    assert rel_l2(dfp.backproject_host(g, a, p, pj).numpy(), dfp.backproject(g, a, p, proj).cpu().numpy()) <= 1e-6
    got = dfp.backproject_pose_grad_host(g, a, p, pj, wv).numpy()
    ref = dfp.backproject_pose_grad(g, a, p, proj, torch.as_tensor(wv, device=dev)).cpu().numpy()
    assert np.array_equal(got, ref)


def test_host_buffer_chunks_keep_alignment_on_odd_detectors(dfp):
    """nu * nv odd (21 x 17) with 9..11 views: a chunk that started at view 2 had an image offset of 8 mod 16 bytes
    (DFP_ERR_ALIGN after chunk 0 was queued).  Chunk boundaries are multiples of 4 views; all four host calls."""
    g = aniso_geom()
    assert (g.nu * g.nv) % 2 == 1
    rng = np.random.default_rng(11)
    dev = torch.device("cuda:0")
    for V in (9, 10, 11, 13):
        a = f32(np.linspace(0.0, 5.0, V))
        p = f32(np.concatenate([rng.uniform(-3, 3, (V, 3)), rng.uniform(-0.2, 0.2, (V, 3))], axis=1))
        vol = rng.standard_normal(g.vol_shape).astype(np.float32)
        up = rng.standard_normal((V,) + g.det_shape).astype(np.float32)
        wv = rng.standard_normal(g.vol_shape).astype(np.float32)
        vd, ud, wd = (torch.as_tensor(x, device=dev) for x in (vol, up, wv))
        proj = dfp.forward(g, a, p, vd)
        assert torch.equal(dfp.forward_host(g, a, p, vol), proj.cpu())
        assert torch.equal(dfp.forward_pose_grad_host(g, a, p, vol, up), dfp.forward_pose_grad(g, a, p, vd, ud).cpu())
        pj = proj.cpu().numpy()
        assert rel_l2(dfp.backproject_host(g, a, p, pj).numpy(), dfp.backproject(g, a, p, proj).cpu().numpy()) <= 1e-6
        assert torch.equal(dfp.backproject_pose_grad_host(g, a, p, pj, wv),
                           dfp.backproject_pose_grad(g, a, p, proj, wd).cpu())


def test_more_views_than_one_grid_holds(dfp):
    """70 000 views (> 65 535, the grid-z limit): the library slices the batch internally; every view's result equals
    the one it has in a small batch.  All four calls and the unit counter, on a tiny scanner."""
    g = W.Geometry(nx=8, ny=8, nz=8, vx=1.0, vy=1.0, vz=1.0, nu=8, nv=4, du=1.5, dv=1.5, sad=60.0, sdd=90.0)
    V = 70000
    rng = np.random.default_rng(12)
    dev = torch.device("cuda:0")
    a = f32(rng.uniform(0, 6.28, V))
    p = f32(np.concatenate([rng.uniform(-1, 1, (V, 3)), rng.uniform(-0.1, 0.1, (V, 3))], axis=1))
    vol = torch.as_tensor(rng.random(g.vol_shape).astype(np.float32), device=dev)
    up = torch.as_tensor(rng.standard_normal((V,) + g.det_shape).astype(np.float32), device=dev)
    wv = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
    proj = dfp.forward(g, a, p, vol)
    grad = dfp.forward_pose_grad(g, a, p, vol, up)
    bgrad = dfp.backproject_pose_grad(g, a, p, proj, wv)
    bp = dfp.backproject(g, a, p, proj)
    assert all(torch.isfinite(t).all() for t in (proj, grad, bgrad, bp))
    sel = np.array([0, 1, 65531, 65532, 65535, 65536, 69999])
    ps, us = proj[sel].contiguous(), up[sel].contiguous()
    # (another batch may get another staging box / tile depth: the same terms in another fp32 order)
    assert rel_l2(dfp.forward(g, a[sel], p[sel], vol).cpu().numpy(), ps.cpu().numpy()) <= 1e-6
    assert grad_err_u9(dfp.forward_pose_grad(g, a[sel], p[sel], vol, us).cpu().numpy(), grad[sel].cpu().numpy()).max() <= 1e-4
    assert grad_err_u9(dfp.backproject_pose_grad(g, a[sel], p[sel], ps, wv).cpu().numpy(),
                       bgrad[sel].cpu().numpy()).max() <= 1e-4
    # the volume is the sum over all views: two halves accumulated == the whole, up to the fp32 order of the sum
    h = dfp.backproject(g, a[:35000], p[:35000], proj[:35000].contiguous())
    dfp.backproject(g.replace(flags=dfp.FLAG_ACCUMULATE), a[35000:], p[35000:], proj[35000:].contiguous(), out=h)
    assert rel_l2(h.cpu().numpy(), bp.cpu().numpy()) <= 1e-5
    n_all = dfp.count_ray_steps(g, a, p)
    assert n_all == dfp.count_ray_steps(g, a[:65532], p[:65532]) + dfp.count_ray_steps(g, a[65532:], p[65532:])


# ------------------------------------------------------------------ DFP_FLAG_SIDDON
def run_siddon_case(dfp, g, angles, poses, vol, up):
    dev = torch.device("cuda:0")
    gs = g.replace(flags=g.flags | dfp.FLAG_SIDDON)
    angles, poses = f32(angles), f32(poses).reshape(-1, 6)
    vol_d = torch.as_tensor(vol, dtype=torch.float32, device=dev).contiguous()
    up_d = torch.as_tensor(up, dtype=torch.float32, device=dev).contiguous()
    proj = dfp.forward(gs, angles, poses, vol_d).cpu().numpy()
    grad = dfp.forward_pose_grad(gs, angles, poses, vol_d, up_d).cpu().numpy()
    o_proj = oracle.forward_siddon(g, angles, poses, vol_d.cpu().numpy())
    o_grad = oracle.forward_pose_grad_siddon(g, angles, poses, vol_d.cpu().numpy(), up_d.cpu().numpy())
    return proj, grad, o_proj, o_grad


def test_siddon_ragged_anisotropic_and_degenerate(dfp):
    g = aniso_geom(nx=37, ny=29, nz=23, nu=45, nv=21)
    rng = np.random.default_rng(30)
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((3,) + g.det_shape).astype(np.float32)
    check_forward(run_siddon_case(dfp, g, ANGLES3, POSES3, vol, up))
    # axis-parallel central ray (beta = 0, identity pose, odd detector: the middle ray has e_y = e_z = 0 exactly)
    g = small_geom(n=12, nu=11, nv=9)
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((1,) + g.det_shape).astype(np.float32)
    check_forward(run_siddon_case(dfp, g, [0.0], [[0] * 6], vol, up))
    # diagonal views of an even grid: the middle ray runs through voxel CORNERS (x and y planes crossed together, to
    # within rounding of cos / sin) inside the plane z = 0 - coincident crossings, which the DDA may take in either
    # order or count differently from its fp64 set-up (zero-length segments either way)
    g = small_geom(n=16, nu=11, nv=9)
    vol = rng.random(g.vol_shape).astype(np.float32)
    diag = [math.pi / 4, 3 * math.pi / 4, -math.pi / 4, 5 * math.pi / 4]
    up4 = rng.standard_normal((4,) + g.det_shape).astype(np.float32)
    check_forward(run_siddon_case(dfp, g, diag, [[0] * 6] * 4, vol, up4))
    g = small_geom(n=12, nu=11, nv=9)
    # misses and an empty volume: exact zeros
    proj, grad, _, _ = run_siddon_case(dfp, g, [0.3], [[0, 0, 700.0, 0, 0, 0]], vol[:12, :12, :12].copy(), up)
    assert np.all(proj == 0) and np.all(grad == 0)
    # single voxel
    g1 = small_geom(n=1, voxel=4.0, nu=3, nv=3, pix=1.0)
    check_forward(run_siddon_case(dfp, g1, [0.2], [[0.3, 0.2, -0.1, 0.01, 0.02, 0.03]], np.full(g1.vol_shape, 0.7, np.float32),
                                  np.ones((1,) + g1.det_shape, np.float32)))


@pytest.mark.parametrize("index,scale,views", [(1, 1.0, None), (2, 0.25, 3), (4, 0.125, 4), (5, 0.125, 3)])
def test_siddon_configs_reduced(dfp, index, scale, views):
    w = W.make_config(index, scale=scale, n_views=views)
    check_forward(run_siddon_case(dfp, w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy(),
                                  w.fwd_upstream().numpy()))


def test_siddon_rejects_modes_it_does_not_have(dfp):
    w = W.make_config(1)
    dev = torch.device("cuda:0")
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    vol, up = w.volume(dev), w.fwd_upstream(dev)
    with pytest.raises(dfp.DfpError):
        dfp.forward_pose_grad(w.geom.replace(flags=dfp.FLAG_SIDDON | dfp.FLAG_GRAD_INTERP), a, p, vol, up)
    with pytest.raises(dfp.DfpError):
        dfp.forward_fused_moments(w.geom.replace(flags=dfp.FLAG_SIDDON), a, p, vol, up)


def test_tma_paths_axis_aligned_views_and_other_step_sizes(dfp):
    """Gantry at 0 / 90 / 180 / 270 degrees with the identity pose (ray direction components exactly zero: chunk
    lengths limited by one axis only), and ray-march steps of 0.45 and 1.7 voxels (longer / shorter chunks)."""
    w = W.make_config(2, scale=0.25, n_views=4)
    vol = w.volume().numpy()
    up = w.fwd_upstream().numpy()
    angles = [0.0, math.pi / 2, math.pi, 1.5 * math.pi]
    zero = np.zeros((4, 6))
    dev = torch.device("cuda:0")
    for step in (0.0, 0.45 * w.geom.vx, 1.7 * w.geom.vx):
        g = w.geom.replace(step_mm=step)
        res = run_forward_case(dfp, g, angles, zero, vol, up)
        assert dfp.last_path() == dfp.PATH_TMA
        check_forward(res)
    w.angles = torch.tensor(angles, dtype=torch.float64)        # closed-form projections at these four views
    proj = w.projections().numpy()
    bup = np.random.default_rng(31).standard_normal(w.geom.vol_shape).astype(np.float32)
    resb = run_back_case(dfp, w.geom, angles, zero, proj, bup)
    assert dfp.last_path() == dfp.PATH_TMA
    check_back(resb)


def test_backproject_accumulate_flag_sums_view_slices(dfp):
    """DFP_FLAG_ACCUMULATE: back-projecting views [0, k) and then adding views [k, V) equals the whole call (Eq.21 is a
    sum over views), on both kernel paths; without the flag the second call would overwrite."""
    w = W.make_config(3, scale=0.25, n_views=10)
    dev = torch.device("cuda:0")
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    proj = w.projections(dev)
    for base in (0, dfp.FLAG_NO_TMA):
        g = w.geom.replace(flags=base)
        whole = dfp.backproject(g, a, p, proj).cpu().numpy()
        vol = dfp.backproject(g, a[:4], p[:4], proj[:4].contiguous())
        first = vol.cpu().numpy().copy()
        ga = g.replace(flags=base | dfp.FLAG_ACCUMULATE)
        dfp.backproject(ga, a[4:], p[4:], proj[4:].contiguous(), out=vol)
        assert rel_l2(vol.cpu().numpy(), whole) <= 1e-6
        assert rel_l2(first, whole) > 0.1                      # the first slice alone is not the answer


# ------------------------------------------------------------------ DFP_FLAG_JOSEPH
def run_joseph_case(dfp, g, angles, poses, vol, up):
    dev = torch.device("cuda:0")
    gj = g.replace(flags=g.flags | dfp.FLAG_JOSEPH)
    angles, poses = f32(angles), f32(poses).reshape(-1, 6)
    vol_d = torch.as_tensor(vol, dtype=torch.float32, device=dev).contiguous()
    up_d = torch.as_tensor(up, dtype=torch.float32, device=dev).contiguous()
    proj = dfp.forward(gj, angles, poses, vol_d).cpu().numpy()
    grad = dfp.forward_pose_grad(gj, angles, poses, vol_d, up_d).cpu().numpy()
    o_proj = oracle.forward_joseph(g, angles, poses, vol_d.cpu().numpy())
    o_grad = oracle.forward_pose_grad_joseph(g, angles, poses, vol_d.cpu().numpy(), up_d.cpu().numpy())
    return proj, grad, o_proj, o_grad


def test_joseph_ragged_anisotropic_all_driving_axes_and_degenerate(dfp):
    g = aniso_geom(nx=37, ny=29, nz=23, nu=45, nv=21)
    rng = np.random.default_rng(40)
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((4,) + g.det_shape).astype(np.float32)
    # views driven along x, along y, and (tilted by 70 degrees about y) along z
    angles = [0.4, math.pi / 2, 4.1, 0.1]
    poses = POSES3 + [[0.5, 0.3, 0.2, 0.05, 1.2, 0.0]]
    check_forward(run_joseph_case(dfp, g, angles, poses, vol, up))
    g = small_geom(n=12, nu=11, nv=9)                        # axis-parallel central ray
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((1,) + g.det_shape).astype(np.float32)
    check_forward(run_joseph_case(dfp, g, [0.0], [[0] * 6], vol, up))
    proj, grad, _, _ = run_joseph_case(dfp, g, [0.3], [[0, 0, 700.0, 0, 0, 0]], vol, up)
    assert np.all(proj == 0) and np.all(grad == 0)
    g1 = small_geom(n=1, voxel=4.0, nu=3, nv=3, pix=1.0)
    check_forward(run_joseph_case(dfp, g1, [0.2], [[0.3, 0.2, -0.1, 0.01, 0.02, 0.03]], np.full(g1.vol_shape, 0.7, np.float32),
                                  np.ones((1,) + g1.det_shape, np.float32)))


@pytest.mark.parametrize("index,scale,views", [(1, 1.0, None), (2, 0.25, 3), (4, 0.125, 4), (5, 0.125, 3)])
def test_joseph_configs_reduced(dfp, index, scale, views):
    w = W.make_config(index, scale=scale, n_views=views)
    check_forward(run_joseph_case(dfp, w.geom, w.angles.numpy(), w.poses.numpy(), w.volume().numpy(),
                                  w.fwd_upstream().numpy()))


def test_joseph_and_siddon_flags_exclude_each_other(dfp):
    w = W.make_config(1)
    dev = torch.device("cuda:0")
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    with pytest.raises(dfp.DfpError):
        dfp.forward(w.geom.replace(flags=dfp.FLAG_SIDDON | dfp.FLAG_JOSEPH), a, p, w.volume(dev))


# ------------------------------------------------------------------ dfp_microbench (roofline denominators)
def test_microbench_rates_are_those_of_a_b200_class_sm():
    """One warp-wide LDS per clock per SM and 128 fp32 lanes per SM at 1-2.5 GHz on >= 100 SMs.
    The probes live in libdfp_bench.so (include/dfp_bench.h), outside the product library."""
    from paper_2508_13304_b200 import microbench as mb
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    lds = mb.run(mb.MB_LDS) / n_sm
    assert 0.8e9 < lds < 2.6e9, lds                              # ~1 per clock
    for kind in (mb.MB_FADD, mb.MB_FFMA, mb.MB_FFMA2):
        r = mb.run(kind) / n_sm
        assert 100 * 0.9e9 < r < 130 * 2.6e9, (kind, r)          # ~128 per clock


# ------------------------------------------------------------------ DFP_FLAG_DD (distance-driven pair)
def run_dd_case(dfp, g, angles, poses, vol, up, proj, bup, model="dd"):
    """All four calls with distance-driven (O15) or separable-footprint (O16) weights against the oracle."""
    dev = torch.device("cuda:0")
    gd = g.replace(flags=g.flags | (dfp.FLAG_DD if model == "dd" else dfp.FLAG_SF))
    angles, poses = f32(angles), f32(poses).reshape(-1, 6)
    t = lambda x: torch.as_tensor(np.asarray(x), dtype=torch.float32, device=dev).contiguous()
    vol_d, up_d, proj_d, bup_d = t(vol), t(up), t(proj), t(bup)
    got = (dfp.forward(gd, angles, poses, vol_d).cpu().numpy(),
           dfp.forward_pose_grad(gd, angles, poses, vol_d, up_d).cpu().numpy(),
           dfp.backproject(gd, angles, poses, proj_d).cpu().numpy(),
           dfp.backproject_pose_grad(gd, angles, poses, proj_d, bup_d).cpu().numpy())
    vol_c, up_c, proj_c, bup_c = (x.cpu().numpy() for x in (vol_d, up_d, proj_d, bup_d))
    o = {k: getattr(oracle, k + "_" + model) for k in ("forward", "forward_pose_grad", "backproject", "backproject_pose_grad")}
    ref = (o["forward"](g, angles, poses, vol_c), o["forward_pose_grad"](g, angles, poses, vol_c, up_c),
           o["backproject"](g, angles, poses, proj_c), o["backproject_pose_grad"](g, angles, poses, proj_c, bup_c))
    return got, ref


def check_dd(res, zero_border=False):
    got, ref = res
    check_values(got[0], ref[0], TOL_VAL, zero_border=zero_border)
    check_values(got[2], ref[2], TOL_VAL, zero_border=False)
    for k in (1, 3):
        assert np.all(np.isfinite(got[k]))
        e = grad_err_u9(got[k], ref[k])
        assert e.max() <= TOL_GRAD, (k, e)


def test_dd_ragged_anisotropic_all_driving_axes_and_degenerate(dfp):
    """Non-cubic grid, odd sizes, shifted principal point; views driven along x, along y and - the pose tilted by 70
    degrees about y - along z; a 45-degree in-plane rotation (u pairs with the other in-plane axis); missing rays."""
    g = aniso_geom(nx=37, ny=29, nz=23, nu=45, nv=21)
    rng = np.random.default_rng(40)
    vol = rng.random(g.vol_shape).astype(np.float32)
    angles = [0.4, math.pi / 2, 4.1, 0.1, 0.3]
    poses = POSES3 + [[0.5, 0.3, 0.2, 0.05, 1.2, 0.0], [1.0, -1.0, 0.5, 0.9, 0.1, -0.1]]
    up = rng.standard_normal((5,) + g.det_shape).astype(np.float32)
    iv, iu = np.meshgrid(np.arange(g.nv), np.arange(g.nu), indexing="ij")
    proj = np.stack([np.sin(0.21 * iu + 0.13 * iv + k) + 0.5 * np.cos(0.07 * iu - 0.19 * iv + 2 * k) for k in range(5)])
    bup = rng.standard_normal(g.vol_shape).astype(np.float32)
    check_dd(run_dd_case(dfp, g, angles, poses, vol, up, proj, bup))
    # the object pushed out of the cone: exact zeros everywhere
    got, _ = run_dd_case(dfp, g, [0.2], [[0, 0, 400.0, 0, 0, 0]], vol, up[:1], proj[:1], bup)
    assert not got[0].any() and not got[1].any() and not got[2].any() and not got[3].any()


@pytest.mark.parametrize("index,scale,views", [(1, 1.0, None), (2, 0.25, 3), (3, 0.25, 6), (5, 0.125, 4)])
def test_dd_configs_reduced(dfp, index, scale, views):
    w = W.make_config(index, scale=scale, n_views=views)
    g = w.geom.replace(bp_weight=0)
    check_dd(run_dd_case(dfp, g, w.angles.numpy(), w.poses.numpy(), w.volume().numpy(), w.fwd_upstream().numpy(),
                         w.projections().numpy(), w.bp_upstream().numpy()), zero_border=True)


def test_dd_is_a_matched_pair_and_rejects_what_it_does_not_have(dfp):
    """<A x, y> = <x, A^T y> on the GPU (the DD back-projector is the exact transpose of the DD forward projector,
    Eq.18 / 21: both kernels evaluate the same weight formula), the ACCUMULATE flag, and the error codes."""
    dev = torch.device("cuda:0")
    w = W.make_config(2, scale=0.25, n_views=4)
    g = w.geom.replace(flags=dfp.FLAG_DD)
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    rng = np.random.default_rng(41)
    x = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
    y = torch.as_tensor(rng.standard_normal((4,) + g.det_shape).astype(np.float32), device=dev)
    Ax, ATy = dfp.forward(g, a, p, x), dfp.backproject(g, a, p, y)
    lhs, rhs = float((Ax.double() * y.double()).sum()), float((x.double() * ATy.double()).sum())
    assert abs(lhs - rhs) <= 2e-6 * abs(lhs), (lhs, rhs)
    half = dfp.backproject(g, a[:2], p[:2], y[:2].contiguous())
    dfp.backproject(g.replace(flags=dfp.FLAG_DD | dfp.FLAG_ACCUMULATE), a[2:], p[2:], y[2:].contiguous(), out=half)
    assert rel_l2(half.cpu().numpy(), ATy.cpu().numpy()) <= 1e-6
    for bad in (g.replace(flags=dfp.FLAG_DD | dfp.FLAG_SIDDON), g.replace(flags=dfp.FLAG_DD | dfp.FLAG_GRAD_INTERP)):
        with pytest.raises(dfp.DfpError):
            dfp.forward_pose_grad(bad, a, p, x, y)
    with pytest.raises(dfp.DfpError):
        dfp.backproject(g.replace(bp_weight=1), a, p, y)
    with pytest.raises(dfp.DfpError):
        dfp.forward_fused_moments(g, a, p, x, y)


# ------------------------------------------------------------------ DFP_FLAG_SF (separable-footprint pair)
def test_sf_ragged_anisotropic_general_poses_and_degenerate(dfp):
    g = aniso_geom(nx=37, ny=29, nz=23, nu=45, nv=21)
    rng = np.random.default_rng(50)
    vol = rng.random(g.vol_shape).astype(np.float32)
    angles = [0.4, math.pi / 2, 4.1, 0.1, 0.3]
    poses = POSES3 + [[0.5, 0.3, 0.2, 0.05, 1.2, 0.0], [1.0, -1.0, 0.5, 0.9, 0.1, -0.1]]
    up = rng.standard_normal((5,) + g.det_shape).astype(np.float32)
    iv, iu = np.meshgrid(np.arange(g.nv), np.arange(g.nu), indexing="ij")
    proj = np.stack([np.sin(0.21 * iu + 0.13 * iv + k) + 0.5 * np.cos(0.07 * iu - 0.19 * iv + 2 * k) for k in range(5)])
    bup = rng.standard_normal(g.vol_shape).astype(np.float32)
    check_dd(run_dd_case(dfp, g, angles, poses, vol, up, proj, bup, model="sf"))
    got, _ = run_dd_case(dfp, g, [0.2], [[0, 0, 400.0, 0, 0, 0]], vol, up[:1], proj[:1], bup, model="sf")
    assert not got[0].any() and not got[1].any() and not got[2].any() and not got[3].any()


@pytest.mark.parametrize("index,scale,views", [(1, 1.0, None), (2, 0.25, 3), (3, 0.25, 6), (5, 0.125, 4)])
def test_sf_configs_reduced(dfp, index, scale, views):
    w = W.make_config(index, scale=scale, n_views=views)
    g = w.geom.replace(bp_weight=0)
    check_dd(run_dd_case(dfp, g, w.angles.numpy(), w.poses.numpy(), w.volume().numpy(), w.fwd_upstream().numpy(),
                         w.projections().numpy(), w.bp_upstream().numpy(), model="sf"), zero_border=True)


def test_sf_is_a_matched_pair_and_rejects_what_it_does_not_have(dfp):
    dev = torch.device("cuda:0")
    w = W.make_config(2, scale=0.25, n_views=4)
    g = w.geom.replace(flags=dfp.FLAG_SF)
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    rng = np.random.default_rng(51)
    x = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
    y = torch.as_tensor(rng.standard_normal((4,) + g.det_shape).astype(np.float32), device=dev)
    Ax, ATy = dfp.forward(g, a, p, x), dfp.backproject(g, a, p, y)
    lhs, rhs = float((Ax.double() * y.double()).sum()), float((x.double() * ATy.double()).sum())
    assert abs(lhs - rhs) <= 2e-6 * abs(lhs), (lhs, rhs)
    half = dfp.backproject(g, a[:2], p[:2], y[:2].contiguous())
    dfp.backproject(g.replace(flags=dfp.FLAG_SF | dfp.FLAG_ACCUMULATE), a[2:], p[2:], y[2:].contiguous(), out=half)
    assert rel_l2(half.cpu().numpy(), ATy.cpu().numpy()) <= 1e-6
    for bad in (g.replace(flags=dfp.FLAG_SF | dfp.FLAG_DD), g.replace(flags=dfp.FLAG_SF | dfp.FLAG_GRAD_INTERP)):
        with pytest.raises(dfp.DfpError):
            dfp.forward_pose_grad(bad, a, p, x, y)
        with pytest.raises(dfp.DfpError):
            dfp.backproject(bad, a, p, y)
    with pytest.raises(dfp.DfpError):
        dfp.backproject(g.replace(bp_weight=1), a, p, y)


def test_sf_forward_is_deterministic_and_scale_free(dfp):
    """The SF forward projector scatters with 64-bit fixed-point integer atomics (dfp_sf.cuh): the sum does not depend
    on the order the atomics land in, so repeated calls agree BIT FOR BIT; the fixed-point scale follows max|mu|, so the
    result is exactly homogeneous in powers of two of the volume's magnitude, tiny and huge; an all-zero volume gives
    exact zeros and a NaN in the volume reaches every pixel of the call (no silent integer garbage)."""
    dev = torch.device("cuda:0")
    w = W.make_config(2, scale=0.25, n_views=3)
    g = w.geom.replace(flags=dfp.FLAG_SF)
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    rng = np.random.default_rng(52)
    x = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
    ref = dfp.forward(g, a, p, x).clone()
    for _ in range(3):
        assert torch.equal(dfp.forward(g, a, p, x), ref)
    for k in (-100, -20, 30, 90):
        s = float(2.0 ** k)
        assert torch.equal(dfp.forward(g, a, p, x * s), ref * s), k
    assert not dfp.forward(g, a, p, torch.zeros_like(x)).any()
    bad = x.clone()
    bad[3, 4, 5] = float("nan")
    assert torch.isnan(dfp.forward(g, a, p, bad)).all()


def test_dd_backprojector_is_deterministic_scale_free_and_accumulates(dfp):
    """The DD back-projector is the forward traversal with the read turned into a scatter of 64-bit fixed-point
    integers (dfp_dd.cuh): repeated calls agree BIT FOR BIT, the result is exactly homogeneous in powers of two of the
    projections' magnitude (the scale follows max|l|), zero projections give exact zeros, a NaN pixel reaches every
    voxel of the call, and DFP_FLAG_ACCUMULATE adds a second slice of views onto the first."""
    dev = torch.device("cuda:0")
    w = W.make_config(2, scale=0.25, n_views=4)
    g = w.geom.replace(flags=dfp.FLAG_DD)
    a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
    rng = np.random.default_rng(53)
    y = torch.as_tensor(rng.standard_normal((4,) + g.det_shape).astype(np.float32), device=dev)
    ref = dfp.backproject(g, a, p, y).clone()
    for _ in range(3):
        assert torch.equal(dfp.backproject(g, a, p, y), ref)
    for k in (-100, -20, 30, 90):
        s = float(2.0 ** k)
        assert torch.equal(dfp.backproject(g, a, p, y * s), ref * s), k
    assert not dfp.backproject(g, a, p, torch.zeros_like(y)).any()
    bad = y.clone()
    bad[1, 3, 4] = float("nan")
    assert torch.isnan(dfp.backproject(g, a, p, bad)).all()
    half = dfp.backproject(g, a[:2], p[:2], y[:2].contiguous())
    dfp.backproject(g.replace(flags=dfp.FLAG_DD | dfp.FLAG_ACCUMULATE), a[2:], p[2:], y[2:].contiguous(), out=half)
    assert rel_l2(half.cpu().numpy(), ref.cpu().numpy()) <= 1e-6


# ------------------------------------------------------------------ gradient kernels by view class
@pytest.mark.parametrize("nx,ny", [(48, 40), (48, 42), (46, 41)])
def test_gradient_kernels_by_view_class_non_cubic_grid(dfp, nx, ny):
    """At >= 0.45 voxel per pixel dfp_forward_pose_grad sorts its views by the in-plane direction of their central ray:
    near the diagonals -> fwd_tma_kernel<1, 3>, along y -> <5, 6>, along x -> <6, 6> on a TRANSPOSED copy of the volume.
    A non-cubic, anisotropic grid (the transposed tensor map, the swapped centre indices and the swapped sums would all
    show), views of all three classes in one call in mixed order, general poses; the launch count proves that the three
    kernels ran (3 + transpose + contraction).  nx % 4 != 0 / ny % 4 != 0: the row-padded copy of the volume and the
    row-padded transposed volume."""
    launches = 5
    g = W.Geometry(nx=nx, ny=ny, nz=28, vx=0.5, vy=0.55, vz=0.5, nu=64, nv=40, du=0.4, dv=0.4, sad=400.0, sdd=600.0,
                   cx=0.7, cy=-0.4, cz=0.3, u0=0.6, v0=-0.8).f32()
    angles = [0.05, 0.8, 1.6, 3.1, 2.4, 4.75, 5.5, 6.2, 1.45]
    rng = np.random.default_rng(77)
    poses = np.concatenate([rng.uniform(-1.5, 1.5, (len(angles), 3)), rng.uniform(-0.06, 0.06, (len(angles), 3))], axis=1)
    vol = rng.random(g.vol_shape).astype(np.float32)
    up = rng.standard_normal((len(angles),) + g.det_shape).astype(np.float32)
    res = run_forward_case(dfp, g, angles, poses, vol, up)
    dev = torch.device("cuda:0")
    dfp.forward_pose_grad(g, f32(angles), f32(poses), torch.as_tensor(vol, device=dev), torch.as_tensor(up, device=dev))
    assert dfp.last_path() == dfp.PATH_TMA and dfp.last_launch_count() == launches
    check_forward(res)
    # and the same numbers as the gather path to fp32 rounding
    gg = g.replace(flags=dfp.FLAG_NO_TMA)
    ref = dfp.forward_pose_grad(gg, f32(angles), f32(poses), torch.as_tensor(vol, device=dev),
                                torch.as_tensor(up, device=dev)).cpu().numpy()
    assert grad_err_u9(res[1], ref).max() <= 1e-4


# ------------------------------------------------------------------ dfp_workspace_bytes_for_views
def test_exact_size_workspace_serves_the_call_and_one_byte_less_does_not(dfp):
    """A workspace of dfp_workspace_bytes_for_views bytes (no 4x packed copy: the views take the TMA path) gives the
    same results, bit for bit, as the any-views size; 256 bytes less is DFP_ERR_WORKSPACE before any launch (the output
    stays untouched).  Odd row lengths: the exact size holds the row-padded copy.  A geometry on the gather path: the
    two sizes coincide."""
    dev = torch.device("cuda:0")
    for kw in (dict(), dict(nx=62, nu=126)):
        w = W.make_config(2, scale=0.25, n_views=4)
        g = w.geom.replace(**kw)
        a, p = f32(w.angles.numpy()), f32(w.poses.numpy()).reshape(-1, 6)
        rng = np.random.default_rng(61)
        vol = torch.as_tensor(rng.random(g.vol_shape).astype(np.float32), device=dev)
        up = torch.as_tensor(rng.standard_normal((4,) + g.det_shape).astype(np.float32), device=dev)
        upv = torch.as_tensor(rng.standard_normal(g.vol_shape).astype(np.float32), device=dev)
        calls = ((dfp.OP_FORWARD, lambda ws, out: dfp.forward(g, a, p, vol, out=out, ws=ws), (4,) + g.det_shape),
                 (dfp.OP_FORWARD_POSE_GRAD, lambda ws, out: dfp.forward_pose_grad(g, a, p, vol, up, out=out, ws=ws), (4, 6)),
                 (dfp.OP_BACKPROJECT, lambda ws, out: dfp.backproject(g, a, p, up, out=out, ws=ws), g.vol_shape),
                 (dfp.OP_BACKPROJECT_POSE_GRAD, lambda ws, out: dfp.backproject_pose_grad(g, a, p, up, upv, out=out, ws=ws), (4, 6)))
        for op, fn, shape in calls:
            full, exact = dfp.workspace_bytes(g, 4, op), dfp.workspace_bytes_for_views(g, a, p, op)
            assert 0 < exact < full // 2, (op, exact, full)
            ref = fn(torch.empty(full, dtype=torch.uint8, device=dev), torch.empty(shape, device=dev)).clone()
            assert dfp.last_path() == dfp.PATH_TMA
            got = fn(torch.empty(exact, dtype=torch.uint8, device=dev), torch.empty(shape, device=dev))
            assert dfp.last_path() == dfp.PATH_TMA and torch.equal(got, ref), op
            untouched = torch.full(shape, 7.0, device=dev)
            with pytest.raises(dfp.DfpError) as e:
                fn(torch.empty(exact - 256, dtype=torch.uint8, device=dev), untouched)
            assert e.value.status == -5 and bool((untouched == 7.0).all())
    gg = small_geom(n=64, voxel=0.25, nu=20, nv=18, pix=2.4)
    a1, p1 = f32([0.3]), f32([POSES3[0]])
    assert dfp.workspace_bytes_for_views(gg, a1, p1, dfp.OP_FORWARD) == dfp.workspace_bytes(gg, 1, dfp.OP_FORWARD)


def test_exact_size_workspace_is_enough_for_random_geometries(dfp):
    """dfp_workspace_bytes_for_views and the calls decide the kernel path with the same host code: over random grids,
    detectors, magnifications, poses, weights and modes a workspace of exactly that size is never too small, whichever
    path the call then takes, and the results do not depend on the workspace size."""
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(97)
    seen = set()
    for trial in range(24):
        n = [int(rng.integers(9, 41)) for _ in range(3)]
        nu, nv = int(rng.integers(8, 70)), int(rng.integers(8, 50))
        vox = float(rng.uniform(0.4, 1.5))
        sad = float(rng.uniform(150.0, 600.0))
        sdd = sad * float(rng.uniform(1.2, 2.0))
        pix = vox * sdd / sad * float(rng.uniform(0.3, 2.5))
        flags = int(rng.choice([0, 0, dfp.FLAG_GRAD_INTERP, dfp.FLAG_NO_TMA]))
        g = W.Geometry(nx=n[0], ny=n[1], nz=n[2], vx=vox, vy=vox * 1.1, vz=vox * 0.9, nu=nu, nv=nv, du=pix, dv=pix * 1.05,
                       sad=sad, sdd=sdd, bp_weight=int(rng.integers(0, 2)), flags=flags).f32()
        V = int(rng.integers(1, 6))
        a = f32(rng.uniform(0, 2 * np.pi, V))
        p = f32(np.concatenate([rng.uniform(-2, 2, (V, 3)), rng.uniform(-0.1, 0.1, (V, 3))], axis=1))
        vol = torch.as_tensor(rng.random(g.vol_shape).astype(np.float32), device=dev)
        img = torch.as_tensor(rng.random((V,) + g.det_shape).astype(np.float32), device=dev)
        for op, fn in ((dfp.OP_FORWARD, lambda ws: dfp.forward(g, a, p, vol, ws=ws)),
                       (dfp.OP_FORWARD_POSE_GRAD, lambda ws: dfp.forward_pose_grad(g, a, p, vol, img, ws=ws)),
                       (dfp.OP_BACKPROJECT, lambda ws: dfp.backproject(g, a, p, img, ws=ws)),
                       (dfp.OP_BACKPROJECT_POSE_GRAD, lambda ws: dfp.backproject_pose_grad(g, a, p, img, vol, ws=ws))):
            exact, full = dfp.workspace_bytes_for_views(g, a, p, op), dfp.workspace_bytes(g, V, op)
            assert 0 < exact <= full
            got = fn(torch.empty(exact, dtype=torch.uint8, device=dev)).clone()
            path = dfp.last_path()
            assert (exact < full) == (path == dfp.PATH_TMA), (trial, op, exact, full, path)
            ref = fn(torch.empty(full + 4096, dtype=torch.uint8, device=dev))
            assert dfp.last_path() == path and torch.equal(got, ref), (trial, op)
            seen.add((op, path))
    assert len(seen) == 8, seen          # both paths of all four calls were exercised
