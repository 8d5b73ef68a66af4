"""GPU-vs-oracle parity at BASELINE.json's FULL sizes (`-m gpu`), in the launch configuration `bench.py` times.

The CUDA path runs the whole config (all views, full grids) through the C ABI; the fp64 oracle recomputes
SAMPLED outputs one by one on the same seeded inputs:
  * projections: seeded views x a band of detector rows (the band is an exact sub-detector: `v0` shifts the
    principal point so that its rays are rays of the full detector);
  * forward pose gradients: seeded views, the full 6-vector (every ray of the view enters the sum);
  * back-projections: seeded z-slabs, all views;
  * back-projection pose gradients: seeded views, all voxels.
Tolerances as in test_gpu_parity.py (BASELINE.json north_star; U9).
"""
import numpy as np
import pytest
import torch

import oracle
import workloads as W
from helpers import check_values, grad_err_u9, rel_l2

pytestmark = pytest.mark.gpu

TOL_VAL = 1e-5
TOL_GRAD = 1e-3


@pytest.fixture(scope="module")
def dfp():
    import paper_2508_13304_b200 as m
    return m


def row_band(g, r0, rows):
    """Sub-detector made of rows [r0, r0+rows) of g: c_v' = c_v - r0."""
    v0 = (g.nv - 1) / 2.0 + g.v0 - r0 - (rows - 1) / 2.0
    return g.replace(nv=rows, v0=v0)


def pick(seed, n, k):
    rng = W.SplitMix64(seed)
    out = []
    while len(out) < k:
        v = int(rng.uniform(0.0, n)) % n
        if v not in out:
            out.append(v)
    return out


def check_forward_full(dfp, index, n_check_views, band_rows, n_grad_views):
    dev = torch.device("cuda:0")
    w = W.make_config(index)
    g = w.geom
    a = w.angles.float().numpy()
    p = w.poses.float().numpy()
    vol = w.volume(dev)
    up = w.fwd_upstream(dev)
    proj = dfp.forward(g, a, p, vol)
    grad = dfp.forward_pose_grad(g, a, p, vol, up).cpu().numpy()
    torch.cuda.synchronize()
    assert torch.isfinite(proj).all() and np.isfinite(grad).all()
    vol_c = vol.cpu().numpy()
    views = pick(w.seed + 101, w.n_views, n_check_views)
    for i, v in enumerate(views):
        r0 = pick(w.seed + 211 + v, g.nv - band_rows + 1, 1)[0]
        gb = row_band(g, r0, band_rows)
        o = oracle.forward(gb, a[v:v + 1], p[v:v + 1], vol_c)[0]
        got = proj[v, r0:r0 + band_rows].cpu().numpy()
        assert np.linalg.norm(o) > 0
        check_values(got, o, TOL_VAL, zero_border=True)
    gviews = pick(w.seed + 131, w.n_views, n_grad_views)
    o = oracle.forward_pose_grad(g, a[gviews], p[gviews], vol_c, up[gviews].cpu().numpy())
    e = grad_err_u9(grad[gviews], o)
    report(f"C{index} forward_pose_grad, {len(gviews)} seeded views", e)
    assert e.max() <= TOL_GRAD, (index, gviews, e)
    return w


def report(what, e):
    """Error quantiles of a [views, 6] table of U9 errors, into the test log (pytest -s / -rP shows it)."""
    q = np.quantile(e, [0.5, 0.9, 1.0])
    print(f"{what}: U9 error median {q[0]:.2e}  p90 {q[1]:.2e}  max {q[2]:.2e}  (tolerance {TOL_GRAD:.0e}); "
          f"per-view max " + " ".join(f"{x:.1e}" for x in e.max(axis=1)))


def check_back_full(dfp, index, n_slabs, slab, n_grad_views):
    dev = torch.device("cuda:0")
    w = W.make_config(index)
    g = w.geom
    a = w.angles.float().numpy()
    p = w.poses.float().numpy()
    proj = w.projections(dev)
    up = w.bp_upstream(dev)
    vol = dfp.backproject(g, a, p, proj)
    grad = dfp.backproject_pose_grad(g, a, p, proj, up).cpu().numpy()
    torch.cuda.synchronize()
    assert torch.isfinite(vol).all() and np.isfinite(grad).all()
    proj_c = proj.cpu().numpy()
    # the back-projection tolerance is on the whole volume: accumulate the sampled slabs into one relative L2
    num = den = 0.0
    for z0 in pick(w.seed + 307, g.nz - slab + 1, n_slabs):
        o = oracle.backproject(g, a, p, proj_c, z0, z0 + slab)
        d = vol[z0:z0 + slab].cpu().numpy().astype(np.float64) - o
        num += float((d * d).sum())
        den += float((o * o).sum())
        assert np.abs(d).max() <= 5e-5 * np.abs(o).max(), (index, z0)      # per element: no wrong voxel hides in the L2
    assert den > 0 and (num / den) ** 0.5 <= TOL_VAL, (index, (num / den) ** 0.5)
    up_c = up.cpu().numpy()
    gviews = pick(w.seed + 401, w.n_views, n_grad_views)
    o = oracle.backproject_pose_grad(g, a[gviews], p[gviews], proj_c[gviews], up_c)
    e = grad_err_u9(grad[gviews], o)
    report(f"C{index} backproject_pose_grad, {len(gviews)} seeded views", e)
    assert e.max() <= TOL_GRAD, (index, gviews, e)


def test_c2_registration_full(dfp):
    """The workload bench.py times: 256^3, 64 candidate poses, 512x512 detector."""
    check_forward_full(dfp, 2, n_check_views=3, band_rows=64, n_grad_views=8)


def test_c3_mcfdk_full(dfp):
    """256^3, 360 ramp-filtered views of 512x384, FDK weight."""
    check_back_full(dfp, 3, n_slabs=3, slab=2, n_grad_views=8)


def test_c4_calibration_full(dfp):
    """512^3, 720 views of 768x768."""
    check_forward_full(dfp, 4, n_check_views=2, band_rows=32, n_grad_views=8)


def test_c5_sweep_full(dfp):
    """512^3, 360 views of 1024x1024: all four calls (the largest config; everything resident at once)."""
    check_forward_full(dfp, 5, n_check_views=2, band_rows=24, n_grad_views=8)
    torch.cuda.empty_cache()
    check_back_full(dfp, 5, n_slabs=2, slab=1, n_grad_views=8)


def test_c2_registration_full_grad_interp_mode(dfp):
    """DFP_FLAG_GRAD_INTERP at full C2 size: eight seeded views' 6-vectors against the oracle's GRAD_INTERP mode."""
    dev = torch.device("cuda:0")
    w = W.make_config(2)
    g = w.geom.replace(flags=dfp.FLAG_GRAD_INTERP)
    a = w.angles.float().numpy()
    p = w.poses.float().numpy()
    vol = w.volume(dev)
    up = w.fwd_upstream(dev)
    grad = dfp.forward_pose_grad(g, a, p, vol, up).cpu().numpy()
    assert dfp.last_path() == dfp.PATH_TMA and np.isfinite(grad).all()
    vol_c = vol.cpu().numpy()
    for v in pick(w.seed + 503, w.n_views, 8):
        o = oracle.forward_pose_grad(w.geom, a[v:v + 1], p[v:v + 1], vol_c, up[v:v + 1].cpu().numpy(),
                                     grad_mode=oracle.GRAD_INTERP)
        e = grad_err_u9(grad[v:v + 1], o)
        assert e.max() <= TOL_GRAD, (v, e)


@pytest.mark.parametrize("model", ["siddon", "joseph"])
def test_c2_registration_full_other_weight_models(dfp, model):
    """DFP_FLAG_SIDDON / DFP_FLAG_JOSEPH at the bench's size: a row band of two seeded views and one view's 6-vector
    vs the oracle."""
    dev = torch.device("cuda:0")
    w = W.make_config(2)
    g = w.geom.replace(flags=dfp.FLAG_SIDDON if model == "siddon" else dfp.FLAG_JOSEPH)
    o_fwd = oracle.forward_siddon if model == "siddon" else oracle.forward_joseph
    o_grad = oracle.forward_pose_grad_siddon if model == "siddon" else oracle.forward_pose_grad_joseph
    a = w.angles.float().numpy()
    p = w.poses.float().numpy()
    vol = w.volume(dev)
    up = w.fwd_upstream(dev)
    proj = dfp.forward(g, a, p, vol)
    grad = dfp.forward_pose_grad(g, a, p, vol, up).cpu().numpy()
    assert torch.isfinite(proj).all() and np.isfinite(grad).all()
    vol_c = vol.cpu().numpy()
    views = pick(w.seed + 601, w.n_views, 2)
    for v in views:
        r0 = pick(w.seed + 611 + v, w.geom.nv - 32 + 1, 1)[0]
        o = o_fwd(row_band(w.geom, r0, 32), a[v:v + 1], p[v:v + 1], vol_c)[0]
        assert rel_l2(proj[v, r0:r0 + 32].cpu().numpy(), o) <= TOL_VAL
    v = views[0]
    o = o_grad(w.geom, a[v:v + 1], p[v:v + 1], vol_c, up[v:v + 1].cpu().numpy())
    assert grad_err_u9(grad[v:v + 1], o).max() <= TOL_GRAD


def test_volume_1024_cubed_indices_and_sizes(dfp):
    """Beyond the configs: a 1024^3 volume (4 GiB) with 2048x2048 views (config 5 at twice the resolution, 4 views) -
    32-bit index arithmetic, tensor-map extents and tile counts at the upper end.  Row bands / one slab vs the oracle."""
    dev = torch.device("cuda:0")
    w = W.make_config(5, scale=2.0, n_views=4)
    g = w.geom
    assert (g.nx, g.nu) == (1024, 2048)
    a = w.angles.float().numpy()
    p = w.poses.float().numpy()
    vol = w.volume(dev)
    vol_c = vol.cpu().numpy()
    v, r0, rows = 2, 1000, 4
    for flags, fwd in ((0, oracle.forward), (dfp.FLAG_SIDDON, oracle.forward_siddon)):
        proj = dfp.forward(g.replace(flags=flags), a, p, vol)
        assert torch.isfinite(proj).all()
        o = fwd(row_band(g, r0, rows), a[v:v + 1], p[v:v + 1], vol_c)[0]
        assert rel_l2(proj[v, r0:r0 + rows].cpu().numpy(), o) <= TOL_VAL
        del proj
    up = w.fwd_upstream(dev)
    grad = dfp.forward_pose_grad(g, a, p, vol, up).cpu().numpy()
    assert dfp.last_path() == dfp.PATH_TMA and np.isfinite(grad).all()
    del vol, up
    torch.cuda.empty_cache()
    pin = w.projections(dev)
    bp = dfp.backproject(g, a, p, pin)
    assert dfp.last_path() == dfp.PATH_TMA
    o = oracle.backproject(g, a, p, pin.cpu().numpy(), 777, 778)
    assert rel_l2(bp[777:778].cpu().numpy(), o) <= TOL_VAL


def test_c2_view_results_do_not_depend_on_the_batch(dfp):
    """Property that holds at any size: views are independent (Eq.18-22 sum over the rays / voxels of ONE
    view), so a view computed alone, in a pair or inside the 64-view batch of config 2 gives the same projection
    bit for bit and the same 6-vectors / moments up to the fp32 order of its block partial sums - whatever staging
    box, chunking or grid the host picks for the batch.  The back-projection is the sum over the batch's views:
    the volume of the whole batch equals the ACCUMULATE-d volumes of its two halves."""
    dev = torch.device("cuda:0")
    w = W.make_config(2)
    g = w.geom
    a = w.angles.float().numpy()
    p = w.poses.float().numpy()
    vol = w.volume(dev)
    up = w.fwd_upstream(dev)
    proj = dfp.forward(g, a, p, vol)
    grad = dfp.forward_pose_grad(g, a, p, vol, up)
    projf, mom = dfp.forward_fused_moments(g, a, p, vol, up)   # two lanes per ray: another fp32 order than `forward`
    assert rel_l2(projf.cpu().numpy(), proj.cpu().numpy()) <= 1e-6
    for sel in ([0], [63], [17, 40], [5, 6, 7]):
        s = np.asarray(sel)
        proj_s = dfp.forward(g, a[s], p[s], vol)
        assert torch.equal(proj_s, proj[s]), sel
        up_s = up[s].contiguous()
        grad_s = dfp.forward_pose_grad(g, a[s], p[s], vol, up_s)
        e = grad_err_u9(grad_s.cpu().numpy(), grad[s].cpu().numpy())
        assert e.max() <= 2e-5, (sel, e)
        proj_f, mom_s = dfp.forward_fused_moments(g, a[s], p[s], vol, up_s)
        assert torch.equal(proj_f, projf[s]), sel
        for k in range(3):
            e = grad_err_u9(mom_s[:, k].cpu().numpy(), mom[s, k].cpu().numpy())
            assert e.max() <= 2e-5, (sel, k, e)
    del proj, projf, up, grad, mom
    # upstream = the voxelised phantom (one sign): with config 2's N(0,1) field a view's 6-vector is the nearly
    # cancelled sum of 1.7e7 random-sign terms and the fp32 rounding of the terms themselves shows at 1e-3 of U9
    bup = vol
    bproj = w.projections(dev)
    bgrad = dfp.backproject_pose_grad(g, a, p, bproj, bup)
    for sel in ([0], [63], [17, 40]):
        s = np.asarray(sel)
        bgrad_s = dfp.backproject_pose_grad(g, a[s], p[s], bproj[s].contiguous(), bup)
        e = grad_err_u9(bgrad_s.cpu().numpy(), bgrad[s].cpu().numpy())
        assert e.max() <= 1e-4, (sel, e)   # small batches get another tile depth / grid: fp32 partials in another order
    whole = dfp.backproject(g, a, p, bproj)
    halves = dfp.backproject(g, a[:32], p[:32], bproj[:32].contiguous())
    ga = g.replace(flags=g.flags | dfp.FLAG_ACCUMULATE)
    dfp.backproject(ga, a[32:], p[32:], bproj[32:].contiguous(), out=halves)
    assert rel_l2(halves.cpu().numpy(), whole.cpu().numpy()) <= 2e-7


@pytest.mark.parametrize("model", ["dd", "sf"])
def test_c2_registration_full_distance_driven(dfp, model):
    """DFP_FLAG_DD / DFP_FLAG_SF at full C2 size (256^3, 64 views of 512x512): a row band of two seeded views, one z-slab
    of the back-projection (all 64 views) and one view's 6-vectors of both gradients against the oracle's O15 / O16."""
    dev = torch.device("cuda:0")
    w = W.make_config(2)
    g0 = w.geom
    g = g0.replace(flags=dfp.FLAG_DD if model == "dd" else dfp.FLAG_SF)
    ora = {k: getattr(oracle, k + "_" + model) for k in ("forward", "forward_pose_grad", "backproject", "backproject_pose_grad")}
    a = w.angles.float().numpy()
    p = w.poses.float().numpy()
    vol = w.volume(dev)
    up = w.fwd_upstream(dev)
    proj = dfp.forward(g, a, p, vol)
    grad = dfp.forward_pose_grad(g, a, p, vol, up).cpu().numpy()
    assert torch.isfinite(proj).all() and np.isfinite(grad).all()
    vol_c = vol.cpu().numpy()
    views = pick(w.seed + 701, w.n_views, 2)
    for v in views:
        r0 = pick(w.seed + 711 + v, g0.nv - 32 + 1, 1)[0]
        o = ora["forward"](row_band(g0, r0, 32), a[v:v + 1], p[v:v + 1], vol_c)[0]
        check_values(proj[v, r0:r0 + 32].cpu().numpy(), o, TOL_VAL, zero_border=True)
    v = views[0]
    o = ora["forward_pose_grad"](g0, a[v:v + 1], p[v:v + 1], vol_c, up[v:v + 1].cpu().numpy())
    e = grad_err_u9(grad[v:v + 1], o)
    report(f"C2 {model} forward_pose_grad, 1 view", e)
    assert e.max() <= TOL_GRAD
    del up, proj
    pin = w.projections(dev)
    bup = w.bp_upstream(dev)
    bp = dfp.backproject(g, a, p, pin)
    bgrad = dfp.backproject_pose_grad(g, a, p, pin, bup).cpu().numpy()
    assert torch.isfinite(bp).all() and np.isfinite(bgrad).all()
    pin_c = pin.cpu().numpy()
    z0 = pick(w.seed + 721, g0.nz - 1, 1)[0]
    o = ora["backproject"](g0, a, p, pin_c, z0, z0 + 1)
    check_values(bp[z0:z0 + 1].cpu().numpy(), o, TOL_VAL, zero_border=False)
    o = ora["backproject_pose_grad"](g0, a[v:v + 1], p[v:v + 1], pin_c[v:v + 1], bup.cpu().numpy())
    e = grad_err_u9(bgrad[v:v + 1], o)
    report(f"C2 {model} backproject_pose_grad, 1 view", e)
    assert e.max() <= TOL_GRAD
