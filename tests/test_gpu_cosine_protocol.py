"""The paper's accuracy protocol (PAPER.md :211-222, Eq.23-24) on the CUDA path (`-m gpu`): cosine similarity between
the analytical pose gradient and central finite differences of the loss through the library's OWN projector /
back-projector, L2 losses, random rigid motions (sigma 20 mm / 10 degrees scaled to the phantom), on the seeded
synthetic phantoms that stand in for CQ500.  The paper reports means of 0.9952 (forward) and
0.9984 (back, voxel-driven); the oracle's own pins assert >= 0.995 in fp64 - here the same level is asked of the
fp32 kernels end to end through the C ABI, in the paper's (central-difference) mode and in GRAD_INTERP mode."""
import math

import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu
DEG = math.pi / 180.0


def cos_sim(a, b):
    return float(np.dot(a, b) / (np.linalg.norm(a) * np.linalg.norm(b)))


def fd_grad(loss, theta, eps):
    g = np.zeros(6)
    for k in range(6):
        tp, tm = theta.copy(), theta.copy()
        tp[k] += eps[k]
        tm[k] -= eps[k]
        g[k] = (loss(tp) - loss(tm)) / (2 * eps[k])
    return g


@pytest.mark.parametrize("mode", ["central", "interp"])
def test_forward_gradient_cosine_similarity(mode):
    import paper_2508_13304_b200 as dfp
    dev = torch.device("cuda:0")
    w = W.make_config(2, scale=0.5, n_views=1)
    g = w.geom.replace(flags=dfp.FLAG_GRAD_INTERP if mode == "interp" else 0)
    vol = w.volume(dev)
    rng = np.random.default_rng(24)
    eps = np.array([0.05, 0.05, 0.05, 2e-4, 2e-4, 2e-4])
    sims = []
    for trial in range(6):
        beta = np.array([rng.uniform(0, math.pi / 2)], np.float32)                  # views over 0-90 degrees (:211)
        target = dfp.forward(g, beta, np.zeros((1, 6), np.float32), vol).double()   # the measurement: no motion
        theta = np.concatenate([rng.normal(0, 6.0, 3), rng.normal(0, 4.0 * DEG, 3)])

        def loss(t):
            l = dfp.forward(g, beta, t[None].astype(np.float32), vol).double()
            return float(((l - target) ** 2).sum())                                 # Eq.23a

        l = dfp.forward(g, beta, theta[None].astype(np.float32), vol)
        up = (2.0 * (l.double() - target)).float().contiguous()
        ana = dfp.forward_pose_grad(g, beta, theta[None].astype(np.float32), vol, up)[0].double().cpu().numpy()
        sims.append(cos_sim(ana, fd_grad(loss, theta, eps)))
    assert np.mean(sims) >= 0.995 and min(sims) >= 0.98, sims


@pytest.mark.parametrize("mode", ["central", "interp"])
def test_backprojection_gradient_cosine_similarity(mode):
    import paper_2508_13304_b200 as dfp
    dev = torch.device("cuda:0")
    w = W.make_config(3, scale=0.25, n_views=8)
    g = w.geom.replace(bp_weight=0, flags=dfp.FLAG_GRAD_INTERP if mode == "interp" else 0)
    a = w.angles.float().numpy()
    # smooth (unfiltered) closed-form projections: the paper's Eq.23b compares back-projections, no ramp filter
    proj = w.closed_form(w.data_poses, dev).float().contiguous()
    mu0 = dfp.backproject(g, a, np.zeros((8, 6), np.float32), proj).double()
    rng = np.random.default_rng(25)
    eps = np.array([0.05, 0.05, 0.05, 2e-4, 2e-4, 2e-4])
    sims = []
    for trial in range(4):
        poses = np.concatenate([rng.normal(0, 3.0, (8, 3)), rng.normal(0, 2.0 * DEG, (8, 3))], axis=1)
        v = int(rng.integers(0, 8))

        def loss(t):
            p = poses.copy()
            p[v] = t
            mu = dfp.backproject(g, a, p.astype(np.float32), proj).double()
            return float(((mu - mu0) ** 2).sum())                                   # Eq.23b

        mu = dfp.backproject(g, a, poses.astype(np.float32), proj)
        up = (2.0 * (mu.double() - mu0)).float().contiguous()
        ana = dfp.backproject_pose_grad(g, a, poses.astype(np.float32), proj, up)[v].double().cpu().numpy()
        sims.append(cos_sim(ana, fd_grad(loss, poses[v], eps)))
    assert np.mean(sims) >= 0.995 and min(sims) >= 0.98, sims
