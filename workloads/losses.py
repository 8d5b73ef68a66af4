"""Loss gradients that produce the UPSTREAM arrays fed to the pose-gradient calls.

PAPER.md Eq.20 :185-187 / Eq.22 :200-202: dL/dl^i (resp. dL/dmu^j) "can be easily computed
given a differentiable loss" - it is an input to the method, not part of it.
NCC: Eq.25 :232; image variance / SSD: BASELINE.json configs 3 and 4.  float64 torch.
"""
import torch


def ncc(a: torch.Tensor, b: torch.Tensor) -> torch.Tensor:
    a = a.to(torch.float64).flatten()
    b = b.to(torch.float64).flatten()
    at, bt = a - a.mean(), b - b.mean()
    return (at * bt).sum() / (at.norm() * bt.norm())


def ncc_grad(a: torch.Tensor, b: torch.Tensor) -> torch.Tensor:
    """d NCC(a,b) / d a = bt/(|at||bt|) - NCC * at/|at|^2, at=a-mean(a), bt=b-mean(b)."""
    shp = a.shape
    a = a.to(torch.float64).flatten()
    b = b.to(torch.float64).flatten()
    at, bt = a - a.mean(), b - b.mean()
    na, nb = at.norm(), bt.norm()
    c = (at * bt).sum() / (na * nb)
    return (bt / (na * nb) - c * at / (na * na)).reshape(shp)


def variance_grad(mu: torch.Tensor) -> torch.Tensor:
    """d Var(mu) / d mu_j = 2 (mu_j - mean) / N  (population variance)."""
    m = mu.to(torch.float64)
    return 2.0 * (m - m.mean()) / m.numel()


def ssd_grad(l: torch.Tensor, target: torch.Tensor) -> torch.Tensor:
    """d sum (l - target)^2 / d l = 2 (l - target)."""
    return 2.0 * (l.to(torch.float64) - target.to(torch.float64))


def gradient_entropy(mu: torch.Tensor) -> torch.Tensor:
    """Gradient entropy of a volume, the sharpness criterion of the paper's motion-compensated reconstruction
    (Eq.26 :239, "as in [9]"): with g_j = |forward finite-difference gradient of mu at voxel j| and
    p_j = g_j / sum g, GE = -sum_j p_j log p_j (smaller = sharper).  Differentiable torch code: its autograd gradient
    dGE/dmu is the UPSTREAM array of dfp_backproject_pose_grad - an input of the method, not part of it."""
    m = mu.to(torch.float64)
    gx = m[:-1, :-1, 1:] - m[:-1, :-1, :-1]
    gy = m[:-1, 1:, :-1] - m[:-1, :-1, :-1]
    gz = m[1:, :-1, :-1] - m[:-1, :-1, :-1]
    g = torch.sqrt(gx * gx + gy * gy + gz * gz + 1e-12)
    p = g / g.sum()
    return -(p * torch.log(p + 1e-30)).sum()
