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
