"""Ram-Lak ramp filter along detector rows (input preparation for config 3; Eq.26 :239-242,
"Ramp represents the standard ramp filtering for tomographic reconstruction").
Spatial kernel (pitch du): h[0]=1/(4 du^2), h[n odd]=-1/(pi n du)^2, h[n even]=0; output = du * (l * h) along u.
"""
import math

import torch


def ramp_filter(proj: torch.Tensor, du: float) -> torch.Tensor:
    """proj [..., nv, nu] -> same shape, float64, linear (zero-padded) convolution via FFT."""
    p = proj.to(torch.float64)
    nu = p.shape[-1]
    n = torch.arange(-(nu - 1), nu, dtype=torch.float64, device=p.device)
    h = torch.zeros_like(n)
    odd = (n.abs().to(torch.int64) % 2) == 1
    h[odd] = -1.0 / (math.pi * n[odd] * du) ** 2
    h[nu - 1] = 1.0 / (4.0 * du * du)
    L = 1
    while L < 3 * nu:
        L *= 2
    H = torch.fft.rfft(h, n=L)
    P = torch.fft.rfft(p, n=L, dim=-1)
    full = torch.fft.irfft(P * H, n=L, dim=-1)
    return du * full[..., nu - 1: 2 * nu - 1]
