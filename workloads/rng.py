"""Portable seeded random numbers.

`SplitMix64` is the sequential generator used for the few hundred scalar draws of a
config (ellipsoid parameters, poses).  `uniform_field` / `normal_field` are
counter-based (value i depends only on (seed, i)), written with torch integer ops so
that a 4e8-element upstream array can be generated on whatever device holds it; the
integer part is bit-exact across devices, and the array that results is handed
unchanged to both the oracle and the CUDA path.
"""
import math

import torch

_MASK = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB


class SplitMix64:
    def __init__(self, seed: int):
        self.s = seed & _MASK

    def next_u64(self) -> int:
        self.s = (self.s + _GOLDEN) & _MASK
        z = self.s
        z = ((z ^ (z >> 30)) * _M1) & _MASK
        z = ((z ^ (z >> 27)) * _M2) & _MASK
        return z ^ (z >> 31)

    def uniform(self, a: float = 0.0, b: float = 1.0) -> float:
        return a + (b - a) * ((self.next_u64() >> 11) * 2.0 ** -53)

    def normal(self) -> float:
        u1 = 1.0 - self.uniform()
        u2 = self.uniform()
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)

    def fork(self) -> "SplitMix64":
        return SplitMix64(self.next_u64())


def _s64(x: int) -> int:
    """Python int (mod 2^64) -> the signed value torch.int64 holds for those bits."""
    x &= _MASK
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right on int64 bit patterns."""
    return (z >> k) & ((1 << (64 - k)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _s64(_M1)
    z = (z ^ _lsr(z, 27)) * _s64(_M2)
    return z ^ _lsr(z, 31)


def _u01(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    base = _s64(seed * 0xD1342543DE82EF95 + stream * 0xA0761D6478BD642F + 1)
    z = _mix(idx * _s64(_GOLDEN) + base)
    return _lsr(z, 11).to(torch.float64) * 2.0 ** -53


def uniform_field(seed: int, n: int, device="cpu", lo=0.0, hi=1.0, dtype=torch.float32, chunk=1 << 24):
    out = torch.empty(n, dtype=dtype, device=device)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        idx = torch.arange(a, b, dtype=torch.int64, device=device)
        out[a:b] = (lo + (hi - lo) * _u01(seed, 0, idx)).to(dtype)
    return out


def normal_field(seed: int, n: int, device="cpu", dtype=torch.float32, chunk=1 << 24):
    """N(0,1) by Box-Muller from two counter-based uniform streams."""
    out = torch.empty(n, dtype=dtype, device=device)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        idx = torch.arange(a, b, dtype=torch.int64, device=device)
        u1 = 1.0 - _u01(seed, 1, idx)
        u2 = _u01(seed, 2, idx)
        out[a:b] = (torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)).to(dtype)
    return out
