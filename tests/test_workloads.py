"""Pins for the seeded input generators (workloads/): RNG, loss gradients that produce the upstream arrays,
config recipe.  CPU only; nothing here touches the method's arithmetic."""
import math

import numpy as np
import torch

import workloads as W


def test_splitmix64_reference_stream():
    # first outputs of the public-domain SplitMix64 reference generator for seed 0
    r = W.SplitMix64(0)
    assert [r.next_u64() for _ in range(3)] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]


def test_counter_based_fields_are_reproducible_chunk_independent_and_standard():
    a = W.normal_field(123, 200_000)
    b = W.normal_field(123, 200_000, chunk=777)
    assert torch.equal(a, b)
    assert abs(float(a.mean())) < 0.01 and abs(float(a.std()) - 1.0) < 0.01
    u = W.uniform_field(5, 100_000, lo=-2.0, hi=3.0)
    assert float(u.min()) >= -2.0 and float(u.max()) <= 3.0 and abs(float(u.mean()) - 0.5) < 0.02
    assert not torch.equal(W.normal_field(124, 1000), a[:1000])


def _fd(f, x, eps=1e-6):
    g = torch.zeros_like(x)
    flat = x.flatten()
    for i in range(flat.numel()):
        xp, xm = flat.clone(), flat.clone()
        xp[i] += eps
        xm[i] -= eps
        g.view(-1)[i] = (f(xp.view_as(x)) - f(xm.view_as(x))) / (2 * eps)
    return g


def test_loss_gradients_match_finite_differences():
    torch.manual_seed(0)
    a = torch.randn(5, 7, dtype=torch.float64)
    b = torch.randn(5, 7, dtype=torch.float64)
    assert (W.ncc_grad(a, b) - _fd(lambda x: W.ncc(x, b), a)).abs().max() < 1e-8
    assert (W.variance_grad(a) - _fd(lambda x: x.var(unbiased=False), a)).abs().max() < 1e-8
    assert (W.ssd_grad(a, b) - _fd(lambda x: ((x - b) ** 2).sum(), a)).abs().max() < 1e-7
    assert abs(float(W.ncc(a, 3 * a + 2)) - 1.0) < 1e-12


def test_ramp_filter_kills_dc_and_has_the_ramp_spectrum():
    # a constant row filtered with the (truncated) Ram-Lak kernel is ~0 away from the ends; a cosine of
    # frequency f is scaled by |f| (textbook property of the ramp filter), here f = 8 cycles / 256 samples
    nu, du = 256, 0.8
    x = torch.arange(nu, dtype=torch.float64)
    row = torch.cos(2 * math.pi * 8 * x / nu)[None]
    out = W.ramp_filter(row, du)[0, 96:160]
    f = 8 / (nu * du)
    assert (out - f * row[0, 96:160]).abs().max() < 0.03 * f
    const = W.ramp_filter(torch.ones(1, nu, dtype=torch.float64), du)[0, 96:160]
    assert const.abs().max() < 0.05 * f      # truncation tail of the 1/n^2 kernel


def test_config_recipe_shapes_and_determinism():
    for i, (n, nu, nv, V) in {1: (64, 64, 64, 1), 2: (256, 512, 512, 64), 3: (256, 512, 384, 360),
                              4: (512, 768, 768, 720), 5: (512, 1024, 1024, 360)}.items():
        w = W.make_config(i)
        assert (w.geom.nx, w.geom.nu, w.geom.nv, w.n_views) == (n, nu, nv, V)
        assert w.poses.shape == (V, 6) and w.seed == 250813304 * 10 + i
        w2 = W.make_config(i)
        assert torch.equal(w.poses, w2.poses) and [e.centre for e in w.ells] == [e.centre for e in w2.ells]
    w = W.make_config(2, scale=0.125, n_views=3)
    assert w.geom.nx == 32 and w.geom.nu == 64 and w.n_views == 3 and abs(w.geom.vx - 8.0) < 1e-12
    vol = w.volume()
    assert vol.dtype == torch.float32 and vol.shape == (32, 32, 32) and float(vol.max()) > 0
    up = w.fwd_upstream()
    assert up.shape == (3, 64, 64) and up.dtype == torch.float32
    w3 = W.make_config(3, scale=0.125, n_views=6)
    assert w3.geom.bp_weight == 1 and w3.projections().shape == (6, 48, 64) and w3.bp_upstream().shape == (32, 32, 32)
