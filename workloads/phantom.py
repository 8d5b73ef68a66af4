"""Seeded ellipsoid / Gaussian-blob phantoms and their CLOSED-FORM cone-beam line integrals.

The closed forms are textbook analytic geometry (chord of a line through an ellipsoid;
line integral of an anisotropic Gaussian), not the paper's discrete method.  They serve two
roles: rendering target / measured data for the configs ("targets are rendered
with the closed-form ellipsoid projector, independent of both implementations"), and pinning
the oracle's forward projector in tests (north_star: "closed-form line integrals of ellipsoid
phantoms").  Scanner convention (Table I :27-42):
  view angle b: n=(cos b, sin b, 0); source s=SAD*n; detector centre -(SDD-SAD)*n;
  e_u=(-sin b, cos b, 0); e_v=(0,0,1); pixel (iu,iv) at centre + (iu-c_u)du e_u + (iv-c_v)dv e_v;
  pose theta=(tx,ty,tz,gx,gy,gz): r = R r' + t, R = Rz(gz) Ry(gy) Rx(gx).
All maths in float64 torch (any device).
"""
import dataclasses
import math
from typing import List, Sequence

import torch

from .geometry import Geometry
from .rng import SplitMix64


def rotation_zyx(gx: float, gy: float, gz: float, device="cpu") -> torch.Tensor:
    """R = Rz(gz) Ry(gy) Rx(gx), right-handed basic rotations, float64 3x3."""
    cx, sx = math.cos(gx), math.sin(gx)
    cy, sy = math.cos(gy), math.sin(gy)
    cz, sz = math.cos(gz), math.sin(gz)
    Rx = torch.tensor([[1, 0, 0], [0, cx, -sx], [0, sx, cx]], dtype=torch.float64)
    Ry = torch.tensor([[cy, 0, sy], [0, 1, 0], [-sy, 0, cy]], dtype=torch.float64)
    Rz = torch.tensor([[cz, -sz, 0], [sz, cz, 0], [0, 0, 1]], dtype=torch.float64)
    return (Rz @ Ry @ Rx).to(device)


@dataclasses.dataclass
class Ellipsoid:
    centre: Sequence[float]     # mm, object frame
    semi_axes: Sequence[float]  # mm (for blobs: the three standard deviations)
    euler: Sequence[float]      # orientation Q = Rz Ry Rx of these three angles (rad)
    density: float              # 1/mm (for blobs: peak amplitude)

    def Q(self, device="cpu"):
        return rotation_zyx(*self.euler, device=device)


def random_ellipsoids(rng: SplitMix64, n: int, semi_range, density_range, half_extent_mm: float,
                      margin_mm: float, spheres: bool = False) -> List[Ellipsoid]:
    """Draw order per ellipsoid (fixed, documented in DESIGN.md): a1,a2,a3, density, cx,cy,cz, e1,e2,e3.
    Centres are uniform in the cube that keeps the bounding sphere `margin_mm` inside the volume."""
    out = []
    for _ in range(n):
        a = [rng.uniform(*semi_range) for _ in range(3)]
        if spheres:
            a = [a[0]] * 3
        rho = rng.uniform(*density_range)
        lim = max(0.0, half_extent_mm - max(a) - margin_mm)
        c = [rng.uniform(-lim, lim) for _ in range(3)]
        e = [rng.uniform(-math.pi, math.pi) for _ in range(3)]
        out.append(Ellipsoid(c, a, e, rho))
    return out


def _axis_mm(n, v, c, device):
    return c + (torch.arange(n, dtype=torch.float64, device=device) - (n - 1) / 2.0) * v


def voxelise_ellipsoids(geom: Geometry, ells: Sequence[Ellipsoid], device="cpu") -> torch.Tensor:
    """vol[iz][iy][ix] (float32) = sum of densities of ellipsoids containing the voxel CENTRE."""
    vol = torch.zeros(geom.vol_shape, dtype=torch.float64, device=device)
    xs = _axis_mm(geom.nx, geom.vx, geom.cx, device)
    ys = _axis_mm(geom.ny, geom.vy, geom.cy, device)
    zs = _axis_mm(geom.nz, geom.vz, geom.cz, device)
    for e in ells:
        rmax = max(e.semi_axes)
        c = e.centre

        def rng_idx(ax, cc, n):
            lo = int(torch.searchsorted(ax, torch.tensor(cc - rmax, dtype=torch.float64, device=device)).item())
            hi = int(torch.searchsorted(ax, torch.tensor(cc + rmax, dtype=torch.float64, device=device), right=True).item())
            return max(0, lo), min(n, hi)
        x0, x1 = rng_idx(xs, c[0], geom.nx)
        y0, y1 = rng_idx(ys, c[1], geom.ny)
        z0, z1 = rng_idx(zs, c[2], geom.nz)
        if x1 <= x0 or y1 <= y0 or z1 <= z0:
            continue
        Z, Y, X = torch.meshgrid(zs[z0:z1] - c[2], ys[y0:y1] - c[1], xs[x0:x1] - c[0], indexing="ij")
        Q = e.Q(device)
        a = torch.tensor(e.semi_axes, dtype=torch.float64, device=device)
        # local = Q^T (r' - c), scaled by 1/a
        l0 = (Q[0, 0] * X + Q[1, 0] * Y + Q[2, 0] * Z) / a[0]
        l1 = (Q[0, 1] * X + Q[1, 1] * Y + Q[2, 1] * Z) / a[1]
        l2 = (Q[0, 2] * X + Q[1, 2] * Y + Q[2, 2] * Z) / a[2]
        inside = (l0 * l0 + l1 * l1 + l2 * l2) <= 1.0
        vol[z0:z1, y0:y1, x0:x1] += e.density * inside.to(torch.float64)
    return vol.to(torch.float32)


def voxelise_blobs(geom: Geometry, blobs: Sequence[Ellipsoid], device="cpu") -> torch.Tensor:
    """vol = sum_b a_b exp(-0.5 |D^-1 Q^T (r'-c)|^2) sampled at voxel centres, float32."""
    xs = _axis_mm(geom.nx, geom.vx, geom.cx, device)
    ys = _axis_mm(geom.ny, geom.vy, geom.cy, device)
    zs = _axis_mm(geom.nz, geom.vz, geom.cz, device)
    Z, Y, X = torch.meshgrid(zs, ys, xs, indexing="ij")
    vol = torch.zeros(geom.vol_shape, dtype=torch.float64, device=device)
    for b in blobs:
        Q = b.Q(device)
        s = torch.tensor(b.semi_axes, dtype=torch.float64, device=device)
        x, y, z = X - b.centre[0], Y - b.centre[1], Z - b.centre[2]
        l0 = (Q[0, 0] * x + Q[1, 0] * y + Q[2, 0] * z) / s[0]
        l1 = (Q[0, 1] * x + Q[1, 1] * y + Q[2, 1] * z) / s[1]
        l2 = (Q[0, 2] * x + Q[1, 2] * y + Q[2, 2] * z) / s[2]
        vol += b.density * torch.exp(-0.5 * (l0 * l0 + l1 * l1 + l2 * l2))
    return vol.to(torch.float32)


def _object_frame_rays(geom: Geometry, angle, pose, device, rows=None):
    """Source position s' [3] and unit directions e' [nrows,nu,3] in the OBJECT frame for one view.
    `angle`: a gantry angle (circular orbit) or a 12-number view frame (s, c, U, V; workloads.circular_frame)."""
    pose = [float(p) for p in pose]
    R = rotation_zyx(pose[3], pose[4], pose[5], device)
    t = torch.tensor(pose[:3], dtype=torch.float64, device=device)
    cu = (geom.nu - 1) / 2.0 + geom.u0
    cv = (geom.nv - 1) / 2.0 + geom.v0
    iu = torch.arange(geom.nu, dtype=torch.float64, device=device)
    iv = torch.arange(geom.nv, dtype=torch.float64, device=device) if rows is None else \
        torch.as_tensor(rows, dtype=torch.float64, device=device)
    if not isinstance(angle, (int, float)) and len(torch.as_tensor(angle).reshape(-1)) == 12:
        f = torch.as_tensor(angle, dtype=torch.float64, device=device).reshape(4, 3)
        s, dc = f[0], f[1]
        pix = dc[None, None, :] + (iu - cu)[None, :, None] * f[2] + (iv - cv)[:, None, None] * f[3]
    else:
        angle = float(angle)
        cb, sb = math.cos(angle), math.sin(angle)
        n = torch.tensor([cb, sb, 0.0], dtype=torch.float64, device=device)
        eu = torch.tensor([-sb, cb, 0.0], dtype=torch.float64, device=device)
        ev = torch.tensor([0.0, 0.0, 1.0], dtype=torch.float64, device=device)
        s = geom.sad * n
        dc = -(geom.sdd - geom.sad) * n
        pix = dc[None, None, :] + ((iu - cu) * geom.du)[None, :, None] * eu + \
            ((iv - cv) * geom.dv)[:, None, None] * ev
    d = pix - s
    e = d / torch.linalg.norm(d, dim=-1, keepdim=True)
    s_obj = R.T @ (s - t)
    e_obj = e @ R          # row-vector form of R^T e
    return s_obj, e_obj


def ellipsoid_projection(geom: Geometry, ells: Sequence[Ellipsoid], angle: float, pose, device="cpu",
                         rows=None) -> torch.Tensor:
    """Exact line integrals [nv,nu] (float64) of the ellipsoid phantom for one view.
    Ray s'+tau e' in the object frame; p=D^-1 Q^T (s'-c), q=D^-1 Q^T e';
    chord = 2 sqrt((p.q)^2 - (q.q)(p.p-1)) / (q.q) when the radicand is positive."""
    s_obj, e_obj = _object_frame_rays(geom, angle, pose, device, rows)
    out = torch.zeros(e_obj.shape[:2], dtype=torch.float64, device=device)
    for e in ells:
        Q = e.Q(device)
        a = torch.tensor(e.semi_axes, dtype=torch.float64, device=device)
        c = torch.tensor(e.centre, dtype=torch.float64, device=device)
        p = (Q.T @ (s_obj - c)) / a
        q = (e_obj @ Q) / a
        pq = (q * p).sum(-1)
        qq = (q * q).sum(-1)
        pp = (p * p).sum()
        rad = pq * pq - qq * (pp - 1.0)
        out += e.density * 2.0 * torch.sqrt(torch.clamp(rad, min=0.0)) / qq
    return out


def blob_projection(geom: Geometry, blobs: Sequence[Ellipsoid], angle: float, pose, device="cpu") -> torch.Tensor:
    """Exact line integrals of sum_b a exp(-0.5|D^-1 Q^T (r'-c)|^2):
    a sqrt(2 pi/(q.q)) exp(-0.5 (p.p - (p.q)^2/(q.q))) with p, q as above."""
    s_obj, e_obj = _object_frame_rays(geom, angle, pose, device)
    out = torch.zeros(e_obj.shape[:2], dtype=torch.float64, device=device)
    for b in blobs:
        Q = b.Q(device)
        sg = torch.tensor(b.semi_axes, dtype=torch.float64, device=device)
        c = torch.tensor(b.centre, dtype=torch.float64, device=device)
        p = (Q.T @ (s_obj - c)) / sg
        q = (e_obj @ Q) / sg
        pq = (q * p).sum(-1)
        qq = (q * q).sum(-1)
        pp = (p * p).sum()
        out += b.density * torch.sqrt(2.0 * math.pi / qq) * torch.exp(-0.5 * (pp - pq * pq / qq))
    return out
