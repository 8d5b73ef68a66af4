"""The five BASELINE.json workloads as seeded synthetic inputs (recipe: DESIGN.md §"Input recipe").

The paper's registration / motion-compensation / calibration studies use a CQ500 head CT and two
real bench scans (PAPER.md :211, :228, :237, :244).  None of those is available; seeded ellipsoid
phantoms of the same shapes (Table II :246-257, BASELINE.json `configs`) stand in.

`make_config(i, scale=s, n_views=V)` returns a `Workload`.  `scale` < 1 shrinks every grid
(voxel and pixel counts x s, pitches / s, so physical extents and the cone stay the same) and
`n_views` overrides the view count: these give the reduced cases the fp64 oracle finishes in seconds.
Every large array is produced lazily, on the device asked for, as float32 - the same bits are then
handed to the oracle and to the CUDA path.
"""
import dataclasses
import math
from typing import List, Optional, Sequence

import torch

from .geometry import Geometry, view_angles
from .losses import ncc_grad, ssd_grad, variance_grad
from .phantom import (Ellipsoid, ellipsoid_projection, random_ellipsoids, voxelise_ellipsoids)
from .ramp import ramp_filter
from .rng import SplitMix64, normal_field

DEG = math.pi / 180.0


def base_seed(index: int) -> int:
    return 250813304 * 10 + index


CONFIGS = {
    1: dict(name="C1-tiny", n=64, voxel=0.5, nu=64, nv=64, pix=1.0, sad=600.0, sdd=1000.0, views=1, arc=0.0,
            n_ell=8, semi=(3.0, 12.0), dens=(0.01, 0.04), pose_t=5.0, pose_r=3.0,
            calls=("forward", "forward_pose_grad")),
    2: dict(name="C2-registration", n=256, voxel=1.0, nu=512, nv=512, pix=0.6, sad=785.0, sdd=1200.0, views=64,
            arc=0.0, n_ell=40, semi=(8.0, 40.0), dens=(0.0, 0.05), pose_t=20.0, pose_r=10.0,
            calls=("forward", "forward_pose_grad")),
    3: dict(name="C3-mcfdk", n=256, voxel=0.75, nu=512, nv=384, pix=0.776, sad=785.0, sdd=1200.0, views=360,
            arc=360.0, n_ell=30, semi=(5.0, 30.0), dens=(0.0, 0.05), pose_t=4.0, pose_r=2.0,
            calls=("backproject", "backproject_pose_grad")),
    4: dict(name="C4-calibration", n=512, voxel=0.5, nu=768, nv=768, pix=0.388, sad=785.0, sdd=1200.0, views=720,
            arc=360.0, n_ell=40, semi=(5.0, 40.0), dens=(0.0, 0.05), pose_t=2.0, pose_r=1.0,
            n_spheres=20, sphere_r=(1.0, 2.0), sphere_dens=0.2,
            calls=("forward", "forward_pose_grad")),
    5: dict(name="C5-sweep", n=512, voxel=0.5, nu=1024, nv=1024, pix=0.388, sad=785.0, sdd=1200.0, views=360,
            arc=360.0, n_ell=40, semi=(8.0, 40.0), dens=(0.0, 0.05), pose_t=10.0, pose_r=5.0,
            calls=("forward", "forward_pose_grad", "backproject", "backproject_pose_grad")),
}


@dataclasses.dataclass
class Workload:
    index: int
    name: str
    geom: Geometry
    angles: torch.Tensor            # [V] float64 rad
    poses: torch.Tensor             # [V,6] float64 (mm, rad): the poses the calls are evaluated at
    data_poses: torch.Tensor        # [V,6] float64: the poses the measured/target data were generated at
    ells: List[Ellipsoid]
    calls: Sequence[str]
    seed: int

    @property
    def n_views(self) -> int:
        return int(self.angles.numel())

    # ---- large arrays, generated on demand ------------------------------------------------------
    def volume(self, device="cpu") -> torch.Tensor:
        """vol[iz][iy][ix] float32: the voxelised ellipsoid phantom."""
        return voxelise_ellipsoids(self.geom, self.ells, device)

    def _views(self, views):
        return range(self.n_views) if views is None else list(views)

    def closed_form(self, poses: torch.Tensor, device="cpu", views=None) -> torch.Tensor:
        """[len(views), nv, nu] float64 exact ellipsoid line integrals at `poses`."""
        vs = self._views(views)
        out = torch.empty((len(vs),) + self.geom.det_shape, dtype=torch.float64, device=device)
        for o, v in enumerate(vs):
            out[o] = ellipsoid_projection(self.geom, self.ells, float(self.angles[v]), poses[v].tolist(), device)
        return out

    def fwd_upstream(self, device="cpu", views=None) -> torch.Tensor:
        """dL/dl for `forward_pose_grad`, [len(views), nv, nu] float32.
        C1, C5: N(0,1).  C2: d NCC(l, target)/dl.  C4: 2 (l - target).  In C2/C4 `l` is the closed-form
        projection at the evaluated pose (a stand-in for the discrete forward projection, so that the
        array depends on neither implementation) and target the closed-form projection at `data_poses`."""
        vs = self._views(views)
        nv, nu = self.geom.det_shape
        if self.index in (2, 4):
            out = torch.empty((len(vs), nv, nu), dtype=torch.float32, device=device)
            for o, v in enumerate(vs):
                l = self.closed_form(self.poses, device, [v])[0]
                tgt = self.closed_form(self.data_poses, device, [v])[0]
                g = ncc_grad(l, tgt) if self.index == 2 else ssd_grad(l, tgt)
                out[o] = g.to(torch.float32)
            return out
        out = torch.empty((len(vs), nv, nu), dtype=torch.float32, device=device)
        for o, v in enumerate(vs):
            out[o] = normal_field(self.seed * 4096 + 17 + v, nv * nu, device).reshape(nv, nu)
        return out

    def projections(self, device="cpu", views=None) -> torch.Tensor:
        """Input of `backproject`, [len(views), nv, nu] float32: closed-form projections at `data_poses`
        (the object as it really moved); ramp-filtered along u for C3 (FDK input)."""
        p = self.closed_form(self.data_poses, device, views)
        if self.index == 3:
            p = ramp_filter(p, self.geom.du)
        return p.to(torch.float32)

    def bp_upstream(self, device="cpu") -> torch.Tensor:
        """dL/dmu for `backproject_pose_grad`, [nz,ny,nx] float32.
        C3: image-variance gradient 2(mu - mean)/N evaluated on the voxelised phantom (a stand-in for
        the reconstruction, so that the array depends on neither implementation).  Others: N(0,1)."""
        if self.index == 3:
            return variance_grad(self.volume(device)).to(torch.float32)
        g = self.geom
        return normal_field(self.seed * 4096 + 5, g.nx * g.ny * g.nz, device).reshape(g.vol_shape)


def _draw_pose(rng: SplitMix64, t_mm: float, r_deg: float):
    return [rng.uniform(-t_mm, t_mm) for _ in range(3)] + [rng.uniform(-r_deg, r_deg) * DEG for _ in range(3)]


def make_config(index: int, scale: float = 1.0, n_views: Optional[int] = None) -> Workload:
    c = CONFIGS[index]
    seed = base_seed(index)
    rng = SplitMix64(seed)

    def sc(n):
        return max(4, int(round(n * scale)))
    n = sc(c["n"])
    nu, nv = sc(c["nu"]), sc(c["nv"])
    voxel = c["voxel"] * c["n"] / n
    du = c["pix"] * c["nu"] / nu
    dv = c["pix"] * c["nv"] / nv
    geom = Geometry(nx=n, ny=n, nz=n, vx=voxel, vy=voxel, vz=voxel, nu=nu, nv=nv, du=du, dv=dv,
                    sad=c["sad"], sdd=c["sdd"], bp_weight=1 if index == 3 else 0).f32()
    half = 0.5 * c["n"] * c["voxel"]
    # 1) phantom (always drawn at full-resolution margins so every scale shows the same object)
    ells = random_ellipsoids(rng, c["n_ell"], c["semi"], c["dens"], half, 2.0 * c["voxel"])
    if "n_spheres" in c:
        ells += random_ellipsoids(rng, c["n_spheres"], c["sphere_r"], (c["sphere_dens"], c["sphere_dens"]),
                                  half, 2.0 * c["voxel"], spheres=True)
    # 2) views
    V_full = c["views"]
    V = V_full if n_views is None else n_views
    angles = view_angles(V, c["arc"]) if c["arc"] > 0 else torch.zeros(V, dtype=torch.float64)
    # 3) poses
    if index == 3:
        # smooth per-view motion theta*_v[k] = A_k sin(2 pi f_k v/V + phi_k); evaluated at half of it
        A = [rng.uniform(0.5, 1.0) * c["pose_t"] for _ in range(3)] + \
            [rng.uniform(0.5, 1.0) * c["pose_r"] * DEG for _ in range(3)]
        f = [1 + int(rng.uniform(0.0, 3.0)) for _ in range(6)]
        ph = [rng.uniform(0.0, 2.0 * math.pi) for _ in range(6)]
        v = torch.arange(V, dtype=torch.float64)
        data_poses = torch.stack([A[k] * torch.sin(2.0 * math.pi * f[k] * v / V + ph[k]) for k in range(6)], dim=1)
        poses = 0.5 * data_poses
    elif index == 4:
        data_poses = torch.tensor([_draw_pose(rng, c["pose_t"], c["pose_r"]) for _ in range(V)], dtype=torch.float64)
        poses = 0.5 * data_poses
    elif index == 2:
        hidden = _draw_pose(rng, c["pose_t"], c["pose_r"])
        poses = torch.tensor([_draw_pose(rng, c["pose_t"], c["pose_r"]) for _ in range(V)], dtype=torch.float64)
        data_poses = torch.tensor([hidden] * V, dtype=torch.float64)
    else:
        poses = torch.tensor([_draw_pose(rng, c["pose_t"], c["pose_r"]) for _ in range(V)], dtype=torch.float64)
        data_poses = poses.clone()
    return Workload(index=index, name=c["name"], geom=geom, angles=angles, poses=poses, data_poses=data_poses,
                    ells=ells, calls=c["calls"], seed=seed)
