"""Scanner / grid description as plain numbers (the fields of `dfp_geometry`, include/dfp.h).

No projector arithmetic lives here: each implementation (oracle, CUDA host code,
closed-form renderer) builds its own rays and matrices from these numbers.
"""
import dataclasses
import math

import torch


@dataclasses.dataclass
class Geometry:
    nx: int
    ny: int
    nz: int
    vx: float
    vy: float
    vz: float
    nu: int
    nv: int
    du: float
    dv: float
    sad: float
    sdd: float
    cx: float = 0.0
    cy: float = 0.0
    cz: float = 0.0
    u0: float = 0.0
    v0: float = 0.0
    step_mm: float = 0.0      # <=0: min(vx,vy,vz)
    bp_weight: int = 0        # 0 unit, 1 FDK (sad/w')^2
    flags: int = 0            # bit0: add dW/dtheta term in backproject_pose_grad; bit6 (64): views are 12-number frames

    def replace(self, **kw) -> "Geometry":
        return dataclasses.replace(self, **kw)

    def f32(self) -> "Geometry":
        """The same scanner with every real number rounded to float32 - the precision of `dfp_geometry` (the C ABI takes
        fp32).  Workloads are emitted this way so that the oracle (fp64 fields) and the CUDA path see the SAME numbers:
        a pitch such as 0.388 mm otherwise differs by 3e-8 relative between the two, which moves a ray by ~1e-5 voxel."""
        import numpy as np
        kw = {f.name: float(np.float32(getattr(self, f.name))) for f in dataclasses.fields(self) if f.type is float}
        return dataclasses.replace(self, **kw)

    def as_dict(self) -> dict:
        return dataclasses.asdict(self)

    @property
    def step(self) -> float:
        return self.step_mm if self.step_mm > 0 else min(self.vx, self.vy, self.vz)

    @property
    def vol_shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def det_shape(self):
        return (self.nv, self.nu)


def view_angles(n_views: int, arc_deg: float = 360.0, start_deg: float = 0.0) -> torch.Tensor:
    """Gantry angles in radians, evenly spaced over `arc_deg` (end point excluded), float64."""
    k = torch.arange(n_views, dtype=torch.float64)
    return (start_deg + arc_deg * k / n_views) * (math.pi / 180.0)


FLAG_VIEW_FRAMES = 64   # dfp_geometry.flags bit6: the view array holds [V][12] frames instead of [V] gantry angles


def circular_frame(geom: Geometry, angle: float) -> torch.Tensor:
    """The 12 numbers (source s, detector reference point c, pixel steps U, V; world frame, mm) that describe the
    circular-orbit view of gantry angle `angle` (include/dfp.h conventions), float64."""
    cb, sb = math.cos(angle), math.sin(angle)
    n = torch.tensor([cb, sb, 0.0], dtype=torch.float64)
    return torch.cat([geom.sad * n, -(geom.sdd - geom.sad) * n,
                      geom.du * torch.tensor([-sb, cb, 0.0], dtype=torch.float64),
                      geom.dv * torch.tensor([0.0, 0.0, 1.0], dtype=torch.float64)])


def move_frame(frame, Q, tau) -> torch.Tensor:
    """The scanner of `frame` moved rigidly as a whole: points x -> Q x + tau, directions d -> Q d."""
    f = torch.as_tensor(frame, dtype=torch.float64).reshape(4, 3)
    Q = torch.as_tensor(Q, dtype=torch.float64)
    tau = torch.as_tensor(tau, dtype=torch.float64)
    return torch.cat([Q @ f[0] + tau, Q @ f[1] + tau, Q @ f[2], Q @ f[3]])


def _axis_rotation(axis: torch.Tensor, angle: float) -> torch.Tensor:
    """Rotation by `angle` about the unit vector `axis` (Rodrigues), float64."""
    k = axis / torch.linalg.norm(axis)
    K = torch.tensor([[0.0, -k[2], k[1]], [k[2], 0.0, -k[0]], [-k[1], k[0], 0.0]], dtype=torch.float64)
    return torch.eye(3, dtype=torch.float64) + math.sin(angle) * K + (1.0 - math.cos(angle)) * (K @ K)


def noncircular_orbit(geom: Geometry, angles, seed: int, tilt_deg: float = 10.0, wobble_mm: float = 3.0,
                      spin_deg: float = 1.5, sdd_mm: float = 15.0) -> torch.Tensor:
    """[V,12] view frames of a seeded NON-CIRCULAR orbit (stands in for the calibrated non-circular geometry of
    PAPER.md :244): the circular view of each gantry angle, then (a) source and detector tilted out of the orbit
    plane about the view's u axis by tilt_deg * sin(2 beta + phase) (a saddle orbit), (b) the detector spun about
    its normal, shifted in its own plane and moved along the normal by smooth seeded sinusoids of the given
    amplitudes, (c) the source moved by up to wobble_mm in each direction.  float64; round to fp32 before use."""
    from .rng import SplitMix64
    rng = SplitMix64(seed)
    ph = [rng.uniform(0.0, 2.0 * math.pi) for _ in range(8)]
    out = []
    for beta in [float(b) for b in torch.as_tensor(angles, dtype=torch.float64).reshape(-1)]:
        f = circular_frame(geom, beta).reshape(4, 3)
        eu = f[2] / torch.linalg.norm(f[2])
        Q = _axis_rotation(eu, tilt_deg * math.pi / 180.0 * math.sin(2.0 * beta + ph[0]))
        f = move_frame(f, Q, [0.0, 0.0, 0.0]).reshape(4, 3)
        n = torch.linalg.cross(f[2], f[3])
        n = n / torch.linalg.norm(n)
        S = _axis_rotation(n, spin_deg * math.pi / 180.0 * math.sin(beta + ph[1]))
        U, V = S @ f[2], S @ f[3]
        c = f[1] + wobble_mm * math.sin(beta + ph[2]) * U / torch.linalg.norm(U) + \
            wobble_mm * math.sin(3.0 * beta + ph[3]) * V / torch.linalg.norm(V) + sdd_mm * math.sin(beta + ph[4]) * n
        s = f[0] + wobble_mm * torch.tensor([math.sin(beta + ph[5]), math.sin(2.0 * beta + ph[6]),
                                             math.sin(beta + ph[7])], dtype=torch.float64)
        out.append(torch.cat([s, c, U, V]))
    return torch.stack(out)
