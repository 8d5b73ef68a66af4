"""fp64 CPU oracle for the dfp hot path - TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes loader around `dfp_oracle.cpp` (see that file's header for what it computes, the
passages of PAPER.md it follows and what pins it).  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` leg may import this package; the product package
`paper_2508_13304_b200` never does, and this package never imports it.

All functions take / return numpy arrays; big inputs are float32 (the same bits the CUDA path gets)
and every result is float64.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dfp_oracle.cpp")
_LIB = os.path.join(_HERE, "libdfp_oracle.so")

LEVER_SAMPLE, LEVER_VOXEL = 0, 1
GRAD_CENTRAL, GRAD_INTERP = 0, 1
ROUTE_SIX, ROUTE_TWELVE = 0, 1


class _Geom(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("vx", ctypes.c_double), ("vy", ctypes.c_double), ("vz", ctypes.c_double),
                ("cx", ctypes.c_double), ("cy", ctypes.c_double), ("cz", ctypes.c_double),
                ("nu", ctypes.c_int32), ("nv", ctypes.c_int32),
                ("du", ctypes.c_double), ("dv", ctypes.c_double), ("u0", ctypes.c_double), ("v0", ctypes.c_double),
                ("sad", ctypes.c_double), ("sdd", ctypes.c_double), ("step_mm", ctypes.c_double),
                ("bp_weight", ctypes.c_int32), ("flags", ctypes.c_int32)]


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.ora_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().ora_num_threads())


def set_num_threads(n: int) -> None:
    _load().ora_set_num_threads(int(n))


def _geom(g) -> _Geom:
    d = g.as_dict() if hasattr(g, "as_dict") else dict(g)
    return _Geom(**{k: d[k] for k, _ in _Geom._fields_})


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape is not None:
        a = a.reshape(shape)
    return a


def _f32(a):
    if hasattr(a, "detach"):
        a = a.detach().cpu().numpy()
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


FLAG_VIEW_FRAMES = 64    # O14: `angles` holds [V][12] view frames (s, c, U, V) instead of [V] gantry angles


def _views(angles, poses, g):
    angles = _f64(angles).reshape(-1)
    poses = _f64(poses).reshape(-1, 6)
    per_view = 12 if (int(_geom(g).flags) & FLAG_VIEW_FRAMES) else 1
    assert angles.shape[0] == per_view * poses.shape[0]
    return angles, poses, int(poses.shape[0])


def forward(g, angles, poses, vol, return_steps=False):
    """O6.  vol [nz,ny,nx] float32 or float64 -> proj [V,nv,nu] float64 (and the ray-step count)."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    if hasattr(vol, "detach"):
        vol = vol.detach().cpu().numpy()
    gg = _geom(g)
    proj = np.empty((V, gg.nv, gg.nu), dtype=np.float64)
    steps = ctypes.c_int64(0)
    if np.asarray(vol).dtype == np.float64:
        vol = np.ascontiguousarray(vol)
        fn = lib.ora_forward_f64
    else:
        vol = _f32(vol)
        fn = lib.ora_forward_f32
    assert vol.shape == (gg.nz, gg.ny, gg.nx)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(proj), ctypes.byref(steps))
    return (proj, int(steps.value)) if return_steps else proj


def forward_T(g, angles, poses, y):
    """O10: explicit transpose of `forward` (adjointness pin).  y [V,nv,nu] -> vol float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    y = _f64(y, (V, gg.nv, gg.nu))
    out = np.empty((gg.nz, gg.ny, gg.nx), dtype=np.float64)
    lib.ora_forward_T(ctypes.byref(gg), V, _p(angles), _p(poses), _p(y), _p(out))
    return out


def forward_pose_grad(g, angles, poses, vol, upstream, lever_arm=LEVER_SAMPLE, grad_mode=GRAD_CENTRAL,
                      route=ROUTE_SIX):
    """O7.  upstream [V,nv,nu] float32 -> dL/dtheta [V,6] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    if hasattr(vol, "detach"):
        vol = vol.detach().cpu().numpy()
    up = _f32(upstream).reshape(V, gg.nv, gg.nu)
    grad = np.empty((V, 6), dtype=np.float64)
    if np.asarray(vol).dtype == np.float64:
        vol = np.ascontiguousarray(vol)
        fn = lib.ora_forward_pose_grad_f64
    else:
        vol = _f32(vol)
        fn = lib.ora_forward_pose_grad_f32
    assert vol.shape == (gg.nz, gg.ny, gg.nx)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(up), _p(grad), int(lever_arm), int(grad_mode),
       int(route))
    return grad


def backproject(g, angles, poses, proj, iz0=0, iz1=None):
    """O8.  proj [V,nv,nu] float32 -> vol[iz0:iz1] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    iz1 = gg.nz if iz1 is None else iz1
    proj = _f32(proj).reshape(V, gg.nv, gg.nu)
    out = np.empty((iz1 - iz0, gg.ny, gg.nx), dtype=np.float64)
    lib.ora_backproject(ctypes.byref(gg), V, _p(angles), _p(poses), _p(proj), _p(out), int(iz0), int(iz1))
    return out


def backproject_T(g, angles, poses, x):
    """O10: explicit transpose of `backproject` (splat), adjointness pin.  x [nz,ny,nx] -> [V,nv,nu] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    x = _f64(x, (gg.nz, gg.ny, gg.nx))
    out = np.empty((V, gg.nv, gg.nu), dtype=np.float64)
    lib.ora_backproject_T(ctypes.byref(gg), V, _p(angles), _p(poses), _p(x), _p(out))
    return out


def backproject_pose_grad(g, angles, poses, proj, upstream, grad_mode=GRAD_CENTRAL, route=ROUTE_SIX):
    """O9.  proj [V,nv,nu] float32, upstream [nz,ny,nx] float32 -> dL/dtheta [V,6] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    proj = _f32(proj).reshape(V, gg.nv, gg.nu)
    up = _f32(upstream).reshape(gg.nz, gg.ny, gg.nx)
    grad = np.empty((V, 6), dtype=np.float64)
    lib.ora_backproject_pose_grad(ctypes.byref(gg), V, _p(angles), _p(poses), _p(proj), _p(up), _p(grad),
                                  int(grad_mode), int(route))
    return grad


def rotation(pose6):
    """R(gamma) [3,3] and dR/dgamma_k [3,3,3] as the oracle builds them (O4, U4)."""
    lib = _load()
    p = _f64(pose6).reshape(6)
    R = np.empty((3, 3)); dR = np.empty((3, 3, 3))
    lib.ora_rotation(_p(p), _p(R), _p(dR))
    return R, dR


def projection_matrix(g, angle):
    """P [3,4] in pixel-index units (O5 / O14, Eq.1).  `angle`: gantry angle, or a 12-number view frame
    when the geometry carries FLAG_VIEW_FRAMES."""
    lib = _load()
    gg = _geom(g)
    view = _f64(angle).reshape(-1)
    assert view.shape[0] == (12 if (int(gg.flags) & FLAG_VIEW_FRAMES) else 1)
    P = np.empty((3, 4))
    lib.ora_projection_matrix(ctypes.byref(gg), _p(view), _p(P))
    return P


# ---------------------------------------------------------------------------------------------------------------
# O12: Siddon's exact radiological path - the paper's own ray-driven weights (PAPER.md :213, :395)
def forward_siddon(g, angles, poses, vol):
    """l_i = sum_j a^ij mu_j, a^ij = length of ray i inside voxel j.  vol [nz,ny,nx] -> proj [V,nv,nu] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    if hasattr(vol, "detach"):
        vol = vol.detach().cpu().numpy()
    gg = _geom(g)
    proj = np.empty((V, gg.nv, gg.nu), dtype=np.float64)
    if np.asarray(vol).dtype == np.float64:
        vol = np.ascontiguousarray(vol)
        fn = lib.ora_forward_siddon_f64
    else:
        vol = _f32(vol)
        fn = lib.ora_forward_siddon_f32
    assert vol.shape == (gg.nz, gg.ny, gg.nx)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(proj))
    return proj


def forward_siddon_T(g, angles, poses, y):
    """Explicit transpose of `forward_siddon` (adjointness pin).  y [V,nv,nu] -> vol float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    y = _f64(y, (V, gg.nv, gg.nu))
    out = np.empty((gg.nz, gg.ny, gg.nx), dtype=np.float64)
    lib.ora_forward_siddon_T(ctypes.byref(gg), V, _p(angles), _p(poses), _p(y), _p(out))
    return out


def forward_pose_grad_siddon(g, angles, poses, vol, upstream, route=ROUTE_SIX):
    """Pose gradient with Siddon weights and per-voxel G_f^j (Eq.19-20, :189).  -> [V,6] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    if hasattr(vol, "detach"):
        vol = vol.detach().cpu().numpy()
    up = _f32(upstream).reshape(V, gg.nv, gg.nu)
    grad = np.empty((V, 6), dtype=np.float64)
    if np.asarray(vol).dtype == np.float64:
        vol = np.ascontiguousarray(vol)
        fn = lib.ora_forward_pose_grad_siddon_f64
    else:
        vol = _f32(vol)
        fn = lib.ora_forward_pose_grad_siddon_f32
    assert vol.shape == (gg.nz, gg.ny, gg.nx)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(up), _p(grad), int(route))
    return grad


# ---------------------------------------------------------------------------------------------------------------
# O13: Joseph's projector (plane-by-plane along the driving axis, bilinear in each plane)
def _model_call(name, g, angles, poses, vol, extra=()):
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    if hasattr(vol, "detach"):
        vol = vol.detach().cpu().numpy()
    gg = _geom(g)
    if np.asarray(vol).dtype == np.float64:
        vol = np.ascontiguousarray(vol)
        fn = getattr(lib, name + "_f64")
    else:
        vol = _f32(vol)
        fn = getattr(lib, name + "_f32")
    assert vol.shape == (gg.nz, gg.ny, gg.nx)
    return fn, gg, angles, poses, V, vol


def forward_joseph(g, angles, poses, vol):
    """l_i = (v_a*/|e_a*|) sum over voxel-centre planes of the bilinear interpolant.  -> proj [V,nv,nu] float64."""
    fn, gg, angles, poses, V, vol = _model_call("ora_forward_joseph", g, angles, poses, vol)
    proj = np.empty((V, gg.nv, gg.nu), dtype=np.float64)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(proj))
    return proj


def forward_joseph_T(g, angles, poses, y):
    """Explicit transpose of `forward_joseph` (adjointness pin).  y [V,nv,nu] -> vol float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    y = _f64(y, (V, gg.nv, gg.nu))
    out = np.empty((gg.nz, gg.ny, gg.nx), dtype=np.float64)
    lib.ora_forward_joseph_T(ctypes.byref(gg), V, _p(angles), _p(poses), _p(y), _p(out))
    return out


def forward_pose_grad_joseph(g, angles, poses, vol, upstream):
    """Pose gradient with Joseph weights and per-voxel G_f^j (Eq.19-20, :189).  -> [V,6] float64."""
    fn, gg, angles, poses, V, vol = _model_call("ora_forward_pose_grad_joseph", g, angles, poses, vol)
    up = _f32(upstream).reshape(V, gg.nv, gg.nu)
    grad = np.empty((V, 6), dtype=np.float64)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(up), _p(grad))
    return grad


# ---------------------------------------------------------------------------------------------------------------
# O15: distance-driven projector pair (PAPER.md :213 [44]; reading DESIGN.md U14)
def forward_dd(g, angles, poses, vol):
    """l_i = sum_j a^ij mu_j with distance-driven weights.  -> proj [V,nv,nu] float64."""
    fn, gg, angles, poses, V, vol = _model_call("ora_forward_dd", g, angles, poses, vol)
    proj = np.empty((V, gg.nv, gg.nu), dtype=np.float64)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(proj))
    return proj


def backproject_dd(g, angles, poses, proj, iz0=0, iz1=None):
    """The DD back-projector = the exact transpose of `forward_dd` (Eq.21).  proj [V,nv,nu] float32 -> vol[iz0:iz1]."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    iz1 = gg.nz if iz1 is None else iz1
    proj = _f32(proj).reshape(V, gg.nv, gg.nu)
    out = np.empty((iz1 - iz0, gg.ny, gg.nx), dtype=np.float64)
    lib.ora_backproject_dd(ctypes.byref(gg), V, _p(angles), _p(poses), _p(proj), _p(out), int(iz0), int(iz1))
    return out


def forward_pose_grad_dd(g, angles, poses, vol, upstream):
    """Pose gradient through the DD forward projector, per-voxel G_f^j (Eq.19-20).  -> [V,6] float64."""
    fn, gg, angles, poses, V, vol = _model_call("ora_forward_pose_grad_dd", g, angles, poses, vol)
    up = _f32(upstream).reshape(V, gg.nv, gg.nu)
    grad = np.empty((V, 6), dtype=np.float64)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(up), _p(grad))
    return grad


def backproject_pose_grad_dd(g, angles, poses, proj, upstream):
    """Pose gradient through the DD back-projector, per-pixel G_b^i (Eq.22).  -> [V,6] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    proj = _f32(proj).reshape(V, gg.nv, gg.nu)
    up = _f32(upstream).reshape(gg.nz, gg.ny, gg.nx)
    grad = np.empty((V, 6), dtype=np.float64)
    lib.ora_backproject_pose_grad_dd(ctypes.byref(gg), V, _p(angles), _p(poses), _p(proj), _p(up), _p(grad))
    return grad


# ---------------------------------------------------------------------------------------------------------------
# O16: separable-footprint projector pair SF-TR (PAPER.md :213 [29]; reading DESIGN.md U16)
def forward_sf(g, angles, poses, vol):
    """l_i = sum_j a^ij mu_j with separable-footprint weights (voxel-driven).  -> proj [V,nv,nu] float64."""
    fn, gg, angles, poses, V, vol = _model_call("ora_forward_sf", g, angles, poses, vol)
    proj = np.empty((V, gg.nv, gg.nu), dtype=np.float64)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(proj))
    return proj


def backproject_sf(g, angles, poses, proj, iz0=0, iz1=None):
    """The SF back-projector = the exact transpose of `forward_sf`.  proj [V,nv,nu] float32 -> vol[iz0:iz1] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    iz1 = gg.nz if iz1 is None else iz1
    proj = _f32(proj).reshape(V, gg.nv, gg.nu)
    out = np.empty((iz1 - iz0, gg.ny, gg.nx), dtype=np.float64)
    lib.ora_backproject_sf(ctypes.byref(gg), V, _p(angles), _p(poses), _p(proj), _p(out), int(iz0), int(iz1))
    return out


def forward_pose_grad_sf(g, angles, poses, vol, upstream):
    """Pose gradient through the SF forward projector, per-voxel G_f^j (Eq.19-20).  -> [V,6] float64."""
    fn, gg, angles, poses, V, vol = _model_call("ora_forward_pose_grad_sf", g, angles, poses, vol)
    up = _f32(upstream).reshape(V, gg.nv, gg.nu)
    grad = np.empty((V, 6), dtype=np.float64)
    fn(ctypes.byref(gg), V, _p(angles), _p(poses), _p(vol), _p(up), _p(grad))
    return grad


def backproject_pose_grad_sf(g, angles, poses, proj, upstream):
    """Pose gradient through the SF back-projector, per-pixel G_b^i (Eq.22).  -> [V,6] float64."""
    lib = _load()
    angles, poses, V = _views(angles, poses, g)
    gg = _geom(g)
    proj = _f32(proj).reshape(V, gg.nv, gg.nu)
    up = _f32(upstream).reshape(gg.nz, gg.ny, gg.nx)
    grad = np.empty((V, 6), dtype=np.float64)
    lib.ora_backproject_pose_grad_sf(ctypes.byref(gg), V, _p(angles), _p(poses), _p(proj), _p(up), _p(grad))
    return grad
