"""ctypes binding of include/dfp.h.  Marshals arguments and nothing else.

Device-pointer calls take torch CUDA tensors (fp32, contiguous) and run asynchronously on torch's current
stream; `*_host` calls take CPU tensors / numpy arrays.  `angles` / `poses` are host arrays (any float
sequence; rounded to fp32, which is what the C ABI takes).
"""
import contextlib
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libdfp.so")

OP_FORWARD, OP_FORWARD_POSE_GRAD, OP_BACKPROJECT, OP_BACKPROJECT_POSE_GRAD, OP_FORWARD_FUSED, OP_NCC = 0, 1, 2, 3, 4, 5
FLAG_DW = 1
FLAG_NO_TMA = 2
FLAG_GRAD_INTERP = 4
FLAG_SIDDON = 8
FLAG_ACCUMULATE = 16
FLAG_JOSEPH = 32
FLAG_DD = 128              # distance-driven weights in all four calls (include/dfp.h)
FLAG_SF = 256              # separable-footprint weights in all four calls
FLAG_VIEW_FRAMES = 64      # `angles` arguments hold [V,12] explicit view frames (s, c, U, V), include/dfp.h
PATH_GATHER, PATH_TMA = 0, 1


class DfpError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"dfp status {status}: {text}")
        self.status = status


class Geometry(ctypes.Structure):
    """Mirror of `dfp_geometry` (include/dfp.h)."""
    _fields_ = [("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("vx", ctypes.c_float), ("vy", ctypes.c_float), ("vz", ctypes.c_float),
                ("cx", ctypes.c_float), ("cy", ctypes.c_float), ("cz", ctypes.c_float),
                ("nu", ctypes.c_int32), ("nv", ctypes.c_int32),
                ("du", ctypes.c_float), ("dv", ctypes.c_float), ("u0", ctypes.c_float), ("v0", ctypes.c_float),
                ("sad", ctypes.c_float), ("sdd", ctypes.c_float), ("step_mm", ctypes.c_float),
                ("bp_weight", ctypes.c_int32), ("flags", ctypes.c_int32)]

    @classmethod
    def of(cls, g) -> "Geometry":
        """From a Geometry, a mapping, or any object with these attributes (e.g. workloads.Geometry)."""
        if isinstance(g, cls):
            return g
        get = (lambda k: g[k]) if isinstance(g, dict) else (lambda k: getattr(g, k))
        return cls(**{k: get(k) for k, _ in cls._fields_})


def _load():
    # (re)build when the library is missing or older than its sources and nvcc is here; on a box without nvcc
    # a prebuilt in-tree library is used as is.  Never fall back to anything else.
    from .build import build, stale
    import shutil
    if stale() and (shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc") or not os.path.exists(_LIB_PATH)):
        try:
            build()
        except Exception as e:
            raise ImportError(f"libdfp.so is missing or stale and could not be built ({e}); the dfp CUDA library "
                              "is required - there is no CPU fallback") from e
    lib = ctypes.CDLL(_LIB_PATH)
    vp, cp, sz, ci = ctypes.c_void_p, ctypes.c_char_p, ctypes.c_size_t, ctypes.c_int
    gp = ctypes.POINTER(Geometry)
    dev = [gp, ci, vp, vp, vp, vp, vp, sz, vp]
    devg = [gp, ci, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.dfp_forward.argtypes = dev
    lib.dfp_backproject.argtypes = dev
    lib.dfp_forward_pose_grad.argtypes = devg
    lib.dfp_backproject_pose_grad.argtypes = devg
    lib.dfp_forward_fused_moments.argtypes = [gp, ci, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.dfp_forward_fused_moments.restype = ci
    lib.dfp_ncc_pose_grad.argtypes = [gp, ci, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.dfp_ncc_pose_grad.restype = ci
    lib.dfp_ncc_pose_grad_static.argtypes = [gp, ci, vp, vp, vp, vp, vp, vp]
    lib.dfp_ncc_pose_grad_static.restype = ci
    lib.dfp_forward_host.argtypes = [gp, ci, vp, vp, vp, vp, vp]
    lib.dfp_backproject_host.argtypes = [gp, ci, vp, vp, vp, vp, vp]
    lib.dfp_forward_pose_grad_host.argtypes = [gp, ci, vp, vp, vp, vp, vp, vp]
    lib.dfp_backproject_pose_grad_host.argtypes = [gp, ci, vp, vp, vp, vp, vp, vp]
    for f in (lib.dfp_forward, lib.dfp_backproject, lib.dfp_forward_pose_grad, lib.dfp_backproject_pose_grad,
              lib.dfp_forward_host, lib.dfp_backproject_host, lib.dfp_forward_pose_grad_host,
              lib.dfp_backproject_pose_grad_host, lib.dfp_last_launch_count, lib.dfp_last_path, lib.dfp_version):
        f.restype = ci
    lib.dfp_workspace_bytes.argtypes = [gp, ci, ci]
    lib.dfp_workspace_bytes.restype = sz
    lib.dfp_workspace_bytes_for_views.argtypes = [gp, ci, vp, vp, ci]
    lib.dfp_workspace_bytes_for_views.restype = sz
    lib.dfp_count_ray_steps.argtypes = [gp, ci, vp, vp]
    lib.dfp_count_ray_steps.restype = ctypes.c_int64
    lib.dfp_set_kernel_timing.argtypes = [ci]
    lib.dfp_set_kernel_timing.restype = ci
    lib.dfp_last_kernel_ms.argtypes = []
    lib.dfp_last_kernel_ms.restype = ctypes.c_float
    lib.dfp_status_string.argtypes = [ci]
    lib.dfp_status_string.restype = cp
    return lib


_lib = _load()


def lib_path() -> str:
    return _LIB_PATH


def version() -> int:
    return int(_lib.dfp_version())


def status_string(status: int) -> str:
    return _lib.dfp_status_string(int(status)).decode()


def last_launch_count() -> int:
    return int(_lib.dfp_last_launch_count())


def last_path() -> int:
    """PATH_GATHER or PATH_TMA: which kernels the last device-pointer call on this thread ran."""
    return int(_lib.dfp_last_path())


def set_kernel_timing(enable: bool) -> None:
    _lib.dfp_set_kernel_timing(1 if enable else 0)


def last_kernel_ms() -> float:
    """Milliseconds of the dominant kernel of the last device-pointer call (waits for it); -1 if timing is off."""
    return float(_lib.dfp_last_kernel_ms())


def _check(status):
    if status != 0:
        raise DfpError(status, status_string(status))


def _views(angles, poses, geom):
    """`angles`: [V] gantry angles, or [V,12] view frames (s, c, U, V) when geom.flags has FLAG_VIEW_FRAMES."""
    a = np.ascontiguousarray(np.asarray(torch.as_tensor(angles).cpu().numpy() if torch.is_tensor(angles) else angles,
                                        dtype=np.float32).reshape(-1))
    p = np.ascontiguousarray(np.asarray(torch.as_tensor(poses).cpu().numpy() if torch.is_tensor(poses) else poses,
                                        dtype=np.float32).reshape(-1, 6))
    per_view = 12 if (int(Geometry.of(geom).flags) & FLAG_VIEW_FRAMES) else 1
    if a.shape[0] != per_view * p.shape[0]:
        raise ValueError("angles / view frames and poses disagree on the number of views")
    return a, p, int(p.shape[0])


def _dev(t: torch.Tensor, shape, name):
    if not (torch.is_tensor(t) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float32 CUDA tensor")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name} has shape {tuple(t.shape)}, expected {tuple(shape)}")
    return ctypes.c_void_p(t.data_ptr())


def workspace_bytes(geom, n_views: int, op: int) -> int:
    return int(_lib.dfp_workspace_bytes(ctypes.byref(Geometry.of(geom)), int(n_views), int(op)))


def workspace_bytes_for_views(geom, angles, poses, op: int) -> int:
    """dfp_workspace_bytes_for_views: the bytes the op needs for THESE views (<= workspace_bytes; without the gather
    path's 4x packed copy when the views take the TMA-staged kernels)."""
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    return int(_lib.dfp_workspace_bytes_for_views(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p), int(op)))


def _workspace(g, V, op, ws, device, a=None, p=None):
    """The caller's workspace as (tensor, pointer, bytes) - its size is checked by the library - or, if none was given, a
    new one of the size these views need."""
    if ws is None:
        if a is None:
            need = workspace_bytes(g, V, op)
        else:
            need = int(_lib.dfp_workspace_bytes_for_views(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p), int(op)))
        if need == 0:
            _check(-2)
        ws = torch.empty(need, dtype=torch.uint8, device=device)
    return ws, ctypes.c_void_p(ws.data_ptr()), ctypes.c_size_t(ws.numel() * ws.element_size())


def _stream(t=None):
    """torch's current stream ON THE TENSORS' DEVICE (the library launches on the thread's current device, which the
    device-pointer wrappers set to that device for the duration of the call)."""
    dev = t.device if (torch.is_tensor(t) and t.is_cuda) else None
    return ctypes.c_void_p(torch.cuda.current_stream(dev).cuda_stream)


def _same_device(*tensors):
    ts = [t for t in tensors if torch.is_tensor(t) and t.is_cuda]
    if not ts:
        return contextlib.nullcontext()          # the argument checks of the call report what is wrong
    for t in ts:
        if t.device != ts[0].device:
            raise ValueError(f"all device tensors of a call must live on one device ({ts[0].device} vs {t.device})")
    return torch.cuda.device(ts[0].device)


def _np_ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def forward(geom, angles, poses, vol, out=None, ws=None):
    """dfp_forward: vol [nz,ny,nx] cuda fp32 -> proj [V,nv,nu]."""
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((V, g.nv, g.nu), dtype=torch.float32, device=vol.device)
    ws, wp, wn = _workspace(g, V, OP_FORWARD, ws, vol.device, a, p)
    with _same_device(vol, out, ws):
        _check(_lib.dfp_forward(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p), _dev(vol, (g.nz, g.ny, g.nx), "vol"),
                                _dev(out, (V, g.nv, g.nu), "proj"), wp, wn, _stream(vol)))
    return out


def forward_pose_grad(geom, angles, poses, vol, dLdproj, out=None, ws=None):
    """dfp_forward_pose_grad: vol, dL/dproj [V,nv,nu] -> dL/dtheta [V,6]."""
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((V, 6), dtype=torch.float32, device=vol.device)
    ws, wp, wn = _workspace(g, V, OP_FORWARD_POSE_GRAD, ws, vol.device, a, p)
    with _same_device(vol, dLdproj, out, ws):
        _check(_lib.dfp_forward_pose_grad(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p),
                                          _dev(vol, (g.nz, g.ny, g.nx), "vol"),
                                          _dev(dLdproj, (V, g.nv, g.nu), "dLdproj"), _dev(out, (V, 6), "grad"), wp, wn,
                                          _stream(vol)))
    return out


def forward_fused_moments(geom, angles, poses, vol, target, out_proj=None, out_moments=None, ws=None):
    """dfp_forward_fused_moments: vol, target [V,nv,nu] -> (proj [V,nv,nu], moments [V,3,6]) in one traversal."""
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out_proj is None:
        out_proj = torch.empty((V, g.nv, g.nu), dtype=torch.float32, device=vol.device)
    if out_moments is None:
        out_moments = torch.empty((V, 3, 6), dtype=torch.float32, device=vol.device)
    ws, wp, wn = _workspace(g, V, OP_FORWARD_FUSED, ws, vol.device, a, p)
    with _same_device(vol, target, out_proj, out_moments, ws):
        _check(_lib.dfp_forward_fused_moments(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p),
                                              _dev(vol, (g.nz, g.ny, g.nx), "vol"),
                                              _dev(target, (V, g.nv, g.nu), "target"),
                                              _dev(out_proj, (V, g.nv, g.nu), "proj"),
                                              _dev(out_moments, (V, 3, 6), "moments"), wp, wn, _stream(vol)))
    return out_proj, out_moments


def ncc_pose_grad(geom, proj, target, moments, out_ncc=None, out_grad=None, ws=None):
    """dfp_ncc_pose_grad: NCC(l_v, b_v) [V] and dNCC/dtheta_v [V,6] from the outputs of forward_fused_moments."""
    g = Geometry.of(geom)
    V = int(proj.shape[0])
    if out_ncc is None:
        out_ncc = torch.empty((V,), dtype=torch.float32, device=proj.device)
    if out_grad is None:
        out_grad = torch.empty((V, 6), dtype=torch.float32, device=proj.device)
    ws, wp, wn = _workspace(g, V, OP_NCC, ws, proj.device)
    with _same_device(proj, target, moments, out_ncc, out_grad, ws):
        _check(_lib.dfp_ncc_pose_grad(ctypes.byref(g), V, _dev(proj, (V, g.nv, g.nu), "proj"),
                                      _dev(target, (V, g.nv, g.nu), "target"), _dev(moments, (V, 3, 6), "moments"),
                                      _dev(out_ncc, (V,), "ncc"), _dev(out_grad, (V, 6), "grad"), wp, wn, _stream(proj)))
    return out_ncc, out_grad


NCC_STATIC_MAX_VIEWS = 256      # DFP_NCC_STATIC_MAX_VIEWS (include/dfp.h)


def ncc_pose_grad_static(geom, proj, target, moments, out_ncc, out_grad):
    """dfp_ncc_pose_grad_static: dfp_ncc_pose_grad without a workspace - the partial sums live in a fixed device array
    of the library, the call allocates nothing (the caller passes BOTH outputs).  At most NCC_STATIC_MAX_VIEWS views;
    calls that can overlap on the GPU race on the shared array (include/dfp.h)."""
    g = Geometry.of(geom)
    V = int(proj.shape[0])
    with _same_device(proj, target, moments, out_ncc, out_grad):
        _check(_lib.dfp_ncc_pose_grad_static(ctypes.byref(g), V, _dev(proj, (V, g.nv, g.nu), "proj"),
                                             _dev(target, (V, g.nv, g.nu), "target"),
                                             _dev(moments, (V, 3, 6), "moments"), _dev(out_ncc, (V,), "ncc"),
                                             _dev(out_grad, (V, 6), "grad"), _stream(proj)))
    return out_ncc, out_grad


def backproject(geom, angles, poses, proj, out=None, ws=None):
    """dfp_backproject: proj [V,nv,nu] cuda fp32 -> vol [nz,ny,nx]."""
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((g.nz, g.ny, g.nx), dtype=torch.float32, device=proj.device)
    ws, wp, wn = _workspace(g, V, OP_BACKPROJECT, ws, proj.device, a, p)
    with _same_device(proj, out, ws):
        _check(_lib.dfp_backproject(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p), _dev(proj, (V, g.nv, g.nu), "proj"),
                                    _dev(out, (g.nz, g.ny, g.nx), "vol"), wp, wn, _stream(proj)))
    return out


def backproject_pose_grad(geom, angles, poses, proj, dLdvol, out=None, ws=None):
    """dfp_backproject_pose_grad: proj, dL/dvol [nz,ny,nx] -> dL/dtheta [V,6]."""
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((V, 6), dtype=torch.float32, device=proj.device)
    ws, wp, wn = _workspace(g, V, OP_BACKPROJECT_POSE_GRAD, ws, proj.device, a, p)
    with _same_device(proj, dLdvol, out, ws):
        _check(_lib.dfp_backproject_pose_grad(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p),
                                              _dev(proj, (V, g.nv, g.nu), "proj"),
                                              _dev(dLdvol, (g.nz, g.ny, g.nx), "dLdvol"), _dev(out, (V, 6), "grad"), wp,
                                              wn, _stream(proj)))
    return out


def _host(t, shape, name):
    if torch.is_tensor(t):
        if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
            raise TypeError(f"{name} must be a contiguous float32 CPU tensor")
        if tuple(t.shape) != tuple(shape):
            raise ValueError(f"{name} has shape {tuple(t.shape)}, expected {tuple(shape)}")
        return ctypes.c_void_p(t.data_ptr())
    if not (isinstance(t, np.ndarray) and t.dtype == np.float32 and t.flags["C_CONTIGUOUS"]):
        raise TypeError(f"{name} must be a contiguous float32 array")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name} has shape {tuple(t.shape)}, expected {tuple(shape)}")
    return _np_ptr(t)


def forward_host(geom, angles, poses, vol, out=None):
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((V, g.nv, g.nu), dtype=torch.float32, pin_memory=True)
    _check(_lib.dfp_forward_host(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p), _host(vol, (g.nz, g.ny, g.nx), "vol"),
                                 _host(out, (V, g.nv, g.nu), "proj"), _stream()))
    return out


def forward_pose_grad_host(geom, angles, poses, vol, dLdproj, out=None):
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((V, 6), dtype=torch.float32, pin_memory=True)
    _check(_lib.dfp_forward_pose_grad_host(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p),
                                           _host(vol, (g.nz, g.ny, g.nx), "vol"),
                                           _host(dLdproj, (V, g.nv, g.nu), "dLdproj"), _host(out, (V, 6), "grad"),
                                           _stream()))
    return out


def backproject_host(geom, angles, poses, proj, out=None):
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((g.nz, g.ny, g.nx), dtype=torch.float32, pin_memory=True)
    _check(_lib.dfp_backproject_host(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p),
                                     _host(proj, (V, g.nv, g.nu), "proj"), _host(out, (g.nz, g.ny, g.nx), "vol"),
                                     _stream()))
    return out


def backproject_pose_grad_host(geom, angles, poses, proj, dLdvol, out=None):
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    if out is None:
        out = torch.empty((V, 6), dtype=torch.float32, pin_memory=True)
    _check(_lib.dfp_backproject_pose_grad_host(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p),
                                               _host(proj, (V, g.nv, g.nu), "proj"),
                                               _host(dLdvol, (g.nz, g.ny, g.nx), "dLdvol"),
                                               _host(out, (V, 6), "grad"), _stream()))
    return out


def count_ray_steps(geom, angles, poses) -> int:
    """Ray-steps one forward / forward_pose_grad call marches over (the unit of the Gray-steps/s metric)."""
    g = Geometry.of(geom)
    a, p, V = _views(angles, poses, geom)
    n = int(_lib.dfp_count_ray_steps(ctypes.byref(g), V, _np_ptr(a), _np_ptr(p)))
    if n < 0:
        raise DfpError(-6, status_string(-6))
    return n
