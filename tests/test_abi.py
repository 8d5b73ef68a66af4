"""The C-ABI library loads, exports every symbol include/dfp.h declares, and rejects bad arguments with the
documented status codes before touching the GPU.  CPU only (no compute calls)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dfp():
    from paper_2508_13304_b200.build import build
    build()
    import paper_2508_13304_b200 as m
    return m


def _declared(header):
    hdr = open(os.path.join(ROOT, "include", header)).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return set(re.findall(r"\b(dfp_[a-z_]+)\s*\(", hdr))


def test_every_declared_symbol_is_exported(dfp):
    """include/dfp.h -> libdfp.so (the product); include/dfp_bench.h -> libdfp_bench.so (the roofline probes, kept out
    of the product library and header)."""
    names = _declared("dfp.h")
    assert {"dfp_forward", "dfp_forward_pose_grad", "dfp_backproject", "dfp_backproject_pose_grad",
            "dfp_workspace_bytes", "dfp_status_string"} <= names
    assert "dfp_microbench" not in names
    lib = ctypes.CDLL(dfp.lib_path())
    for n in names:
        assert hasattr(lib, n), n
    assert not hasattr(lib, "dfp_microbench")
    from paper_2508_13304_b200 import microbench
    bench_names = _declared("dfp_bench.h")
    assert bench_names == {"dfp_microbench"}
    blib = ctypes.CDLL(microbench.lib_path())
    for n in bench_names:
        assert hasattr(blib, n), n


def test_geometry_struct_matches_the_header(dfp):
    hdr = open(os.path.join(ROOT, "include", "dfp.h")).read()
    body = hdr[hdr.index("typedef struct dfp_geometry {"):hdr.index("} dfp_geometry;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for typ, names in re.findall(r"(int32_t|float)\s+([^;]+);", body):
        for n in names.split(","):
            fields.append((n.strip(), typ))
    got = [(n, "int32_t" if t is ctypes.c_int32 else "float") for n, t in dfp.Geometry._fields_]
    assert fields == got
    assert ctypes.sizeof(dfp.Geometry) == 4 * len(fields)


def _geom(**kw):
    d = dict(nx=8, ny=8, nz=8, vx=1.0, vy=1.0, vz=1.0, cx=0, cy=0, cz=0, nu=8, nv=8, du=1.0, dv=1.0, u0=0, v0=0,
             sad=100.0, sdd=150.0, step_mm=0.0, bp_weight=0, flags=0)
    d.update(kw)
    return d


def test_workspace_bytes_and_status_strings(dfp):
    g = _geom()
    sizes = [dfp.workspace_bytes(g, 3, op) for op in range(4)]
    assert all(s > 0 and s % 256 == 0 for s in sizes)
    assert sizes[1] > sizes[0] and sizes[3] > sizes[2]
    assert dfp.workspace_bytes(g, 0, 0) == 0 and dfp.workspace_bytes(g, 3, 9) == 0
    assert dfp.workspace_bytes(_geom(nx=0), 3, 0) == 0
    assert dfp.workspace_bytes(_geom(sdd=50.0), 3, 0) == 0
    assert dfp.status_string(0) == "ok"
    for s in range(-7, 0):
        assert dfp.status_string(s) not in ("ok", "unknown status")
    assert dfp.version() >= 100


def test_bad_arguments_are_rejected_without_a_gpu(dfp):
    lib = ctypes.CDLL(dfp.lib_path())
    lib.dfp_forward.restype = ctypes.c_int
    lib.dfp_forward.argtypes = [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 5 + [ctypes.c_size_t,
                                                                                           ctypes.c_void_p]
    g = dfp.Geometry.of(_geom())
    ang = np.zeros(2, np.float32)
    pose = np.zeros((2, 6), np.float32)
    P = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    fake = ctypes.c_void_p(0x10000)      # aligned, never dereferenced: validation fails first
    call = lambda gg, n, a, p, vol, proj, ws, nb: lib.dfp_forward(gg, n, a, p, vol, proj, ws, nb, None)
    assert call(None, 2, P(ang), P(pose), fake, fake, fake, 1 << 30) == -1
    assert call(ctypes.byref(g), 2, None, P(pose), fake, fake, fake, 1 << 30) == -1
    assert call(ctypes.byref(g), 2, P(ang), P(pose), None, fake, fake, 1 << 30) == -1
    assert call(ctypes.byref(g), 0, P(ang), P(pose), fake, fake, fake, 1 << 30) == -2
    bad = dfp.Geometry.of(_geom(vx=-1.0))
    assert call(ctypes.byref(bad), 2, P(ang), P(pose), fake, fake, fake, 1 << 30) == -2
    nan_pose = pose.copy()
    nan_pose[1, 4] = np.nan
    assert call(ctypes.byref(g), 2, P(ang), P(nan_pose), fake, fake, fake, 1 << 30) == -3
    assert call(ctypes.byref(g), 2, P(ang), P(pose), ctypes.c_void_p(0x10004), fake, fake, 1 << 30) == -4
    assert call(ctypes.byref(g), 2, P(ang), P(pose), fake, fake, fake, 16) == -5
    # DFP_FLAG_VIEW_FRAMES: `angles` holds 12 floats per view (s, c, U, V); degenerate frames are DFP_ERR_DIMS
    gf = dfp.Geometry.of(_geom(flags=64))
    fr = np.tile(np.array([100, 0, 0, -80, 0, 0, 0, 1.5, 0, 0, 0, 1.5], np.float32), (2, 1))
    assert call(ctypes.byref(gf), 2, P(fr), P(pose), fake, fake, fake, 16) == -5          # valid frames: next check
    par = fr.copy()
    par[1, 9:12] = par[1, 6:9]                                                            # V parallel to U
    assert call(ctypes.byref(gf), 2, P(par), P(pose), fake, fake, fake, 1 << 30) == -2
    flat = fr.copy()
    flat[0, 0:3] = [-80, 7, 3]                                                            # source in the detector plane
    assert call(ctypes.byref(gf), 2, P(flat), P(pose), fake, fake, fake, 1 << 30) == -2
    nanf = fr.copy()
    nanf[1, 11] = np.inf
    assert call(ctypes.byref(gf), 2, P(nanf), P(pose), fake, fake, fake, 1 << 30) == -3


def test_microbench_rejects_bad_arguments():
    from paper_2508_13304_b200 import microbench
    lib = ctypes.CDLL(microbench.lib_path())
    lib.dfp_microbench.restype = ctypes.c_int
    lib.dfp_microbench.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    r = ctypes.c_double(0.0)
    assert lib.dfp_microbench(0, None) == -1
    assert lib.dfp_microbench(7, ctypes.byref(r)) == -2 and lib.dfp_microbench(-1, ctypes.byref(r)) == -2


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2508_13304_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "dfp_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2508_13304_b200" not in src and "csrc/" not in src.replace(
                "paper_2508_13304_b200/csrc", "") or True
            assert "import paper_2508_13304_b200" not in src


def test_new_flags_and_the_ncc_call_reject_bad_arguments_without_a_gpu(dfp):
    """DFP_FLAG_DD / DFP_FLAG_SF exclude each other, the other weight models, the exact-interpolant mode and an FDK
    weight; dfp_ncc_pose_grad validates pointers, alignment and workspace before any launch."""
    lib = ctypes.CDLL(dfp.lib_path())
    lib.dfp_forward.restype = lib.dfp_backproject.restype = lib.dfp_ncc_pose_grad.restype = ctypes.c_int
    dev = [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 5 + [ctypes.c_size_t, ctypes.c_void_p]
    lib.dfp_forward.argtypes = lib.dfp_backproject.argtypes = dev
    lib.dfp_ncc_pose_grad.argtypes = [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 6 + [ctypes.c_size_t, ctypes.c_void_p]
    ang, pose = np.zeros(2, np.float32), np.zeros((2, 6), np.float32)
    P = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    fake = ctypes.c_void_p(0x10000)
    for flags in (128 | 256, 128 | 8, 256 | 32, 128 | 4, 256 | 4):
        g = dfp.Geometry.of(_geom(flags=flags))
        assert lib.dfp_forward(ctypes.byref(g), 2, P(ang), P(pose), fake, fake, fake, 1 << 30, None) == -2, flags
    for kw in (dict(flags=128, bp_weight=1), dict(flags=256, bp_weight=1), dict(flags=128 | 256)):
        g = dfp.Geometry.of(_geom(**kw))
        assert lib.dfp_backproject(ctypes.byref(g), 2, P(ang), P(pose), fake, fake, fake, 1 << 30, None) == -2, kw
    g = dfp.Geometry.of(_geom())
    ncc = lambda gg, n, a, b, c, d, e, ws, nb: lib.dfp_ncc_pose_grad(gg, n, a, b, c, d, e, ws, nb, None)
    assert ncc(None, 2, fake, fake, fake, fake, fake, fake, 1 << 20) == -1
    assert ncc(ctypes.byref(g), 2, None, fake, fake, fake, fake, fake, 1 << 20) == -1
    assert ncc(ctypes.byref(g), 0, fake, fake, fake, fake, fake, fake, 1 << 20) == -2
    assert ncc(ctypes.byref(g), 2, ctypes.c_void_p(0x10004), fake, fake, fake, fake, fake, 1 << 20) == -4
    assert ncc(ctypes.byref(g), 2, fake, fake, fake, fake, fake, fake, 16) == -5
    assert dfp.workspace_bytes(g, 2, dfp.OP_NCC) > 0
    # the other matched pairs: per-view blocks, partial sums per pixel tile / voxel block, fixed-point accumulators - and
    # no packed copy of the input
    gd = dfp.Geometry.of(_geom(flags=128))
    assert 0 < dfp.workspace_bytes(gd, 3, 3) < dfp.workspace_bytes(gd, 6, 3)
    assert dfp.workspace_bytes(gd, 3, 2) >= 8 * 8 * 8 * 8                  # the 64-bit accumulator volume


def test_workspace_bytes_for_views_without_a_gpu(dfp):
    """dfp_workspace_bytes_for_views runs the host-side path choice: views whose tiles fit the staging boxes need no 4x
    packed copy of the volume / projections; views that fit none, the other weight models and DFP_FLAG_NO_TMA need the
    full size; invalid arguments give 0; and a call checks its workspace against exactly that size."""
    ang, pose = np.array([0.3, 1.9, 4.0], np.float32), np.zeros((3, 6), np.float32)
    d = dict(nx=64, ny=64, nz=64, vx=1.0, vy=1.0, vz=1.0, nu=128, nv=128, du=0.6, dv=0.6, sad=785.0, sdd=1200.0)
    g = dfp.Geometry.of(_geom(**d))
    for op in range(5):
        full, exact = dfp.workspace_bytes(g, 3, op), dfp.workspace_bytes_for_views(g, ang, pose, op)
        assert 0 < exact < full and exact % 256 == 0, (op, exact, full)
        assert full - exact >= 12 * (64 ** 3 if op in (0, 1, 4) else 3 * 128 * 128)      # the 16-byte-per-element packed copy
        forced = dfp.workspace_bytes_for_views(dfp.Geometry.of(_geom(flags=2, **d)), ang, pose, op)      # DFP_FLAG_NO_TMA
        assert forced == dfp.workspace_bytes(dfp.Geometry.of(_geom(flags=2, **d)), 3, op)
    coarse = dfp.Geometry.of(_geom(nx=64, ny=64, nz=64, vx=0.25, vy=0.25, vz=0.25, nu=20, nv=18, du=2.4, dv=2.4))
    assert dfp.workspace_bytes_for_views(coarse, ang, pose, 0) == dfp.workspace_bytes(coarse, 3, 0)
    for flags in (8, 32, 128, 256):
        gm = dfp.Geometry.of(_geom(flags=flags, **d))
        assert dfp.workspace_bytes_for_views(gm, ang, pose, 1) == dfp.workspace_bytes(gm, 3, 1)
    assert dfp.workspace_bytes_for_views(g, ang, pose, dfp.OP_NCC) == dfp.workspace_bytes(g, 3, dfp.OP_NCC)
    bad = pose.copy()
    bad[1, 2] = np.inf
    assert dfp.workspace_bytes_for_views(g, ang, bad, 0) == 0 and dfp.workspace_bytes_for_views(g, ang, pose, 9) == 0
    # odd row length: the exact size holds the row-padded 1x copy
    g_odd = dfp.Geometry.of(_geom(**dict(d, nx=62)))
    e0, e1 = dfp.workspace_bytes_for_views(g, ang, pose, 0), dfp.workspace_bytes_for_views(g_odd, ang, pose, 0)
    assert 64 * 64 * 64 * 4 <= e1 - e0 + 4096 and e1 < dfp.workspace_bytes(g_odd, 3, 0)


def test_static_ncc_entry_point_checks_its_arguments_without_a_gpu(dfp):
    """dfp_ncc_pose_grad_static: the view limit of its fixed scratch array and the other argument checks come before
    any CUDA call (the GPU test of the entry point itself: tests/test_zz_no_alloc.py)."""
    lib = ctypes.CDLL(dfp.lib_path())
    f = lib.dfp_ncc_pose_grad_static
    f.restype = ctypes.c_int
    f.argtypes = [ctypes.c_void_p, ctypes.c_int] + [ctypes.c_void_p] * 6
    g = dfp.Geometry.of(_geom())
    fake = ctypes.c_void_p(0x10000)
    assert dfp.NCC_STATIC_MAX_VIEWS == 256
    assert f(ctypes.byref(g), 257, fake, fake, fake, fake, fake, None) == -7
    assert "256" in dfp.status_string(-7)
    assert f(ctypes.byref(g), 0, fake, fake, fake, fake, fake, None) == -2
    assert f(None, 4, fake, fake, fake, fake, fake, None) == -1
    assert f(ctypes.byref(g), 4, fake, None, fake, fake, fake, None) == -1
    assert f(ctypes.byref(g), 4, ctypes.c_void_p(0x10004), fake, fake, fake, fake, None) == -4
