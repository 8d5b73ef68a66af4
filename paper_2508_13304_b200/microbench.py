"""ctypes binding of include/dfp_bench.h (libdfp_bench.so): roofline-denominator probes for bench.py.

Not part of the product library: `import paper_2508_13304_b200` does not load it."""
import ctypes
import os

from .build import build_bench

MB_LDS, MB_FADD, MB_FFMA, MB_FFMA2 = 0, 1, 2, 3
_lib = None


def lib_path() -> str:
    return build_bench()


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(lib_path())
        _lib.dfp_microbench.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        _lib.dfp_microbench.restype = ctypes.c_int
    return _lib


def run(kind: int) -> float:
    """Sustained whole-device rate per second of one SM-side pipe on the current device (dfp_microbench)."""
    r = ctypes.c_double(0.0)
    st = _load().dfp_microbench(int(kind), ctypes.byref(r))
    if st != 0:
        raise RuntimeError(f"dfp_microbench status {st}")
    return float(r.value)
