"""Build libdfp.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2508_13304_b200.build [--force]

The .so is git-ignored but travels with the tree to the GPU box; nothing is JIT-compiled at import time on
a machine without nvcc - if the library is missing there, importing the binding fails loudly.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdfp.so")
SOURCES = [os.path.join(CSRC, "dfp_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("dfp_kernels.cuh", "dfp_fwd_tma.cuh", "dfp_bp_tma.cuh", "dfp_siddon.cuh", "dfp_joseph.cuh", "dfp_params.h")] + \
    [os.path.join(os.path.dirname(HERE), "include", "dfp.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        raise RuntimeError("nvcc not found: cannot build libdfp.so (there is no CPU fallback)")
    # DFP_NVCC_EXTRA (e.g. "-DDFP_CHECK_BOUNDS"): debug builds; the TMA kernels then verify every shared-memory index
    extra = os.environ.get("DFP_NVCC_EXTRA", "").split()
    cmd = [nvcc] + NVCC_FLAGS + extra + ["-o", LIB] + SOURCES
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode:
        raise RuntimeError("nvcc failed building libdfp.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
