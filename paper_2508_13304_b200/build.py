"""Build libdfp.so (the C-ABI CUDA library, include/dfp.h) and libdfp_bench.so (the roofline probes, include/dfp_bench.h)
in-tree with nvcc for sm_100a.

    python -m paper_2508_13304_b200.build [--force]

The .so files are git-ignored but travel with the tree to the GPU box; nothing is JIT-compiled at import time on
a machine without nvcc - if the library is missing there, importing the binding fails loudly.
"""
import glob
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libdfp.so")
LIB_BENCH = os.path.join(HERE, "libdfp_bench.so")
SOURCES = [os.path.join(CSRC, "dfp_api.cu")]
BENCH_SOURCES = [os.path.join(CSRC, "dfp_microbench.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _deps(sources, header):
    # every header of csrc/ (each is included by dfp_api.cu) and the public header
    return sources + sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h"))) + \
        [os.path.join(INCLUDE, header)]


def _stale(lib, deps) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in deps)


def stale() -> bool:
    return _stale(LIB, _deps(SOURCES, "dfp.h"))


def _nvcc(lib, sources, verbose):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        raise RuntimeError(f"nvcc not found: cannot build {os.path.basename(lib)} (there is no CPU fallback)")
    # DFP_NVCC_EXTRA (e.g. "-DDFP_CHECK_BOUNDS"): debug builds; the TMA kernels then verify every shared-memory index
    extra = os.environ.get("DFP_NVCC_EXTRA", "").split()
    res = subprocess.run([nvcc] + NVCC_FLAGS + extra + ["-o", lib] + sources, capture_output=True, text=True)
    if verbose or res.returncode:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode:
        raise RuntimeError(f"nvcc failed building {os.path.basename(lib)}")
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    return _nvcc(LIB, SOURCES, verbose)


def build_bench(force: bool = False, verbose: bool = False) -> str:
    deps = BENCH_SOURCES + [os.path.join(INCLUDE, "dfp_bench.h")]
    if not force and not _stale(LIB_BENCH, deps):
        return LIB_BENCH
    if not (shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc")) and os.path.exists(LIB_BENCH):
        return LIB_BENCH                     # a box without nvcc uses the prebuilt in-tree library as is
    return _nvcc(LIB_BENCH, BENCH_SOURCES, verbose)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
    print(build_bench(force="--force" in sys.argv, verbose=False))
