"""Compile the CUDA kernels + C ABI into paper_2603_19764_b200/libsph.so (sm_100a only).

    python -m paper_2603_19764_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  -lineinfo keeps ncu's source page usable.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "libsph.so")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def stale() -> bool:
    return _stale()


def _stale() -> bool:
    if not os.path.exists(OUT):
        return True
    t = os.path.getmtime(OUT)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "sph.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, out: str | None = None, defines=()) -> str:
    """out / defines: a second library with other compile-time constants (e.g. defines=("SPH_UBAND=1.0e-3f",), which
    tests/test_gpu_band.py loads through SPH_LIB to drive the rare paths of k_pair_l); the default builds libsph.so."""
    target = out or OUT
    if out is None and not force and not _stale():
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = target + ".tmp.%d" % os.getpid()           # never leave a half-written library where load() looks
    cmd = [nvcc, "-O3", "-std=c++17", *ARCH, "-lineinfo", "-diag-suppress", "128", "-Xcompiler", "-fPIC", "-shared",
           *["-D" + d for d in defines], "-o", tmp, *sources()]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    try:
        subprocess.check_call(cmd)
        os.replace(tmp, target)
    finally:
        if os.path.exists(tmp):
            os.remove(tmp)
    return target


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
