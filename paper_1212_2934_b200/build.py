"""Build libff.so (the C-ABI CUDA library of include/ff.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libff.so")
SO_CHECKED = os.path.join(HERE, "libff_checked.so")      # the same sources with -DFF_CHECKED (device-side bound checks)

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--fmad=true",            # contraction is fine in the sums; the key and opening-test code uses _rn intrinsics
    "-Xcompiler", "-fPIC", "-shared",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def needs_build(so: str = SO) -> bool:
    if not os.path.exists(so):
        return True
    t = os.path.getmtime(so)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "ff.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """checked=True builds libff_checked.so: every kernel with its index and bound checks compiled in (FF_CHECK in
    csrc/ff_internal.cuh); the binding loads it when FF_CHECKED=1 is set in the environment."""
    so = SO_CHECKED if checked else SO
    if force or needs_build(so):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = so + ".tmp.%d" % os.getpid()
        cmd = [nvcc, *NVCC_FLAGS, *(["-DFF_CHECKED"] if checked else []), *(["-Xptxas", "-v"] if verbose else []),
               "-o", tmp, *sources()]
        subprocess.check_call(cmd)
        os.replace(tmp, so)
    return so


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
