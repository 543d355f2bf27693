"""Builds paper_2309_12496_b200/lib/libopx.so from csrc/*.cu with nvcc for sm_100a.

In-tree on purpose: the built library travels to the GPU box with the repo snapshot.
`-fmad=false`: only the fused multiply-adds written as intrinsics are fused.
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIBDIR = os.path.join(HERE, "lib")
LIB = os.path.join(LIBDIR, "libopx.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-fmad=false",
         "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall", "-shared"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(HERE, "..", "include", "opx.h")]


def build(force=False, verbose=False):
    """OPX_NVCC_FLAGS (environment, optional): extra nvcc flags, e.g. the -D switches of the measured-and-rejected
    variants that profiles/ names (a build with them is for measuring, not the product; it always rebuilds)."""
    os.makedirs(LIBDIR, exist_ok=True)
    extra = os.environ.get("OPX_NVCC_FLAGS", "").split()
    if not force and not extra and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    cmd = [NVCC, *FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), *sources(), "-o", LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
