"""Builds oracle/liboracle.so from oracle/opx_oracle.cpp with g++ (no CUDA, no nvcc).

TEST INFRASTRUCTURE.  `-ffp-contract=off` so that only the fused multiply-adds written in
the source are fused; `-mfma` so that those compile to one instruction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "opx_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-mfma", "-fno-fast-math", "-fPIC", "-shared",
         "-pthread", "-Wall"]


def build(force=False):
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", *FLAGS, SRC, "-o", LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
