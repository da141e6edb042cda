"""Build libpic.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2603_24508_b200.build [--force] [--verbose]

Flags: -O3 -lineinfo, -fmad=false (no fused multiply-add: the arithmetic contract of DESIGN.md
section 3 is also written with __d*_rn intrinsics, this is the belt to those braces), host code
with -ffp-contract=off.  The .so is git-ignored but travels to the GPU box with the snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpic.so")
SOURCES = [os.path.join(CSRC, "pic.cu")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-fmad=false", "-shared", "-Xcompiler", "-fPIC,-ffp-contract=off,-Wall",
         "-cudart", "static", "-ldl"]


def _deps():
    out = list(SOURCES) + [os.path.join(HERE, "..", "include", "pic.h")]
    for f in os.listdir(CSRC):
        if f.endswith(".cuh"):
            out.append(os.path.join(CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB):
        t = os.path.getmtime(LIB)
        if all(os.path.getmtime(d) <= t for d in _deps()):
            return LIB
    cmd = ["nvcc", *ARCH, *FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", LIB, *SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
