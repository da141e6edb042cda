"""Compile the CPU oracle with gcc: oracle/oracle.c -> oracle/liboracle.so (single thread, the
authority) and oracle/oracle_omp.c -> oracle/liboracle_omp.so (its threaded twin, -fopenmp;
SURVEY.md section 8(d)(ii)).

Test infrastructure only.  Flags: -O2 -ffp-contract=off (no fused multiply-add: every
operation of the arithmetic contract is rounded on its own), no
-ffast-math, no -march=native.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle.c")
LIB = os.path.join(HERE, "liboracle.so")
FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra"]


SRC_OMP = os.path.join(HERE, "oracle_omp.c")
LIB_OMP = os.path.join(HERE, "liboracle_omp.so")
SRC_FIELD = os.path.join(HERE, "oracle_field.c")
LIB_FIELD = os.path.join(HERE, "liboracle_field.so")


def _compile(src, lib, extra, force):
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(src):
        return lib
    subprocess.run(["gcc", *FLAGS, *extra, "-o", lib, src, "-lm"], check=True)
    return lib


def build(force: bool = False) -> str:
    """The single-thread oracle (mover, arranger, deposition)."""
    return _compile(SRC, LIB, [], force)


def build_omp(force: bool = False) -> str:
    """The threaded twin (mover, arranger), pinned bit-identical to the single-thread oracle."""
    return _compile(SRC_OMP, LIB_OMP, ["-fopenmp"], force)


def build_field(force: bool = False) -> str:
    """The field-solve oracle (smoother, Poisson solve, E from phi)."""
    return _compile(SRC_FIELD, LIB_FIELD, [], force)


def build_all(force: bool = False):
    return [build(force), build_omp(force), build_field(force)]


if __name__ == "__main__":
    print("\n".join(build_all(force="--force" in sys.argv)))
