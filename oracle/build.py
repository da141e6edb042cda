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


# ORACLE_SANITIZE=1: build and load AddressSanitizer + UndefinedBehaviorSanitizer variants (separate files) instead;
# run the oracle's own test-suite under them with
#   LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 ORACLE_SANITIZE=1 \
#       python -m pytest tests/test_oracle_mover.py tests/test_oracle_arranger.py tests/test_oracle_deposit.py \
#       tests/test_oracle_omp.py tests/test_oracle_field.py -q
SANITIZE = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
SAN_FLAGS = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]


def _compile(src, lib, extra, force):
    flags = list(FLAGS)
    if SANITIZE:
        lib = lib[:-3] + "_san.so"
        flags = [f for f in flags if f != "-O2"] + SAN_FLAGS
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(src):
        return lib
    subprocess.run(["gcc", *flags, *extra, "-o", lib, src, "-lm"], check=True)
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
