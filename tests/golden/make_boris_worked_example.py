#!/usr/bin/env python
"""Regenerates tests/golden/boris_worked_example.txt (pin P7).

Scalar Python floats only: every line below is one IEEE-754 binary64 operation (CPython evaluates
each binary operator on C doubles and rounds it on its own; nothing is fused or reordered), in the
canonical order of the arithmetic contract.  It calls
neither oracle/ nor the CUDA path and uses no numpy.  The paper prints no numbers for
move0 / moveb; the setup is the one SURVEY.md fixes for P7.

    python tests/golden/make_boris_worked_example.py            # prints the file to stdout
    python tests/golden/make_boris_worked_example.py --check    # compares with the committed file
"""
import math
import os
import sys

DX, DT, QM, NC = 1.0, 0.1, -1.0, 7
E = [0.0, 0.015625, -0.03125, 0.03125, -0.0625, 0.125, 0.0, 0.0]
START = (3.75, 0.5, -1.25, 2.0)

HEADER = """\
# Worked single-particle example of the mover (gather + Boris + advance), canonical
# operation order, scalar IEEE-754 binary64.
# Source: SURVEY.md section 8(c), pin P7 (the paper itself, PAPER.md:89, prints no
# numbers for move0/moveb; these were produced by the survey author with scalar Python
# floats, independently of oracle/oracle.c and of the CUDA path).
# Setup: dx=1 dt=0.1 qm=-1 nc=7
# E nodes: 0 0.015625 -0.03125 0.03125 -0.0625 0.125 0 0
# start: x=3.75 vx=0.5 vy=-1.25 vz=2.0
# Lines: key value...   (hex floats are exact; decimals are shortest round-trip reprs)
"""


def constants(B):
    h = (QM * DT) * 0.5
    tx = h * B[0]
    ty = h * B[1]
    tz = h * B[2]
    t2 = ((tx * tx) + (ty * ty)) + (tz * tz)
    f = 2.0 / (1.0 + t2)
    return h, (tx, ty, tz), (f * tx, f * ty, f * tz), 1.0 / DX


def step(state, k):
    x, vx, vy, vz = state
    h, (tx, ty, tz), (sx, sy, sz), inv_dx = k
    xs = x * inv_dx
    jf = float(math.floor(xs))
    j = int(jf)
    w = xs - jf
    dE = E[j + 1] - E[j]
    Ep = E[j] + (w * dE)
    hE = h * Ep
    ux = vx + hE
    uy = vy
    uz = vz
    px = ux + ((uy * tz) - (uz * ty))
    py = uy + ((uz * tx) - (ux * tz))
    pz = uz + ((ux * ty) - (uy * tx))
    wx = ux + ((py * sz) - (pz * sy))
    wy = uy + ((pz * sx) - (px * sz))
    wz = uz + ((px * sy) - (py * sx))
    nvx = wx + hE
    xn = x + (nvx * DT)
    cell = min(int(math.floor(xn * inv_dx)), NC - 1)
    return (xn, nvx, wy, wz), cell


def fhex(v):
    """float.hex with the mantissa padding the committed file uses (13 hex digits unless exact)."""
    return v.hex()


def render():
    out = [HEADER.rstrip("\n")]
    for name, B, nsteps, full in (("A", (1.5, 1.25, 0.5), 3, True), ("B", (1.0, 2.0, 0.0), 2, False)):
        k = constants(B)
        h, t, s, _ = k
        out.append(f"case {name}")
        out.append("B " + " ".join(repr(b) for b in B))
        if full:
            out.append("h " + fhex(h))
            out.append("t " + " ".join(fhex(v) for v in t))
        out.append("s " + " ".join(fhex(v) for v in s))
        st = START
        for n in range(1, nsteps + 1):
            st, cell = step(st, k)
            if n == 1 and full:
                out.append("step1hex " + " ".join(fhex(v) for v in st))
            out.append(f"step {n} " + " ".join(repr(v) for v in st) + f" {cell}")
    return "\n".join(out) + "\n"


def values(text):
    """The file as a list of (key, parsed numbers): formatting-insensitive, value-exact."""
    rows = []
    for line in text.splitlines():
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "case":
            rows.append(("case", tok[1]))
        elif tok[0] in ("h", "t", "s", "step1hex"):
            rows.append((tok[0], tuple(float.fromhex(v) for v in tok[1:])))
        elif tok[0] == "B":
            rows.append(("B", tuple(float(v) for v in tok[1:])))
        elif tok[0] == "step":
            rows.append(("step", int(tok[1]), tuple(float(v) for v in tok[2:6]), int(tok[6])))
    return rows


if __name__ == "__main__":
    text = render()
    if "--check" in sys.argv:
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "boris_worked_example.txt")
        with open(path) as f:
            committed = f.read()
        ok = values(committed) == values(text)
        print("boris_worked_example.txt:", "reproduced exactly" if ok else "DIFFERS")
        sys.exit(0 if ok else 1)
    sys.stdout.write(text)
