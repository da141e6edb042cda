"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md section 4).

This module serves both the CUDA path and the CPU oracle and therefore holds NONE of the
method's arithmetic (no gather, no Boris step, no sort): it only draws E, B and an initial,
cell-grouped particle state with numpy's PCG64.  It imports neither the oracle nor libpic.

The paper's workloads are BIT1 input decks (ionisation case PAPER.md:158, sheath case
PAPER.md:159) that are not available; these inputs take their shape (1D grid, particles per
cell, species, magnetised double-bounded slab with absorbing walls) and stand in for them.

Draw order (fixed): E amplitudes, E phases, E noise, then per species: x offsets, vx, vy, vz.
Seed = 260324508 + config number (+1000 per additional species).  dx = 1, dt = 0.1 everywhere.
"""
import math

import numpy as np

PERIODIC, ABSORBING = 0, 1
SEED0 = 260324508
DX, DT = 1.0, 0.1

# name, nc, ppc, boundary, E kind, modes, (omega_c*dt, theta_deg), v_th, steps, arrange_every
CONFIGS = {
    1: dict(name="oracle-scale periodic", nc=1024, ppc=64, boundary=PERIODIC, modes=4, sheath=False, noise=0.0,
            wcdt=0.2, theta=45.0, vth=1.0, steps=200, arrange_every=1, species=("e",), density="uniform"),
    2: dict(name="absorbing single species", nc=65536, ppc=160, boundary=ABSORBING, modes=8, sheath=False, noise=0.0,
            wcdt=0.2, theta=85.0, vth=1.0, steps=100, arrange_every=1, species=("e",), density="uniform"),
    3: dict(name="two-species plasma-edge slab", nc=100000, ppc=200, boundary=ABSORBING, modes=0, sheath=True,
            noise=1e-3, wcdt=0.2, theta=85.0, vth=1.0, steps=200, arrange_every=1, species=("e", "D+"),
            density="uniform"),
    4: dict(name="bandwidth-scale periodic", nc=1000000, ppc=100, boundary=PERIODIC, modes=16, sheath=False, noise=0.0,
            wcdt=0.2, theta=45.0, vth=1.0, steps=50, arrange_every=1, species=("e",), density="uniform"),
    5: dict(name="non-uniform fast-particle sort stress", nc=262144, ppc=None, n_total=50_000_000, boundary=ABSORBING,
            modes=4, sheath=True, noise=0.0, wcdt=0.5, theta=60.0, vth=4.0, steps=100, arrange_every=10,
            species=("e",), density="gaussian"),
}
QM = {"e": -1.0, "D+": 1.0 / 3672.0}
MASS_RATIO = 3672.0


def field(cfg, nc, rng):
    """E_x on nc+1 nodes (readings S14-S17 of DESIGN.md)."""
    j = np.arange(nc + 1, dtype=np.float64)
    L = float(nc) * DX
    E = np.zeros(nc + 1)
    M = cfg["modes"]
    amp = 0.05 * rng.random(M) if M else np.zeros(0)
    phase = 2.0 * math.pi * rng.random(M) if M else np.zeros(0)
    noise = rng.uniform(-cfg["noise"], cfg["noise"], nc + 1) if cfg["noise"] else None
    if cfg["sheath"]:
        x = j * DX
        E += 0.5 * (np.exp(-x / 20.0) - np.exp(-(L - x) / 20.0))
    for m in range(M):
        E += amp[m] * np.sin(2.0 * math.pi * (m + 1) * j / nc + phase[m])
    if noise is not None:
        E += noise
    if cfg["boundary"] == PERIODIC:
        E[nc] = E[0]
    return E


def cell_counts(cfg, nc, ppc, n_total):
    if cfg["density"] == "uniform":
        return np.full(nc, ppc, dtype=np.int64)
    # S18: density ~ 1 + 99*exp(-(x-L/2)^2/(2 sigma^2)), sigma = L/10; counts by differencing the
    # rounded cumulative target so the total is exactly n_total
    xc = (np.arange(nc) + 0.5) * DX
    L = nc * DX
    dens = 1.0 + 99.0 * np.exp(-((xc - 0.5 * L) ** 2) / (2.0 * (0.1 * L) ** 2))
    cum = np.concatenate([[0.0], np.cumsum(dens)])
    target = np.rint(cum / cum[-1] * n_total).astype(np.int64)
    return np.diff(target)


def particles(counts, vth, rng):
    """Cell-grouped initial state: x = c + u, v = vth * N(0,1); guard against c+u rounding to c+1."""
    nc = len(counts)
    n = int(counts.sum())
    cell = np.repeat(np.arange(nc, dtype=np.int32), counts)
    x = cell.astype(np.float64) + rng.random(n)
    bad = np.floor(x) != cell
    if bad.any():
        x[bad] = np.nextafter(cell[bad].astype(np.float64) + 1.0, 0.0)
    vx = vth * rng.standard_normal(n)
    vy = vth * rng.standard_normal(n)
    vz = vth * rng.standard_normal(n)
    assert np.array_equal(np.floor(x).astype(np.int32), cell) and x.min() >= 0.0 and x.max() < nc
    return x, vx, vy, vz, cell


def make(config, *, nc=None, ppc=None, n_total=None, steps=None, replica=0):
    """Inputs of BASELINE.json config `config` (1..5), optionally scaled down (nc / ppc / n_total /
    steps overrides, used by the parity tests).  replica > 0 draws an independent replica of the same
    workload (seed + 100000*replica; bench.py gives every rank its own).  Returns a dict of plain
    numpy arrays and scalars."""
    cfg = CONFIGS[config]
    nc = int(nc if nc is not None else cfg["nc"])
    ppc = ppc if ppc is not None else cfg["ppc"]
    if cfg["density"] == "gaussian":
        n_total = int(n_total if n_total is not None else round(cfg["n_total"] * (nc / cfg["nc"])))
    seed = SEED0 + config + 100000 * int(replica)
    rng = np.random.Generator(np.random.PCG64(seed))
    E = field(cfg, nc, rng)
    B0 = cfg["wcdt"] / (abs(QM["e"]) * DT)
    th = math.radians(cfg["theta"])
    B = np.array([B0 * math.cos(th), B0 * math.sin(th), 0.0])
    counts = cell_counts(cfg, nc, ppc, n_total)
    species = []
    for si, name in enumerate(cfg["species"]):
        srng = rng if si == 0 else np.random.Generator(np.random.PCG64(seed + 1000 * si))
        vth = cfg["vth"] if name == "e" else cfg["vth"] * math.sqrt(1.0 / MASS_RATIO)
        x, vx, vy, vz, cell = particles(counts, vth, srng)
        species.append(dict(name=name, qm=QM[name], x=x, vx=vx, vy=vy, vz=vz, cell=cell))
    return dict(config=config, name=cfg["name"], nc=nc, dx=DX, dt=DT, boundary=cfg["boundary"], E=E, B=B,
                species=species, steps=int(steps if steps is not None else cfg["steps"]),
                arrange_every=cfg["arrange_every"], numpy=np.__version__)
