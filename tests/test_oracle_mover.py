"""Pins for the oracle's mover (oracle_push / oracle_boris_constants).  CPU only.

None of these retypes the oracle's formula: they are closed forms and invariants of the
Boris scheme (BASELINE.json north_star), a library routine
(numpy.interp) for the gather, an independent extended-precision Rodrigues-rotation form,
and the printed worked example tests/golden/boris_worked_example.txt.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import oracle
from oracle import ABSORBING, PERIODIC


def make(x, v, *, nc, E=None, B=(0, 0, 0), qm=-1.0, dx=1.0, dt=0.1, boundary=PERIODIC, arrange_every=0):
    x = np.atleast_1d(np.asarray(x, dtype=np.float64))
    v = np.atleast_2d(np.asarray(v, dtype=np.float64))
    E = np.zeros(nc + 1) if E is None else np.asarray(E, dtype=np.float64)
    inv_dx = 1.0 / dx
    cell = np.minimum(np.floor(x * inv_dx).astype(np.int32), nc - 1)
    return oracle.State(x, v[:, 0], v[:, 1], v[:, 2], cell, nc=nc, dx=dx, dt=dt, boundary=boundary, E=E, qm=qm,
                        B=B, arrange_every=arrange_every)


def tilted_B(omega_dt, theta_deg, dt=0.1, qm=-1.0):
    B0 = omega_dt / (abs(qm) * dt)
    th = math.radians(theta_deg)
    return np.array([B0 * math.cos(th), B0 * math.sin(th), 0.0])


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("omega_dt,theta", [(0.2, 45.0), (0.2, 85.0), (0.5, 60.0)])
def test_P1_speed_conserved_without_E(omega_dt, theta):
    rng = np.random.default_rng(1)
    n = 64
    st = make(rng.uniform(0, 1024, n), rng.normal(size=(n, 3)), nc=1024, B=tilted_B(omega_dt, theta))
    s0 = np.sqrt(st.vx**2 + st.vy**2 + st.vz**2)
    for _ in range(200):
        st.push_only()
    s1 = np.sqrt(st.vx**2 + st.vy**2 + st.vz**2)
    assert np.max(np.abs(s1 - s0) / s0) <= 1e-13


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("omega_dt,expected", [(0.2, 0.19933730498232408), (0.5, 0.48995732625372829)])
@pytest.mark.parametrize("qm", [-1.0, +1.0])
def test_P2_rotation_angle_and_sense(omega_dt, expected, qm):
    assert abs(2 * math.atan(omega_dt / 2) - expected) < 1e-16
    B = tilted_B(omega_dt, 37.0)
    bhat = B / np.linalg.norm(B)
    rng = np.random.default_rng(2)
    v0 = rng.normal(size=(8, 3))
    st = make(np.full(8, 50.0), v0, nc=100, B=B, qm=qm)
    st.push_only()
    v1 = np.stack([st.vx, st.vy, st.vz], axis=1)
    par0, par1 = v0 @ bhat, v1 @ bhat
    assert np.max(np.abs(par1 - par0)) <= 1e-14
    p0 = v0 - np.outer(par0, bhat)
    p1 = v1 - np.outer(par1, bhat)
    ang = np.arctan2(np.cross(p0, p1) @ bhat, np.sum(p0 * p1, axis=1))
    sense = +1.0 if qm < 0 else -1.0  # right-hand rotation about b for q<0
    assert np.max(np.abs(ang - sense * expected)) <= 1e-14


# ---------------------------------------------------------------- P3
def test_P3_constant_acceleration_closed_form():
    nc, dt, qm, E0 = 4096, 0.125, -1.0, 0.5  # binary-exact so the closed form is exact to a few ulp
    x0, v0 = 2000.0, np.array([0.75, -0.25, 1.5])
    st = make(x0, v0, nc=nc, E=np.full(nc + 1, E0), dt=dt, qm=qm)
    a = qm * E0
    for n in range(1, 201):
        st.push_only()
        vn = v0[0] + n * a * dt
        xn = x0 + n * v0[0] * dt + a * dt * dt * n * (n + 1) / 2
        assert abs(st.vx[0] - vn) <= 4e-16 * n * max(1.0, abs(vn))
        assert abs(st.x[0] - xn) <= 4e-16 * n * abs(xn)
        assert st.vy[0] == v0[1] and st.vz[0] == v0[2]


# ---------------------------------------------------------------- P4
@pytest.mark.parametrize("qm", [-1.0, 1.0 / 3672.0])
def test_P4_ExB_drift_is_a_fixed_point(qm):
    nc, Ex, B0 = 64, 0.03125, 2.0
    st = make(32.0, [0.0, 0.0, Ex / B0], nc=nc, E=np.full(nc + 1, Ex), B=(0.0, B0, 0.0), qm=qm)
    for _ in range(50):
        st.push_only()
        assert abs(st.vx[0]) <= 1e-15 and abs(st.vy[0]) <= 1e-15
        assert abs(st.vz[0] - Ex / B0) <= 1e-15


def test_P4_parallel_acceleration_and_gyro_averaged_drift():
    nc, Ex, dt, qm = 4096, 0.01, 0.1, -1.0
    theta = 60.0
    B = tilted_B(0.2, theta)
    B0 = np.linalg.norm(B)
    bhat = B / B0
    st = make(2048.0, [0.1, 0.2, -0.3], nc=nc, E=np.full(nc + 1, Ex), B=B, qm=qm, dt=dt)
    period = 2 * math.pi / 0.19933730498232408  # steps per gyration
    nsteps = int(round(40 * period))
    vs = []
    par_prev = np.array([st.vx[0], st.vy[0], st.vz[0]]) @ bhat
    for _ in range(nsteps):
        st.push_only()
        v = np.array([st.vx[0], st.vy[0], st.vz[0]])
        par = v @ bhat
        assert abs((par - par_prev) - qm * Ex * math.cos(math.radians(theta)) * dt) <= 1e-15
        par_prev = par
        vs.append(v - par * bhat)
    drift = np.mean(vs, axis=0)
    expected = np.array([0.0, 0.0, Ex * math.sin(math.radians(theta)) / B0])  # E x B / B^2
    assert np.max(np.abs(drift - expected)) <= 1e-2 * abs(expected[2]) + 1e-5


# ---------------------------------------------------------------- P5
def test_P5_implicit_boris_identity():
    rng = np.random.default_rng(5)
    n, nc, dt = 256, 32, 0.1
    for qm in (-1.0, 1.0 / 3672.0, 2.5):
        B = rng.normal(size=3) * 3
        E0 = 0.37
        v0 = rng.normal(size=(n, 3)) * 2
        st = make(rng.uniform(0, nc, n), v0, nc=nc, E=np.full(nc + 1, E0), B=B, qm=qm, dt=dt,
                  boundary=ABSORBING)
        st.push_only()
        v1 = np.stack([st.vx, st.vy, st.vz], axis=1)
        h = qm * dt / 2
        t = h * B
        Evec = np.array([E0, 0.0, 0.0])
        resid = v1 - v0 - 2 * h * Evec - np.cross(v1 + v0, t)
        scale = np.linalg.norm(v0, axis=1) + np.linalg.norm(v1, axis=1) + 1.0
        assert np.max(np.linalg.norm(resid, axis=1) / scale) <= 1e-15


# ---------------------------------------------------------------- P6
def test_P6_field_aligned_B_leaves_x_motion_unmagnetised():
    rng = np.random.default_rng(6)
    n, nc = 128, 256
    E = 0.05 * np.sin(2 * np.pi * np.arange(nc + 1) / nc)
    E[nc] = E[0]
    x0, v0 = rng.uniform(0, nc, n), rng.normal(size=(n, 3))
    a = make(x0, v0, nc=nc, E=E, B=(2.0, 0.0, 0.0))
    b = make(x0, v0, nc=nc, E=E, B=(0.0, 0.0, 0.0))
    for _ in range(100):
        a.push_only()
        b.push_only()
        assert np.array_equal(a.x, b.x) and np.array_equal(a.vx, b.vx)
    assert not np.array_equal(a.vy, b.vy)


# ---------------------------------------------------------------- P7
def _parse_golden(path):
    cases, cur = [], None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "case":
            cur = {"steps": {}}
            cases.append(cur)
        elif tok[0] == "step":
            cur["steps"][int(tok[1])] = ([float(t) for t in tok[2:6]], int(tok[6]))
        elif tok[0] in ("h", "t", "s", "step1hex"):
            cur[tok[0]] = [float.fromhex(t) for t in tok[1:]]
        elif tok[0] == "B":
            cur["B"] = [float(t) for t in tok[1:]]
    return cases


def test_P7_printed_worked_example_bitwise(golden_dir):
    E = np.array([0, 0.015625, -0.03125, 0.03125, -0.0625, 0.125, 0, 0], dtype=np.float64)
    for case in _parse_golden(os.path.join(golden_dir, "boris_worked_example.txt")):
        k = oracle.boris_constants(-1.0, 0.1, 1.0, case["B"])
        if "h" in case:
            assert k["h"] == case["h"][0]
        if "t" in case:
            assert list(k["t"]) == case["t"]
        assert list(k["s"]) == case["s"]  # -0.0 == 0.0 numerically, as the contract allows
        st = make(3.75, [0.5, -1.25, 2.0], nc=7, E=E, B=case["B"], boundary=ABSORBING)
        for step in range(1, max(case["steps"]) + 1):
            st.push_only()
            got = [st.x[0], st.vx[0], st.vy[0], st.vz[0]]
            want, cell = case["steps"][step]
            assert got == want, (step, got, want)
            assert st.cell[0] == cell
            if step == 1 and "step1hex" in case:
                assert got == case["step1hex"]


# ---------------------------------------------------------------- P8 (mover half)
def _rodrigues_step(x, v, E, B, qm, dt, dx, nc):
    """Independent form in 60-digit arithmetic: interpolate E, half kick, rotate v about
    the axis -t/|t| by delta = 2*atan(|t|) with Rodrigues' formula, half kick, advance."""
    mp.mp.dps = 60
    X = mp.mpf(x)
    xs = X / mp.mpf(dx)
    j = int(mp.floor(xs))
    w = xs - j
    Ep = (1 - w) * mp.mpf(E[j]) + w * mp.mpf(E[j + 1])
    h = mp.mpf(qm) * mp.mpf(dt) / 2
    t = [h * mp.mpf(b) for b in B]
    tn = mp.sqrt(sum(c * c for c in t))
    u = [mp.mpf(v[0]) + h * Ep, mp.mpf(v[1]), mp.mpf(v[2])]
    if tn == 0:
        r = u
    else:
        nhat = [-c / tn for c in t]
        delta = 2 * mp.atan(tn)
        cd, sd = mp.cos(delta), mp.sin(delta)
        dot = sum(a * b for a, b in zip(nhat, u))
        cr = [nhat[1] * u[2] - nhat[2] * u[1], nhat[2] * u[0] - nhat[0] * u[2], nhat[0] * u[1] - nhat[1] * u[0]]
        r = [u[i] * cd + cr[i] * sd + nhat[i] * dot * (1 - cd) for i in range(3)]
    vn = [r[0] + h * Ep, r[1], r[2]]
    return X + vn[0] * mp.mpf(dt), vn


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_P8_mover_matches_extended_precision_rodrigues(seed):
    rng = np.random.default_rng(100 + seed)
    n, nc, dt = 16, 24, 0.1
    dx = [1.0, 0.5, 0.1][seed]
    qm = [-1.0, 1.0 / 3672.0, -1.0][seed]
    B = rng.normal(size=3) * [2.0, 500.0, 5.0][seed]
    E = rng.normal(size=nc + 1) * 0.1
    L = nc * dx
    x0 = rng.uniform(0.2 * L, 0.8 * L, n)
    v0 = rng.normal(size=(n, 3)) * (0.5 * dx / dt)
    st = make(x0, v0, nc=nc, E=E, B=B, qm=qm, dx=dx, dt=dt, boundary=ABSORBING)
    st.push_only()
    for i in range(n):
        xe, ve = _rodrigues_step(x0[i], v0[i], E, B, qm, dt, dx, nc)
        assert abs(mp.mpf(st.x[i]) - xe) <= 1e-14 * max(1, abs(xe))
        for got, want in zip((st.vx[i], st.vy[i], st.vz[i]), ve):
            assert abs(mp.mpf(got) - want) <= 1e-14 * max(1, abs(want))
        assert st.cell[i] == int(mp.floor(xe / mp.mpf(dx)))


# ---------------------------------------------------------------- gather vs library routine
@pytest.mark.parametrize("dx", [1.0, 0.5, 0.1])
def test_gather_is_linear_interpolation(dx):
    rng = np.random.default_rng(7)
    nc, n = 50, 400
    E = rng.normal(size=nc + 1)
    L = nc * dx
    x0 = rng.uniform(0, L, n)
    x0[:nc] = np.arange(nc) * dx  # exactly on nodes
    x0 = x0[x0 < L]
    n = len(x0)
    # qm*dt = 1 and v=0: vx' = (0 + Ep/2) + Ep/2 = Ep exactly
    st = make(x0, np.zeros((n, 3)), nc=nc, E=E, qm=1.0, dt=1.0, dx=dx, boundary=ABSORBING)
    st.push_only()
    want = np.interp(x0, np.arange(nc + 1) * dx, E)
    # dx a power of two: x*inv_dx is exact and only the interpolation itself rounds;
    # otherwise w = x*inv_dx - j carries the rounding of a number of size nc (ulp(nc) ~ nc*eps)
    tol = 4e-15 if dx in (1.0, 0.5) else 8 * nc * np.finfo(np.float64).eps
    assert np.max(np.abs(st.vx - want)) <= tol * np.max(np.abs(E))
    on_nodes = st.vx[:nc]
    if dx in (1.0, 0.5):
        assert np.array_equal(on_nodes, E[:nc])  # w == 0 exactly: a particle on a node sees the node value


# ---------------------------------------------------------------- boundaries (S6, S7, S8)
def test_absorbing_wall_is_half_open_and_counts():
    nc, dt = 8, 0.125
    #            stays at 0.0   left       right (==L)  right (>L)  interior
    x0 = np.array([1.0, 1.0, 7.0, 7.5, 4.0])
    vx = np.array([-8.0, -8.5, 8.0, 8.0, 1.0])
    st = make(x0, np.stack([vx, 0 * vx, 0 * vx], 1), nc=nc, dt=dt, boundary=ABSORBING)
    st.push_only()
    assert st.x[0] == 0.0 and st.cell[0] == 0
    assert list(st.cell) == [0, -1, -1, -1, 4]
    assert list(st.wall) == [1, 2]
    snap = [a.copy() for a in (st.x, st.vx, st.vy, st.vz, st.cell)]
    st.push_only()  # dead particles are never touched again and are not counted twice
    for a, b in zip((st.x, st.vx, st.vy, st.vz, st.cell), snap):
        assert np.array_equal(a[1:4], b[1:4])
    assert list(st.wall) == [2, 2]  # particle 0 (x=0, vx<0) now left through the left wall
    assert list(st.cell) == [-1, -1, -1, -1, 4]
    st.arrange()
    assert st.n == 1 and st.cell[0] == 4 and st.x[0] == 4.25


def test_periodic_wrap_cases():
    nc, dt = 8, 0.125
    x0 = np.array([7.5, 0.25, 0.0, 7.0])
    vx = np.array([8.0, -8.0, -1e-20 / dt, 8.0])
    st = make(x0, np.stack([vx, 0 * vx, 0 * vx], 1), nc=nc, dt=dt, boundary=PERIODIC)
    st.push_only()
    assert list(st.x) == [0.5, 7.25, 0.0, 0.0]
    assert list(st.cell) == [0, 7, 0, 0]
    assert list(st.wall) == [0, 0]


def test_cell_clamp_when_scaled_position_rounds_up_to_nc():
    found = None
    for nc in range(3, 400):
        for dx in (0.1, 0.3, 0.7, 1.1, 1.3, 0.01, 0.003):
            L = nc * dx
            x = np.nextafter(L, 0.0)
            if math.floor(x * (1.0 / dx)) == nc:
                found = (nc, dx, x)
                break
        if found:
            break
    assert found, "no rounding-up case in the searched range"
    nc, dx, x = found
    st = make(x, [0.0, 0.0, 0.0], nc=nc, dx=dx, boundary=ABSORBING, E=np.arange(nc + 1, dtype=np.float64))
    assert st.cell[0] == nc - 1
    st.push_only()  # gather must use cell nc-1 (w ~ 1), not read E[nc+1]
    h = -1.0 * 0.1 * 0.5
    assert abs(st.vx[0] - 2 * h * nc) <= 1e-12 * nc  # E_p = E[nc-1] + w*1 with w ~ 1, i.e. ~ nc
    assert abs(st.x[0] - (x + 2 * h * nc * 0.1)) <= 1e-15 and st.cell[0] >= 0


def test_out_of_domain_live_particle_is_rejected():
    st = make(1.0, [0.0, 0.0, 0.0], nc=4)
    st.x[0] = 9.0
    with pytest.raises(RuntimeError):
        st.push_only()


# ---------------------------------------------------------------- P9 (count conservation)
def test_P9_particle_count_plus_absorbed_is_invariant():
    rng = np.random.default_rng(9)
    nc, ppc = 64, 20
    n0 = nc * ppc
    x0 = (np.repeat(np.arange(nc), ppc) + rng.uniform(size=n0)).astype(np.float64)
    v0 = rng.normal(size=(n0, 3)) * 4.0
    E = 0.05 * rng.normal(size=nc + 1)
    st = make(x0, v0, nc=nc, E=E, B=tilted_B(0.5, 60.0), boundary=ABSORBING, arrange_every=3)
    for _ in range(40):
        st.push(1)
        live = int(np.count_nonzero(st.cell[:st.n] >= 0))
        assert live + int(st.wall[0]) + int(st.wall[1]) == n0
        if st.steps % 3 == 0:
            assert live == st.n == st.offset[nc] == st.count.sum()
            assert np.all(np.diff(st.cell[:st.n]) >= 0)
            assert np.array_equal(st.cell[:st.n], np.floor(st.x[:st.n]).astype(np.int32))
    assert st.wall[0] > 0 and st.wall[1] > 0


def test_single_call_equals_step_by_step():
    rng = np.random.default_rng(10)
    nc, ppc = 32, 8
    n0 = nc * ppc
    x0 = np.repeat(np.arange(nc), ppc) + rng.uniform(size=n0)
    v0 = rng.normal(size=(n0, 3)) * 3.0
    a = make(x0, v0, nc=nc, B=tilted_B(0.2, 85.0), boundary=ABSORBING, arrange_every=4)
    b = make(x0, v0, nc=nc, B=tilted_B(0.2, 85.0), boundary=ABSORBING, arrange_every=4)
    a.push(10)
    for k in (3, 3, 4):  # arranges fall on steps 4 and 8 however the calls are split
        b.push(k)
    assert a.n == b.n and a.steps == b.steps == 10
    for p, q in zip(a.live(), b.live()):
        assert np.array_equal(p, q)
    assert np.array_equal(a.wall, b.wall)


def test_neutral_species_is_ballistic():
    """q/m = 0 (the paper's neutral species, `nmove`): no gather, no rotation -- v is untouched
    bit for bit and x advances by the separately rounded product vx*dt each step, whatever E and B are."""
    rng = np.random.default_rng(77)
    nc, n, dt = 50, 300, 0.1
    x0 = rng.random(n) * nc
    v0 = rng.standard_normal((3, n))
    cell = np.floor(x0).astype(np.int32)
    st = oracle.State(x0, v0[0], v0[1], v0[2], cell, nc=nc, dx=1.0, dt=dt, boundary=oracle.PERIODIC,
                      E=rng.uniform(-5, 5, nc + 1), qm=0.0, B=np.array([3.0, -2.0, 7.0]), arrange_every=0)
    x = x0.copy()
    for _ in range(25):
        st.push_only()
        x = x + v0[0] * dt
        x = np.where(x >= nc, x - nc, np.where(x < 0, x + nc, x))
    assert np.array_equal(st.vx, v0[0]) and np.array_equal(st.vy, v0[1]) and np.array_equal(st.vz, v0[2])
    assert np.array_equal(st.x, x)


def test_stale_cell_index_is_rejected():
    """"j == cell by invariant (oracle asserts)".  A harness that hands the oracle a cell array
    that no longer matches floor(x/dx) must be caught, not silently pushed."""
    st = make([2.5, 7.25], [[0.1, 0, 0], [0.2, 0, 0]], nc=16)
    st.cell[1] = 6  # x = 7.25 sits in cell 7
    x_before = st.x.copy()
    with pytest.raises(RuntimeError):
        st.push_only()
    assert st.x[1] == x_before[1], "the offending particle must be left untouched"
    ok = make([2.5, 7.25], [[0.1, 0, 0], [0.2, 0, 0]], nc=16)
    ok.push_only()  # the same input with the right cells passes


def test_P7_file_is_what_its_generator_writes(golden_dir):
    """tests/golden/boris_worked_example.txt is the output of the committed scalar-float script beside it."""
    import subprocess
    import sys
    r = subprocess.run([sys.executable, os.path.join(golden_dir, "make_boris_worked_example.py"), "--check"],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
