"""Pins for the threaded twin of the oracle (oracle/oracle_omp.c, the design the
paper used for `arrj`).  CPU only.

The single-thread oracle (oracle/oracle.c) is the authority and is itself pinned by test_oracle_mover.py /
test_oracle_arranger.py.  The twin must reproduce it BIT FOR BIT -- all five arrays, counts, offsets, walls,
step and slot counts -- for 1, 2, 3 and all host threads: the mover is independent per particle and the stable
counting sort has a unique result, so nothing may depend on how the index range is cut.  Only then may
tests/test_gpu_fullsize.py use it for whole-run, element-wise parity at BASELINE.json's full sizes, and bench.py
report it as the N-core cpu_baseline.
"""
import numpy as np
import pytest

import oracle
from paper_2603_24508_b200 import workloads

THREADS = sorted({1, 2, 3, oracle.omp_max_threads()})


def _states(inp, si, threads, arrange_every=None):
    s = inp["species"][si]
    ae = inp["arrange_every"] if arrange_every is None else arrange_every
    kw = dict(nc=inp["nc"], dx=inp["dx"], dt=inp["dt"], boundary=inp["boundary"], E=inp["E"], qm=s["qm"], B=inp["B"],
              arrange_every=ae)
    args = (s["x"], s["vx"], s["vy"], s["vz"], s["cell"])
    return oracle.State(*args, **kw), oracle.State(*args, threads=threads, **kw)


def _same(a, b, where):
    assert a.n == b.n and a.steps == b.steps, where
    for name, p, q in zip(("x", "vx", "vy", "vz", "cell"), a.live(), b.live()):
        assert np.array_equal(p, q), f"{where}: {name} differs at {np.flatnonzero(p != q)[:8]}"
    assert np.array_equal(a.wall, b.wall), where
    assert np.array_equal(a.count, b.count) and np.array_equal(a.offset, b.offset), where


@pytest.mark.parametrize("threads", THREADS)
def test_config1_in_full_bit_identical(threads):
    inp = workloads.make(1)
    a, b = _states(inp, 0, threads)
    for k in (1, 7, 92, 100):  # 200 steps, split unevenly over calls
        a.push(k)
        b.push(k)
        _same(a, b, f"config 1, {threads} threads, after {a.steps} steps")


# reduced sizes of configs 2-5 (absorbing walls: dead particles appear and are compacted; config 5 arranges every
# 10th step, so flagged-dead particles sit in the arrays between arranges and |dcell| grows to ~12)
REDUCED = [(2, dict(nc=512), 60), (3, dict(nc=400), 50), (4, dict(nc=3000, ppc=20), 30), (5, dict(nc=2048), 60)]


@pytest.mark.parametrize("threads", THREADS)
@pytest.mark.parametrize("config,kw,steps", REDUCED)
def test_reduced_configs_bit_identical(config, kw, steps, threads):
    inp = workloads.make(config, **kw)
    for si in range(len(inp["species"])):
        a, b = _states(inp, si, threads)
        done = 0
        for k in (1, 2, steps // 2, steps - steps // 2 - 3):
            a.push(k)
            b.push(k)
            done += k
            _same(a, b, f"config {config} species {si}, {threads} threads, after {done} steps")
        if inp["boundary"] == workloads.ABSORBING and si == 0:
            assert a.wall.sum() > 0, "the reduced case must absorb something, or compaction is not exercised"


@pytest.mark.parametrize("threads", THREADS)
def test_push_and_arrange_separately_with_dead_and_unsorted_input(threads):
    """oracle_omp_push / oracle_omp_arrange on their own: unsorted input, dead particles present, empty cells."""
    rng = np.random.default_rng(5 + threads)
    nc, n = 97, 5000
    x = rng.uniform(0, nc, n)
    x[(x > 30) & (x < 41)] = 29.5  # cells 30..40 empty
    v = rng.normal(size=(3, n)) * 6.0
    cell = np.floor(x).astype(np.int32)
    E = 0.1 * rng.normal(size=nc + 1)
    kw = dict(nc=nc, dx=1.0, dt=0.1, boundary=oracle.ABSORBING, E=E, qm=-1.0, B=np.array([1.0, 2.0, 0.5]))
    a = oracle.State(x, v[0], v[1], v[2], cell, **kw)
    b = oracle.State(x, v[0], v[1], v[2], cell, threads=threads, **kw)
    for rnd in range(4):
        for _ in range(5):
            a.push_only()
            b.push_only()
        assert np.array_equal(a.cell, b.cell) and np.array_equal(a.x, b.x) and np.array_equal(a.wall, b.wall)
        assert (a.cell[:a.n] < 0).any(), "dead particles must be present before the arrange"
        a.arrange()
        b.arrange()
        _same(a, b, f"round {rnd}, {threads} threads")


def test_more_threads_than_particles_and_empty_input():
    kw = dict(nc=8, dx=1.0, dt=0.1, boundary=oracle.PERIODIC, E=np.zeros(9), qm=-1.0, B=np.zeros(3), arrange_every=1)
    for n in (0, 1, 2, 5):
        x = np.linspace(0.5, 7.5, n) if n else np.zeros(0)
        v = np.ones(n)
        a = oracle.State(x, v, v, v, np.floor(x).astype(np.int32), **kw)
        b = oracle.State(x, v, v, v, np.floor(x).astype(np.int32), threads=0, **kw)
        a.push(12)
        b.push(12)
        _same(a, b, f"n = {n}")


def test_twin_rejects_stale_cell_and_out_of_domain():
    kw = dict(nc=8, dx=1.0, dt=0.1, boundary=oracle.PERIODIC, E=np.zeros(9), qm=-1.0, B=np.zeros(3))
    x = np.array([1.5, 2.5, 3.5])
    v = np.zeros(3)
    st = oracle.State(x, v, v, v, np.array([1, 2, 4], dtype=np.int32), threads=2, **kw)
    with pytest.raises(RuntimeError):
        st.push_only()
    st = oracle.State(np.array([1.5, 99.0]), v[:2], v[:2], v[:2], np.array([1, 7], dtype=np.int32), threads=2, **kw)
    with pytest.raises(RuntimeError):
        st.push_only()
