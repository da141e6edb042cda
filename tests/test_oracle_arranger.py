"""Pins for the oracle's arranger (oracle_arrange).  CPU only.

The arranger reaches a result with a plain definition -- the stable sort of the live
particles by cell (`arrj` PAPER.md:200, `rempar2` PAPER.md:202) -- so it
is pinned against that definition computed two other ways: an O(N^2) rank count written
out in Python, and numpy's stable argsort (a library routine), plus the printed tiny case
and the invariants P9/P10.
"""
import os

import numpy as np
import pytest

import oracle


def brute_force_destinations(cell, nc):
    """dst[i] = #{live j : cell_j < cell_i} + #{live j < i : cell_j == cell_i}; O(N^2)."""
    n = len(cell)
    dst = [-1] * n
    for i in range(n):
        if cell[i] < 0:
            continue
        d = 0
        for j in range(n):
            if cell[j] < 0:
                continue
            if cell[j] < cell[i] or (cell[j] == cell[i] and j < i):
                d += 1
        dst[i] = d
    return dst


def payload(n, rng):
    return [rng.normal(size=n) for _ in range(4)]


def test_printed_tiny_case(golden_dir):
    rows = {}
    for line in open(os.path.join(golden_dir, "arranger_tiny.txt")):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split()
            rows[k] = [int(t) for t in v]
    cell = np.array(rows["cells"], dtype=np.int32)
    ids = np.arange(len(cell), dtype=np.float64)
    xo, vxo, vyo, vzo, co, count, offset, nl = oracle.arrange_arrays(ids, ids + 0.5, -ids, ids * 2, cell, 3)
    assert list(count) == rows["count"] and list(offset) == rows["offset"] and nl == 7
    assert list(xo.astype(int)) == rows["source_order"]
    src = np.array(rows["source_order"])
    assert np.array_equal(vxo, src + 0.5) and np.array_equal(vyo, -src.astype(float)) and np.array_equal(vzo, 2.0 * src)
    assert list(co) == sorted(c for c in rows["cells"] if c >= 0)


@pytest.mark.parametrize("seed", range(12))
def test_P8_brute_force_rank_small(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(0, 17))
    nc = int(rng.integers(1, 6))
    cell = rng.integers(-1, nc, size=n).astype(np.int32)
    x, vx, vy, vz = payload(n, rng)
    xo, vxo, vyo, vzo, co, count, offset, nl = oracle.arrange_arrays(x, vx, vy, vz, cell, nc)
    dst = brute_force_destinations(cell, nc)
    assert nl == sum(1 for c in cell if c >= 0)
    for i in range(n):
        if dst[i] >= 0:
            d = dst[i]
            assert (xo[d], vxo[d], vyo[d], vzo[d], co[d]) == (x[i], vx[i], vy[i], vz[i], cell[i])
    assert list(count) == [int(np.count_nonzero(cell == c)) for c in range(nc)]
    assert list(offset) == [int(np.count_nonzero((cell >= 0) & (cell < c))) for c in range(nc + 1)]


@pytest.mark.parametrize("n,nc,dead_frac", [(5000, 37, 0.0), (20000, 1024, 0.1), (3000, 1, 0.5), (4096, 100000, 0.01)])
def test_matches_numpy_stable_argsort(n, nc, dead_frac):
    rng = np.random.default_rng(n + nc)
    cell = rng.integers(0, nc, size=n).astype(np.int32)
    cell[rng.uniform(size=n) < dead_frac] = -1
    x, vx, vy, vz = payload(n, rng)
    xo, vxo, vyo, vzo, co, count, offset, nl = oracle.arrange_arrays(x, vx, vy, vz, cell, nc)
    live = np.flatnonzero(cell >= 0)
    order = live[np.argsort(cell[live], kind="stable")]
    assert nl == len(live)
    for got, src in zip((xo, vxo, vyo, vzo, co), (x, vx, vy, vz, cell)):
        assert np.array_equal(got, src[order])
    assert np.array_equal(count, np.bincount(cell[live], minlength=nc))
    assert np.array_equal(offset, np.concatenate([[0], np.cumsum(count)]))
    assert np.all(np.diff(co) >= 0) and offset[nc] == nl


def test_P10_idempotent_and_identity_on_arranged_input():
    rng = np.random.default_rng(3)
    n, nc = 6000, 200
    cell = rng.integers(-1, nc, size=n).astype(np.int32)
    a = payload(n, rng)
    once = oracle.arrange_arrays(*a, cell, nc)
    twice = oracle.arrange_arrays(*once[:5], nc)
    for p, q in zip(once[:7], twice[:7]):
        assert np.array_equal(p, q)
    assert once[7] == twice[7]


def test_edge_cases_empty_all_dead_single_cell():
    e = np.zeros(0)
    out = oracle.arrange_arrays(e, e, e, e, np.zeros(0, dtype=np.int32), 4)
    assert out[7] == 0 and list(out[5]) == [0, 0, 0, 0] and list(out[6]) == [0] * 5
    d = np.arange(5.0)
    out = oracle.arrange_arrays(d, d, d, d, np.full(5, -1, dtype=np.int32), 3)
    assert out[7] == 0 and out[6][3] == 0
    out = oracle.arrange_arrays(d, d, d, d, np.zeros(5, dtype=np.int32), 1)
    assert out[7] == 5 and np.array_equal(out[0], d) and list(out[6]) == [0, 5]


def test_out_of_range_cell_is_rejected():
    d = np.arange(3.0)
    with pytest.raises(RuntimeError):
        oracle.arrange_arrays(d, d, d, d, np.array([0, 3, 1], dtype=np.int32), 3)
