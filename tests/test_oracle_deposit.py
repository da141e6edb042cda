"""Pins of the deposition oracle (oracle_deposit; PIC phase (ii); readings S20-S22 of
DESIGN.md) against what the mathematics fixes: none of them calls the oracle to check itself.

A plausible mistake fails at least one: swapped weights (first moment, single particle), a node
shifted by one (single particle, first moment), a dropped (1-w) or w term (total charge), weight
applied twice or not at all (single particle), dead particles counted (total charge), the
periodic fold missing or one-sided (fold pin), the clamp of reading S8 missing (dx != 1 pin)."""
import numpy as np
import pytest

import oracle

PER, ABS = oracle.PERIODIC, oracle.ABSORBING


def _cells(x, dx, nc):
    return np.minimum(np.floor(x * (1.0 / dx)), nc - 1).astype(np.int32)


def test_single_particle_exact_weights():
    # x = 2.25 in cell 2: 3/4 of the charge on node 2, 1/4 on node 3 (exact in binary)
    rho = oracle.deposit(np.array([2.25]), np.array([2], dtype=np.int32), 4, 1.0, ABS, weight=-2.0)
    assert rho.tolist() == [0.0, 0.0, -1.5, -0.5, 0.0]
    # on a node: everything on that node
    rho = oracle.deposit(np.array([3.0]), np.array([3], dtype=np.int32), 4, 1.0, ABS, weight=1.0)
    assert rho.tolist() == [0.0, 0.0, 0.0, 1.0, 0.0]


@pytest.mark.parametrize("boundary", [PER, ABS])
def test_total_charge_and_first_moment(boundary):
    """sum_j rho_j = weight * n_live;  sum_j j*rho_j = weight * sum_i x_i/dx (linear weighting keeps the dipole moment)."""
    rng = np.random.default_rng(5)
    nc, n, dx, wgt = 97, 5000, 0.37, 0.625
    x = rng.random(n) * nc * dx * (1 - 1e-12)
    cell = _cells(x, dx, nc)
    cell[::17] = -1  # flagged dead: skipped
    live = cell >= 0
    rho = oracle.deposit(x, cell, nc, dx, boundary, weight=wgt)
    if boundary == ABS:
        assert abs(rho.sum() - wgt * live.sum()) <= 1e-11 * wgt * live.sum()
        m1 = (np.arange(nc + 1) * rho).sum()
        ref = wgt * (x[live] * (1.0 / dx)).sum()
        assert abs(m1 - ref) <= 1e-11 * abs(ref)
    else:
        # nodes 0 and nc are one point carrying the same value: count it once
        assert rho[0] == rho[nc]
        assert abs(rho[:nc].sum() - wgt * live.sum()) <= 1e-11 * wgt * live.sum()


@pytest.mark.parametrize("boundary", [PER, ABS])
def test_one_particle_per_cell_centre(boundary):
    nc = 64
    x = np.arange(nc) + 0.5
    rho = oracle.deposit(x, _cells(x, 1.0, nc), nc, 1.0, boundary, weight=3.0)
    assert np.all(rho[1:nc] == 3.0)
    edge = 3.0 if boundary == PER else 1.5
    assert rho[0] == edge and rho[nc] == edge


def test_periodic_fold_is_symmetric():
    # one particle in the last cell close to the upper end: its w part lands on node nc == node 0
    nc = 8
    x = np.array([7.75, 0.25])
    rho = oracle.deposit(x, _cells(x, 1.0, nc), nc, 1.0, PER)
    assert rho[0] == rho[nc] == 0.75 + 0.75
    assert rho[1] == 0.25 and rho[nc - 1] == 0.25


def test_linearity_and_brute_force():
    rng = np.random.default_rng(9)
    nc, dx = 33, 1.0
    xa, xb = rng.random(700) * nc, rng.random(400) * nc
    ra = oracle.deposit(xa, _cells(xa, dx, nc), nc, dx, ABS)
    rb = oracle.deposit(xb, _cells(xb, dx, nc), nc, dx, ABS)
    xab = np.concatenate([xa, xb])
    rab = oracle.deposit(xab, _cells(xab, dx, nc), nc, dx, ABS)
    assert np.allclose(rab, ra + rb, rtol=1e-13, atol=1e-13)
    # independent formulation: numpy scatter-add of the two weights
    j = np.floor(xab).astype(int)
    w = xab - j
    ref = np.zeros(nc + 1)
    np.add.at(ref, j, 1.0 - w)
    np.add.at(ref, j + 1, w)
    assert np.allclose(rab, ref, rtol=1e-13, atol=1e-13)


def test_clamp_reading_s8_with_dx_not_one():
    """x just below L with x*(1/dx) rounding to nc: the particle belongs to cell nc-1 with w = 1 (reading S8)."""
    nc, dx = 10, 0.1
    L = nc * dx
    x = np.array([np.nextafter(L, 0.0)])
    xs = x[0] * (1.0 / dx)
    cell = np.array([nc - 1], dtype=np.int32)
    rho = oracle.deposit(x, cell, nc, dx, ABS)
    w = xs - (nc - 1)
    assert rho[nc] == w and rho[nc - 1] == 1.0 - w and 0.99 < w <= 1.0


def test_rejects_out_of_range():
    with pytest.raises(RuntimeError):
        oracle.deposit(np.array([-0.5]), np.array([0], dtype=np.int32), 4, 1.0, ABS)
