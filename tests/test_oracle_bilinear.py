"""Pins for oracle.bilinear (eq. at; readings B1-B4 in DESIGN.md).
None of these retypes the oracle's formula: they are closed forms and invariants."""
import numpy as np
import pytest

import oracle


def _grid(fn, nx, ny, x0=0.0, y0=0.0, dx=1.0, dy=1.0):
    g = oracle.geom(nx, ny, x0, y0, dx, dy)
    x = np.float32(x0) + np.arange(nx) * np.float64(np.float32(dx))
    y = np.float32(y0) + np.arange(ny) * np.float64(np.float32(dy))
    return fn(x[None, :], y[:, None]).astype(np.float32), g


def test_plane_exact():
    # a + b x + c y with dyadic coefficients: fp32 samples are exact, so the result must be the plane
    z, gi = _grid(lambda x, y: 3.0 + 0.5 * x - 0.25 * y, 9, 7, x0=2.0, y0=-1.0, dx=0.5, dy=2.0)
    go = oracle.geom(33, 25, 2.0, -1.0, 0.125, 0.5)
    out = oracle.bilinear(z, gi, go)
    X = 2.0 + np.arange(33) * 0.125
    Y = -1.0 + np.arange(25) * 0.5
    np.testing.assert_allclose(out, 3.0 + 0.5 * X[None, :] - 0.25 * Y[:, None], rtol=0, atol=1e-13)


def test_xy_on_unit_cell():
    # f = x*y is bilinear on a cell, so it is reproduced exactly: (1/2,1/2) -> 1/4, (1/4,3/4) -> 3/16
    z = np.array([[0, 0], [0, 1]], dtype=np.float32)
    gi = oracle.geom(2, 2, 0, 0, 1, 1)
    assert oracle.bilinear(z, gi, oracle.geom(1, 1, 0.5, 0.5, 1, 1))[0, 0] == 0.25
    assert oracle.bilinear(z, gi, oracle.geom(1, 1, 0.25, 0.75, 1, 1))[0, 0] == 0.1875


def test_worked_cell_2_375():
    # corners Q11=1, Q21=2, Q12=3, Q22=5 at (t,s)=(1/4,1/2):
    # bottom edge 1+0.25*(2-1)=1.25, top edge 3+0.25*(5-3)=3.5, halfway between = 2.375
    z = np.array([[1, 2], [3, 5]], dtype=np.float32)      # row 0 = y1: Q11, Q21; row 1 = y2: Q12, Q22
    gi = oracle.geom(2, 2, 0, 0, 1, 1)
    assert oracle.bilinear(z, gi, oracle.geom(1, 1, 0.25, 0.5, 1, 1))[0, 0] == 2.375
    # transposed operand would give (t,s)=(1/2,1/4): 1.5 + 0.25*(4-1.5) = 2.125
    assert oracle.bilinear(z, gi, oracle.geom(1, 1, 0.5, 0.25, 1, 1))[0, 0] == 2.125


def test_knots_bit_exact_and_last_node():
    rng = np.random.default_rng(7)
    z = rng.normal(-5000, 30, (6, 5)).astype(np.float32)
    gi = oracle.geom(5, 6, 0, 0, 1, 1)
    go = oracle.geom(17, 21, 0, 0, 0.25, 0.25)           # (n-1)*4+1 nodes: last node on the last sample
    out = oracle.bilinear(z, gi, go)
    assert np.array_equal(out[::4, ::4], z.astype(np.float64))
    assert out[-1, -1] == z[-1, -1]


def test_convex_combination_bounds():
    rng = np.random.default_rng(8)
    z = rng.uniform(-1, 1, (8, 8)).astype(np.float32)
    gi = oracle.geom(8, 8, 0, 0, 1, 1)
    out = oracle.bilinear(z, gi, oracle.geom(50, 50, 0, 0, 6.9 / 49, 6.8 / 49))
    assert not np.isnan(out).any()
    # weights >= 0 and sum to 1: each value lies inside its cell's corner range
    assert np.all(out <= z.max() + 1e-12) and np.all(out >= z.min() - 1e-12)
    one = oracle.bilinear(np.ones((8, 8), np.float32), gi, oracle.geom(50, 50, 0, 0, 0.14, 0.13))
    np.testing.assert_allclose(one, 1.0, rtol=0, atol=1e-15)


def test_out_of_extent_is_nan_and_nan_poisons_cell():
    z = np.arange(16, dtype=np.float32).reshape(4, 4)
    gi = oracle.geom(4, 4, 0, 0, 1, 1)
    out = oracle.bilinear(z, gi, oracle.geom(6, 6, -0.5, -0.5, 0.8, 0.8))
    xs = -0.5 + np.arange(6) * np.float64(np.float32(0.8))
    inside = (xs >= 0) & (xs <= 3)
    assert np.array_equal(np.isnan(out), ~(inside[None, :] & inside[:, None]))
    # B4: a NaN corner poisons the whole cell, even at a knot where its weight is exactly 0
    z2 = z.copy()
    z2[1, 1] = np.nan
    out2 = oracle.bilinear(z2, gi, oracle.geom(7, 7, 0, 0, 0.5, 0.5))
    assert np.isnan(out2[0, 0])          # node on knot (0,0): cell (0,0) has the NaN corner (1,1)
    assert np.isnan(out2[1, 1]) and np.isnan(out2[3, 3])
    assert not np.isnan(out2[6, 6]) and not np.isnan(out2[0, 5])


def test_argument_errors():
    with pytest.raises(ValueError):
        oracle.bilinear(np.zeros((1, 4), np.float32), oracle.geom(4, 1, 0, 0, 1, 1), oracle.geom(2, 2, 0, 0, 1, 1))
    with pytest.raises(ValueError):
        oracle.bilinear(np.zeros((4, 4), np.float32), oracle.geom(4, 4, 0, 0, 0, 1), oracle.geom(2, 2, 0, 0, 1, 1))
