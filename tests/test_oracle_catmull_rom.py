"""Pins of the oracle's Catmull-Rom cubic (eq. L140) against
what the printed polynomial fixes: C(0) = P1, C(1) = P2, C(1/2) = (-P0 + 9 P1 + 9 P2 - P3)/16, exact
reproduction of quadratics (cubic convolution with a = -1/2), separability, and the fallback to bilinear
 where one of the 16 neighbours is missing."""
import numpy as np

import oracle


def G(nx, ny, x0=0.0, y0=0.0, dx=1.0, dy=1.0):
    return oracle.geom(nx, ny, x0, y0, dx, dy)


def test_knots_and_midpoint_of_the_printed_polynomial():
    # rows all equal -> the y pass reproduces the row value (weights sum to 1): a 1-D check of eq. L140
    P = np.array([3.0, -1.0, 4.0, 10.0, 2.0, 7.0], dtype=np.float32)
    z = np.tile(P, (6, 1))
    out = oracle.catmull_rom(z, G(6, 6), G(3, 1, 2.0, 2.0, 0.5, 1.0))[0]      # x = 2, 2.5, 3 on row y = 2
    assert out[0] == 4.0 and out[2] == 10.0                                   # C(0) = P1, C(1) = P2
    assert abs(out[1] - (-(-1.0) + 9 * 4.0 + 9 * 10.0 - 2.0) / 16.0) < 1e-14  # C(1/2)
    # t = 1/4 by hand from the printed coefficients: P = (-1, 4, 10, 2)
    t = 0.25
    want = 0.5 * (2 * 4 + (1 + 10) * t + (2 * -1 - 5 * 4 + 4 * 10 - 2) * t * t + (1 + 3 * 4 - 3 * 10 + 2) * t ** 3)
    got = oracle.catmull_rom(z, G(6, 6), G(1, 1, 2.25, 2.0, 1.0, 1.0))[0, 0]
    assert abs(got - want) < 1e-14 and abs(want - 5.7578125) < 1e-12   # (8 + 2.75 + 1 - 0.234375) / 2


def test_quadratics_are_reproduced_in_the_interior_and_planes_everywhere():
    yy, xx = np.meshgrid(np.arange(12.0), np.arange(15.0), indexing="ij")
    f = lambda x, y: 2.0 + 0.5 * x - 0.25 * y + 0.125 * x * x - 0.5 * x * y + 0.375 * y * y
    z = f(xx, yy).astype(np.float32)                                          # exactly representable
    go = G(40, 30, 1.0, 1.0, 0.3, 0.3)                                        # inside [1, nx-2] x [1, ny-2]
    out = oracle.catmull_rom(z, G(15, 12), go)
    Y, X = np.meshgrid(1.0 + 0.3 * np.arange(30), 1.0 + 0.3 * np.arange(40), indexing="ij")
    X, Y = X.astype(np.float32).astype(np.float64), Y.astype(np.float32).astype(np.float64)
    # node coordinates are formed from the fp32 geometry fields: compare at those
    Xn = np.float64(np.float32(1.0)) + np.arange(40) * np.float64(np.float32(0.3))
    Yn = np.float64(np.float32(1.0)) + np.arange(30) * np.float64(np.float32(0.3))
    inside = (Xn[None, :] <= 12.0) & (Yn[:, None] <= 9.0)
    assert np.abs(out - f(Xn[None, :], Yn[:, None]))[inside].max() < 1e-10
    plane = (1.0 + 2.0 * xx - 3.0 * yy).astype(np.float32)                    # border cells fall back to bilinear: still exact
    out = oracle.catmull_rom(plane, G(15, 12), G(57, 45, 0.0, 0.0, 0.25, 0.25))
    Xp, Yp = 0.25 * np.arange(57), 0.25 * np.arange(45)
    assert np.abs(out - (1.0 + 2.0 * Xp[None, :] - 3.0 * Yp[:, None])).max() < 1e-12


def test_fallback_is_bilinear_at_borders_and_next_to_nan():
    rng = np.random.default_rng(5)
    z = rng.normal(-5000, 30, (9, 11)).astype(np.float32)
    z[4, 5] = np.nan
    gi, go = G(11, 9), G(41, 33, 0.0, 0.0, 0.25, 0.25)
    cr, bl = oracle.catmull_rom(z, gi, go), oracle.bilinear(z, gi, go)
    Y, X = np.meshgrid(0.25 * np.arange(33), 0.25 * np.arange(41), indexing="ij")
    i, j = np.minimum(np.floor(X), 9).astype(int), np.minimum(np.floor(Y), 7).astype(int)
    border = (i < 1) | (i > 11 - 3) | (j < 1) | (j > 9 - 3)
    near_nan = (np.abs(i + 0.5 - 5) <= 2) & (np.abs(j + 0.5 - 4) <= 2)        # the NaN is one of the 16
    fb = border | near_nan
    assert np.array_equal(cr[fb], bl[fb], equal_nan=True)
    assert np.isfinite(cr[~fb]).all() and np.abs(cr[~fb] - bl[~fb]).max() > 1e-3   # elsewhere it is the cubic
    assert np.isnan(cr[(i == 5) & (j == 4)]).all()                            # bilinear has no fallback (L182)
    out = oracle.catmull_rom(z, gi, G(3, 1, -0.5, 2.0, 6.0, 1.0))             # x = -0.5, 5.5, 11.5
    assert np.isnan(out[0, 0]) and np.isnan(out[0, 2])                        # out of extent (B4)


def test_separable_product():
    f = np.array([0.0, 1.0, 4.0, 9.0, 16.0, 2.0]); g = np.array([1.0, -2.0, 3.0, 0.5, 7.0, 1.0])
    z = np.outer(g, f).astype(np.float32)
    a = oracle.catmull_rom(z, G(6, 6), G(1, 1, 2.25, 2.75, 1, 1))[0, 0]
    fx = oracle.catmull_rom(np.tile(f.astype(np.float32), (6, 1)), G(6, 6), G(1, 1, 2.25, 2.0, 1, 1))[0, 0]
    gy = oracle.catmull_rom(np.tile(g.astype(np.float32)[:, None], (1, 6)), G(6, 6), G(1, 1, 2.0, 2.75, 1, 1))[0, 0]
    assert abs(a - fx * gy) < 1e-12
