"""Pins for oracle.spline / oracle.spline1d (natural cubic spline, reading D1/S1-S3).
Closed forms worked by hand, SciPy's CubicSpline(bc_type='natural') as a library cross-check,
and invariants (knots, linear fields, zero end curvature, separability, pass order)."""
import numpy as np
import pytest

import oracle


def test_hat_0_1_0():
    # knots (0,1,0), h=1: the single interior equation 4 M1 = 6(0-2+0) gives M1 = -3.
    # On [0,1]: S = x + (x^3 - x)(-3)/6 = 1.5 x - 0.5 x^3, so S(0.5) = 0.75 - 0.0625 = 0.6875.
    v, M = oracle.spline1d([0, 1, 0], 1.0, [0.5, 1.5, 0.25])
    np.testing.assert_allclose(M, [0, -3, 0], atol=1e-15)
    assert v[0] == pytest.approx(0.6875, abs=1e-15)
    assert v[1] == pytest.approx(0.6875, abs=1e-15)                      # symmetric
    assert v[2] == pytest.approx(1.5 * 0.25 - 0.5 * 0.25 ** 3, abs=1e-15)


def test_squares_0_1_4_9():
    # second differences are 2,2: 4M1+M2=12, M1+4M2=12 -> M1=M2=2.4.
    # S(1.5) = (1+4)/2 + 2*((0.125-0.5)*2.4)/6 = 2.5 - 0.3 = 2.2 ; S(0.5) = 0.5 - 0.15 = 0.35 ;
    # S(2.5) = 6.5 - 0.15 = 6.35
    v, M = oracle.spline1d([0, 1, 4, 9], 1.0, [1.5, 0.5, 2.5])
    np.testing.assert_allclose(M, [0, 2.4, 2.4, 0], atol=1e-14)
    np.testing.assert_allclose(v, [2.2, 0.35, 6.35], atol=1e-14)


def test_impulse_sevenths():
    # knots (0,0,1,0,0): rhs (6,-12,6); by symmetry M1=M3=a, M2=b: 4a+b=6, 2a+4b=-12 -> a=18/7, b=-30/7
    v, M = oracle.spline1d([0, 0, 1, 0, 0], 1.0, [1.5, 0.5])
    np.testing.assert_allclose(M, [0, 18 / 7, -30 / 7, 18 / 7, 0], atol=1e-14)
    # S(1.5) = 0.5 + (-0.375)(18/7 - 30/7)/6 = 0.5 + 0.75/7 ; S(0.5) = (-0.375)(18/7)/6
    np.testing.assert_allclose(v, [0.5 + 0.75 / 7, -0.375 * 18 / 7 / 6], atol=1e-15)


def test_spacing_h_scales_M():
    # same values on knots h apart: M scales by 1/h^2, values at the same knot-relative abscissa agree
    z = [0.3, -1.0, 2.0, 0.5, 0.7, -0.2]
    v1, M1 = oracle.spline1d(z, 1.0, [0.3, 2.6, 4.9])
    v2, M2 = oracle.spline1d(z, 0.25, [0.3, 2.6, 4.9])
    np.testing.assert_allclose(M2, M1 * 16, rtol=1e-13)
    np.testing.assert_allclose(v2, v1, rtol=1e-13)


def test_against_scipy_natural():
    scipy_interp = pytest.importorskip("scipy.interpolate")
    rng = np.random.default_rng(11)
    for n, h in [(3, 1.0), (4, 0.5), (17, 2.0), (200, 1.0)]:
        z = rng.normal(0, 1, n)
        u = rng.uniform(0, n - 1, 300)
        v, M = oracle.spline1d(z, h, u)
        cs = scipy_interp.CubicSpline(np.arange(n) * h, z, bc_type="natural")
        np.testing.assert_allclose(v, cs(u * h), rtol=0, atol=2e-12)
        np.testing.assert_allclose(M, cs(np.arange(n) * h, 2), rtol=0, atol=1e-10)


def test_linear_and_two_knots():
    v, M = oracle.spline1d([1.0, 3.0], 2.0, [0.0, 0.25, 1.0])
    np.testing.assert_allclose(M, 0)
    np.testing.assert_allclose(v, [1.0, 1.5, 3.0], atol=1e-15)
    z = 2.0 - 0.5 * np.arange(9)
    v, M = oracle.spline1d(z, 1.0, [0.1, 3.7, 8.0])
    np.testing.assert_allclose(M, 0, atol=1e-14)
    np.testing.assert_allclose(v, 2.0 - 0.5 * np.array([0.1, 3.7, 8.0]), atol=1e-14)
    assert np.isnan(oracle.spline1d(z, 1.0, [-0.01])[0][0]) and np.isnan(oracle.spline1d(z, 1.0, [8.01])[0][0])


def test_2d_separable_product_0_47265625():
    # z_ij = f_i g_j  ->  S(x,y) = S_f(y) S_g(x); f=g=(0,1,0): S(1/2,1/2) = 0.6875^2 = 0.47265625
    f = np.array([0, 1, 0], dtype=np.float32)
    z = np.outer(f, f)
    gi = oracle.geom(3, 3, 0, 0, 1, 1)
    assert oracle.spline(z, gi, oracle.geom(1, 1, 0.5, 0.5, 1, 1))[0, 0] == pytest.approx(0.47265625, abs=1e-15)
    # non-symmetric factors catch a transposed pass: f along y = (0,1,4,9), g along x = (0,1,0)
    fy = np.array([0, 1, 4, 9], dtype=np.float32)
    gx = np.array([0, 1, 0], dtype=np.float32)
    z = np.outer(fy, gx)                                   # [ny=4, nx=3]
    out = oracle.spline(z, oracle.geom(3, 4, 0, 0, 1, 1), oracle.geom(1, 1, 0.5, 1.5, 1, 1))
    assert out[0, 0] == pytest.approx(0.6875 * 2.2, abs=1e-14)


def test_2d_additive_and_knots_and_plane():
    rng = np.random.default_rng(12)
    f = rng.normal(0, 1, 7)
    g = rng.normal(0, 1, 9)
    z = (f[:, None] + g[None, :]).astype(np.float32)
    gi = oracle.geom(9, 7, 0, 0, 1, 1)
    go = oracle.geom(33, 25, 0, 0, 0.25, 0.25)
    out = oracle.spline(z, gi, go)
    assert np.allclose(out[::4, ::4], z.astype(np.float64), rtol=0, atol=1e-12)      # passes through knots
    # additive data -> S_f(y) + S_g(x) up to the fp32 rounding of z (compare via the fp32 samples' own splines)
    zf = z[:, 0].astype(np.float64) - z[0, 0]
    zg = z[0, :].astype(np.float64)
    Sf = oracle.spline1d(zf, 1.0, np.arange(25) * 0.25)[0]
    Sg = oracle.spline1d(zg, 1.0, np.arange(33) * 0.25)[0]
    np.testing.assert_allclose(out, Sf[:, None] + Sg[None, :], rtol=0, atol=5e-6)
    # planes with dyadic coefficients are reproduced exactly
    X, Y = np.arange(9)[None, :], np.arange(7)[:, None]
    zp = (-5000 + 0.5 * X + 0.25 * Y).astype(np.float32)
    outp = oracle.spline(zp, gi, go)
    Xo, Yo = (np.arange(33) * 0.25)[None, :], (np.arange(25) * 0.25)[:, None]
    np.testing.assert_allclose(outp, -5000 + 0.5 * Xo + 0.25 * Yo, rtol=0, atol=1e-9)


def test_2d_pass_order_commutes_and_scipy():
    scipy_interp = pytest.importorskip("scipy.interpolate")
    rng = np.random.default_rng(13)
    z = rng.normal(-5000, 20, (11, 14)).astype(np.float32)
    gi = oracle.geom(14, 11, 0, 0, 1, 1)
    go = oracle.geom(40, 31, 0, 0, 13 / 39.5, 10 / 30.5)
    a = oracle.spline(z, gi, go)
    # columns-then-rows == transpose the problem, run rows-then-columns, transpose back
    b = oracle.spline(z.T.copy(), oracle.geom(11, 14, 0, 0, 1, 1), oracle.geom(31, 40, 0, 0, go.dy, go.dx)).T
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-9)
    # library cross-check: natural CubicSpline along x, then along y
    xo = np.arange(40) * np.float64(np.float32(go.dx))
    yo = np.arange(31) * np.float64(np.float32(go.dy))
    T = scipy_interp.CubicSpline(np.arange(14), z.astype(np.float64), axis=1, bc_type="natural")(xo)
    ref = scipy_interp.CubicSpline(np.arange(11), T, axis=0, bc_type="natural")(yo)
    np.testing.assert_allclose(a, ref, rtol=0, atol=1e-9)


def test_2d_out_of_extent_nan():
    z = np.arange(20, dtype=np.float32).reshape(4, 5)
    out = oracle.spline(z, oracle.geom(5, 4, 0, 0, 1, 1), oracle.geom(4, 4, -1, 1, 2, 1))
    # x nodes -1,1,3,5 (extent [0,4]); y nodes 1,2,3,4 (extent [0,3])
    assert np.isnan(out[:, 0]).all() and np.isnan(out[:, 3]).all() and np.isnan(out[3, :]).all()
    assert not np.isnan(out[:3, 1:3]).any()
    np.testing.assert_allclose(out[:3, 1:3], [[6, 8], [11, 13], [16, 18]], atol=1e-12)
    with pytest.raises(ValueError):
        oracle.spline(np.zeros((1, 5), np.float32), oracle.geom(5, 1, 0, 0, 1, 1), oracle.geom(2, 2, 0, 0, 1, 1))
