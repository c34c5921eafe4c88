"""Pins of the oracle's geometric anisotropy (reading Ani):
oracle_aniso_lag, oracle_ok_weights_aniso, oracle_krige_points_aniso -- against hand-computed lags, the two-point
closed form of ordinary kriging, symmetry, and the isotropic oracle on coordinates transformed beforehand (points
rotated and stretched in numpy, not lags: a different route to the same numbers)."""
import math

import numpy as np
import pytest

import oracle


def test_lag_by_hand():
    L = oracle.aniso_lag
    assert L(None, 3.0, 4.0) == 5.0
    a = oracle.aniso(0.0, 0.5)                                  # major axis = x; across it distances count double
    assert L(a, 3.0, 0.0) == pytest.approx(3.0, abs=1e-15) and L(a, 0.0, 2.0) == pytest.approx(4.0, abs=1e-15)
    assert L(a, 3.0, 2.0) == pytest.approx(5.0, abs=1e-14)       # sqrt(3^2 + (2/0.5)^2)
    a = oracle.aniso(90.0, 0.5)                                 # major axis = y
    assert L(a, 0.0, 3.0) == pytest.approx(3.0, abs=1e-14) and L(a, 2.0, 0.0) == pytest.approx(4.0, abs=1e-14)
    a = oracle.aniso(30.0, 0.25)                                # 5 along (cos 30, sin 30), 1 across (-sin 30, cos 30)
    c, s = math.sqrt(3.0) / 2.0, 0.5
    assert L(a, 5.0 * c, 5.0 * s) == pytest.approx(5.0, abs=1e-13)
    assert L(a, -1.0 * s, 1.0 * c) == pytest.approx(4.0, abs=1e-13)
    # the sense of the angle: +45 degrees is counter-clockwise from +x, so (1, 1) runs along and (1, -1) across
    a = oracle.aniso(45.0, 0.5)
    r2 = math.sqrt(2.0)
    assert L(a, 3.0 / r2, 3.0 / r2) == pytest.approx(3.0, abs=1e-13)
    assert L(a, 3.0 / r2, -3.0 / r2) == pytest.approx(6.0, abs=1e-13)
    assert L(a, -2.0, 7.0) == pytest.approx(L(a, 2.0, -7.0), abs=0.0)        # a lag and its negative
    assert L(oracle.aniso(225.0, 0.5), -2.0, 7.0) == pytest.approx(L(a, -2.0, 7.0), abs=1e-13)   # the axis has no sense


def test_ratio_one_is_isotropic_for_any_angle():
    rng = np.random.default_rng(3)
    px, py = rng.uniform(0, 30, 9), rng.uniform(0, 30, 9)
    for model in (0, 1, 2):
        v = oracle.vgm(model, 17.0, 2.5, 0.1)
        lam0, mu0 = oracle.ok_weights(px, py, 11.0, 13.0, v)
        for ang in (0.0, 33.0, 90.0, -120.0):
            lam, mu = oracle.ok_weights(px, py, 11.0, 13.0, v, oracle.aniso(ang, 1.0))
            assert np.allclose(lam, lam0, rtol=0, atol=1e-11) and abs(mu - mu0) <= 1e-11


def test_two_points_closed_form():
    """Two neighbours: lambda_1 = 1/2 + (gamma_02 - gamma_01) / (2 gamma_12) (eliminate mu from the 3 x 3 system)."""
    v = oracle.vgm(0, 10.0, 1.0, 0.0)                            # gamma(h) = 1 - exp(-h / 10)
    a = oracle.aniso(0.0, 0.5)
    # p1 = (4, 0): lag 4.  p2 = (0, 1): lag 1 / 0.5 = 2.  p1 - p2 = (4, -1): lag sqrt(16 + 4)
    g01, g02, g12 = 1 - math.exp(-0.4), 1 - math.exp(-0.2), 1 - math.exp(-math.sqrt(20.0) / 10.0)
    want = 0.5 + (g02 - g01) / (2.0 * g12)
    lam, mu = oracle.ok_weights([4.0, 0.0], [0.0, 1.0], 0.0, 0.0, v, a)
    assert lam[0] == pytest.approx(want, abs=1e-13) and lam[1] == pytest.approx(1.0 - want, abs=1e-13)
    assert want == pytest.approx(0.29421281, abs=1e-8)           # by hand: 1/2 - (0.32967995 - 0.18126925) / (2 x 0.36059494)
    # a neighbour at d along the major axis and one at ratio * d across it are equally far: weights 1/2, 1/2 --
    # in the isotropic metric the second is closer and takes more
    for ang, p1, p2 in ((0.0, (6.0, 0.0), (0.0, 3.0)), (90.0, (0.0, 6.0), (3.0, 0.0)), (90.0, (0.0, -6.0), (-3.0, 0.0))):
        lam, _ = oracle.ok_weights([p1[0], p2[0]], [p1[1], p2[1]], 0.0, 0.0, v, oracle.aniso(ang, 0.5))
        assert lam[0] == pytest.approx(0.5, abs=1e-13)
        lam_iso, _ = oracle.ok_weights([p1[0], p2[0]], [p1[1], p2[1]], 0.0, 0.0, v)
        assert lam_iso[0] < 0.45


def _transform(x, y, ang, ratio):
    t = math.radians(ang)
    x, y = np.asarray(x, dtype=np.float64), np.asarray(y, dtype=np.float64)
    return math.cos(t) * x + math.sin(t) * y, (-math.sin(t) * x + math.cos(t) * y) / ratio


@pytest.mark.parametrize("model", [0, 1, 2])
@pytest.mark.parametrize("ang,ratio", [(0.0, 0.5), (37.0, 0.3), (-64.0, 0.8), (90.0, 0.25), (135.0, 0.6)])
def test_weights_equal_isotropic_weights_on_transformed_points(model, ang, ratio):
    rng = np.random.default_rng(100 + model)
    px, py = rng.uniform(-20, 20, 12), rng.uniform(-20, 20, 12)
    xq, yq = 1.5, -2.5
    v = oracle.vgm(model, 14.0, 3.0, 0.15 if model == 2 else 0.0)
    lam, mu = oracle.ok_weights(px, py, xq, yq, v, oracle.aniso(ang, ratio))
    tx, ty = _transform(px, py, ang, ratio)
    tq = _transform([xq], [yq], ang, ratio)
    lam_t, mu_t = oracle.ok_weights(tx, ty, float(tq[0][0]), float(tq[1][0]), v)
    assert np.allclose(lam, lam_t, rtol=0, atol=1e-9) and abs(mu - mu_t) <= 1e-9
    assert abs(lam.sum() - 1.0) <= 1e-12
    lam_iso, _ = oracle.ok_weights(px, py, xq, yq, v)
    assert np.abs(lam - lam_iso).max() > 1e-3                    # (the anisotropy really changes the weights)


def test_krige_points_equal_isotropic_kriging_of_transformed_points():
    """All n points are neighbours (k = n), so the neighbour search -- which stays isotropic -- cannot differ.  Angle 90,
    ratio 1/2: (x, y) -> (y, -2 x), exact in fp32."""
    rng = np.random.default_rng(21)
    n = 14
    x = rng.integers(-40, 40, n).astype(np.float32) * 0.25
    y = rng.integers(-40, 40, n).astype(np.float32) * 0.25
    keep = np.unique(np.stack([x, y], 1), axis=0, return_index=True)[1]
    x, y = x[np.sort(keep)], y[np.sort(keep)]
    n = x.size
    z = rng.normal(-3000.0, 20.0, n).astype(np.float32)
    xq = np.array([0.125, 3.5, -7.25, 2.0], np.float32)
    yq = np.array([1.375, -2.5, 4.0, 2.0], np.float32)
    v = oracle.vgm(1, 9.0, 400.0, 4.0)
    r = oracle.krige_points(x, y, z, xq, yq, v, n, a=oracle.aniso(90.0, 0.5), want_lambda=True)
    t = oracle.krige_points(y, -2.0 * x, z, yq, -2.0 * xq, v, n, want_lambda=True)
    tv = oracle.krige_points(y, -2.0 * x, z, yq, -2.0 * xq, v, n, want_var=True)
    assert r["failed"] == 0 and t["failed"] == 0
    # the two neighbour orders may differ (keys differ): compare weights per original index
    for q in range(xq.size):
        wr = np.zeros(n); wr[r["nbr"][q]] = r["lam"][q]
        wt = np.zeros(n); wt[t["nbr"][q]] = t["lam"][q]
        assert np.allclose(wr, wt, rtol=0, atol=1e-9)
    assert np.allclose(r["zhat"], t["zhat"], rtol=0, atol=1e-8)
    assert np.allclose(r["var"], tv["var"], rtol=0, atol=1e-8)
    iso = oracle.krige_points(x, y, z, xq, yq, v, n)
    assert np.abs(iso["zhat"] - r["zhat"]).max() > 1e-3


def test_neighbours_stay_the_nearest_by_plain_distance():
    rng = np.random.default_rng(5)
    x, y = rng.uniform(0, 50, 300).astype(np.float32), rng.uniform(0, 50, 300).astype(np.float32)
    z = rng.normal(size=300).astype(np.float32)
    xq, yq = rng.uniform(5, 45, 20).astype(np.float32), rng.uniform(5, 45, 20).astype(np.float32)
    v = oracle.vgm(0, 12.0, 1.0, 0.0)
    r = oracle.krige_points(x, y, z, xq, yq, v, 8, a=oracle.aniso(20.0, 0.2))
    i = oracle.krige_points(x, y, z, xq, yq, v, 8)
    assert np.array_equal(r["nbr"], i["nbr"])


def test_bad_ratio_is_refused():
    v = oracle.vgm(0, 10.0, 1.0, 0.0)
    for ratio in (0.0, -0.5, 1.5, float("nan")):
        with pytest.raises(ValueError):
            oracle.ok_weights([1.0, 2.0], [0.0, 1.0], 0.0, 0.0, v, oracle.aniso(10.0, ratio))
