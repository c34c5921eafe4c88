"""Pins for the oracle's ordinary kriging (readings K1-K5, D2, D3 in DESIGN.md).

Independent checks only: the two-point closed form, the covariance-form system solved by LAPACK
(a different formulation AND a different solver than the oracle's gamma-form LU), symmetry
arguments, invariances, exactness, the paper's two principles, exact rational
arithmetic for the fp32 key, and brute force for the neighbour search."""
from fractions import Fraction

import numpy as np
import pytest

import oracle

EXP, SPH = oracle.EXPONENTIAL, oracle.SPHERICAL


# ------------------------------------------------------------------ variogram (K3)
def test_variogram_values():
    v = oracle.vgm(EXP, 10.0, 2.0, 0.0)
    # gamma(h) = C0 (1 - exp(-h/a)), no factor 3: gamma(a) = C0 (1 - 1/e)
    assert oracle.variogram(v, 10.0)[0] == pytest.approx(2.0 * (1 - np.exp(-1.0)), rel=1e-15)
    assert oracle.variogram(v, 0.0)[0] == 0.0
    assert oracle.variogram(v, 1e9)[0] == pytest.approx(2.0, rel=1e-15)
    vn = oracle.vgm(EXP, 10.0, 2.0, 0.5)
    assert oracle.variogram(vn, 0.0)[0] == 0.0                       # gamma(0) = 0 even with a nugget
    assert oracle.variogram(vn, 1e-9)[0] == pytest.approx(0.5, abs=1e-9)
    assert oracle.variogram(vn, 1e9)[0] == pytest.approx(2.0, rel=1e-15)
    s = oracle.vgm(SPH, 10.0, 2.0, 0.5)
    assert oracle.variogram(s, 5.0)[0] == pytest.approx(0.5 + 1.5 * (0.75 - 0.0625), rel=1e-15)   # 11/16 of c_p
    assert oracle.variogram(s, 10.0)[0] == 2.0 and oracle.variogram(s, 25.0)[0] == 2.0
    assert oracle.variogram(s, 0.0)[0] == 0.0
    h = np.linspace(0.01, 9.99, 50)
    assert np.all(np.diff(oracle.variogram(s, h)) > 0) and np.all(np.diff(oracle.variogram(vn, h)) > 0)


# ------------------------------------------------------------------ solve (K4)
def test_lu_against_lapack():
    rng = np.random.default_rng(3)
    for n in (2, 3, 4, 5, 6, 33):
        A = rng.normal(0, 1, (n, n))
        A[0, 0] = 0.0                                                 # forces a row exchange
        b = rng.normal(0, 1, n)
        np.testing.assert_allclose(oracle.lu_solve(A, b), np.linalg.solve(A, b), rtol=1e-9, atol=1e-11)


def _cov(v, h):
    return v.sill - oracle.variogram(v, h)


def _c_form_weights(px, py, xq, yq, v):
    """Covariance form [C 1; 1^T 0][lam; mu] = [c0; 1] solved by numpy/LAPACK."""
    px, py = np.asarray(px, float), np.asarray(py, float)
    k = len(px)
    H = np.hypot(px[:, None] - px[None, :], py[:, None] - py[None, :])
    A = np.zeros((k + 1, k + 1))
    A[:k, :k] = _cov(v, H.ravel()).reshape(k, k)
    A[:k, k] = A[k, :k] = 1.0
    rhs = np.append(_cov(v, np.hypot(xq - px, yq - py)), 1.0)
    sol = np.linalg.solve(A, rhs)
    return sol[:k], sol[k]


def test_single_point():
    lam, mu = oracle.ok_weights([3.0], [4.0], 0.0, 0.0, oracle.vgm(EXP, 10, 1, 0))
    assert lam[0] == pytest.approx(1.0, abs=1e-15)


@pytest.mark.parametrize("model", [EXP, SPH])
@pytest.mark.parametrize("nugget", [0.0, 0.1])
def test_two_point_closed_form(model, nugget):
    # two points: lambda1 = 1/2 + (c1 - c2) / (2 (sill - c12)), from eliminating mu by hand
    v = oracle.vgm(model, 10.0, 1.0, nugget)
    px, py, xq, yq = [0.0, 4.0], [0.0, 0.0], 1.0, 0.0
    c1, c2, c12 = _cov(v, 1.0)[0], _cov(v, 3.0)[0], _cov(v, 4.0)[0]
    l1 = 0.5 + (c1 - c2) / (2 * (v.sill - c12))
    lam, mu = oracle.ok_weights(px, py, xq, yq, v)
    np.testing.assert_allclose(lam, [l1, 1 - l1], rtol=0, atol=1e-14)
    assert lam[0] > lam[1]                                            # principle 1
    if model == EXP and nugget == 0.0:
        # the same number written out: c = exp(-h/10)
        e1, e3, e4 = np.exp(-0.1), np.exp(-0.3), np.exp(-0.4)
        assert lam[0] == pytest.approx(0.5 + (e1 - e3) / (2 * (1 - e4)), abs=1e-14)
        assert lam[0] == pytest.approx(0.748755187238, abs=1e-12)
        assert 10 * lam[0] + 20 * lam[1] == pytest.approx(12.512448127617, abs=1e-11)
        # mu (gamma form) and kriging variance sigma^2 = sum lam_i gamma0_i + mu
        g0 = oracle.variogram(v, [1.0, 3.0])
        assert mu == pytest.approx(0.012332203659, abs=1e-11)
        assert lam @ g0 + mu == pytest.approx(0.148703758152, abs=1e-11)
    if model == SPH and nugget == 0.0:
        assert lam[0] == pytest.approx(0.752640845070, abs=1e-11)


@pytest.mark.parametrize("model,nugget", [(EXP, 0.0), (EXP, 0.01), (SPH, 0.0), (SPH, 0.3)])
def test_three_to_five_points_vs_c_form_lapack(model, nugget):
    v = oracle.vgm(model, 10.0, 1.0, nugget)
    px, py, z = [0.0, 3.0, 0.0], [0.0, 0.0, 4.0], np.array([1.0, 2.0, 4.0])
    lam, mu = oracle.ok_weights(px, py, 1.0, 1.0, v)
    lam_c, mu_c = _c_form_weights(px, py, 1.0, 1.0, v)
    np.testing.assert_allclose(lam, lam_c, rtol=0, atol=1e-13)
    assert mu == pytest.approx(-mu_c, abs=1e-13)                      # mu_C = -mu_gamma
    assert lam.sum() == pytest.approx(1.0, abs=1e-14)
    if (model, nugget) == (EXP, 0.0):
        np.testing.assert_allclose(lam, [0.506001752437, 0.291556438752, 0.202441808812], atol=1e-11)
        assert lam @ z == pytest.approx(1.898881865186, abs=1e-11)
    if (model, nugget) == (EXP, 0.01):
        assert lam @ z == pytest.approx(1.912659600833, abs=1e-11)
    if (model, nugget) == (SPH, 0.0):
        assert lam @ z == pytest.approx(1.892903424547, abs=1e-11)
    rng = np.random.default_rng(5)
    for k in (4, 5, 9, 32):
        qx, qy = rng.uniform(0, 20, k), rng.uniform(0, 20, k)
        lam, mu = oracle.ok_weights(qx, qy, 7.0, 9.0, v)
        lam_c, mu_c = _c_form_weights(qx, qy, 7.0, 9.0, v)
        np.testing.assert_allclose(lam, lam_c, rtol=0, atol=1e-10)
        assert lam.sum() == pytest.approx(1.0, abs=1e-12)


@pytest.mark.parametrize("model", [EXP, SPH])
def test_equilateral_centroid_thirds(model):
    ang = np.deg2rad([90, 210, 330])
    lam, _ = oracle.ok_weights(5 + 3 * np.cos(ang), -2 + 3 * np.sin(ang), 5.0, -2.0, oracle.vgm(model, 10, 2, 0.2))
    np.testing.assert_allclose(lam, 1 / 3, atol=1e-13)


def test_beyond_spherical_range_is_local_mean():
    # all points farther than the range from each other and from the query: Gamma = sill(1 - I) -> lam = 1/k
    px, py = [0.0, 30.0, 0.0], [0.0, 0.0, 30.0]
    lam, _ = oracle.ok_weights(px, py, 15.0, 15.0, oracle.vgm(SPH, 10, 1, 0))
    np.testing.assert_allclose(lam, 1 / 3, atol=1e-14)
    assert lam @ np.array([1.0, 2.0, 4.0]) == pytest.approx(7 / 3, abs=1e-13)


def test_invariances_scale_and_rigid_motion():
    rng = np.random.default_rng(6)
    px, py = rng.uniform(0, 10, 8), rng.uniform(0, 10, 8)
    v = oracle.vgm(SPH, 12.0, 1.0, 0.01)
    lam, _ = oracle.ok_weights(px, py, 4.0, 5.0, v)
    lam2, _ = oracle.ok_weights(px, py, 4.0, 5.0, oracle.vgm(SPH, 12.0, 37.0, 0.37))   # (sill,nugget)*alpha
    np.testing.assert_allclose(lam2, lam, atol=1e-12)
    th = 0.7
    R = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    P = R @ np.vstack([px, py]) + np.array([[100.0], [-50.0]])
    q = R @ np.array([4.0, 5.0]) + np.array([100.0, -50.0])
    lam3, _ = oracle.ok_weights(P[0], P[1], q[0], q[1], v)
    np.testing.assert_allclose(lam3, lam, atol=1e-10)


def test_declustering_principle():
    # a lone point at x=-1 vs a cluster at x=+1, +1.05, query at 0 (exp, a=10, nugget 0):
    # the pair shares about ONE point's weight, it does not get two
    lam, _ = oracle.ok_weights([-1.0, 1.0, 1.05], [0.0, 0.0, 0.0], 0.0, 0.0, oracle.vgm(EXP, 10, 1, 0))
    assert lam[0] == pytest.approx(0.5, abs=2e-3)
    assert lam[1] + lam[2] == pytest.approx(0.5, abs=2e-3)
    assert lam[0] == pytest.approx(0.499994, abs=2e-6) and lam[1] == pytest.approx(0.497741, abs=2e-6)


# ------------------------------------------------------------------ key and neighbours (K1, K2)
def _round_f32(fr: Fraction) -> np.float32:
    """Correctly rounded (nearest-even) fp32 of an exact rational."""
    c = np.float32(float(fr))
    cands = {c, np.nextafter(c, np.float32(np.inf)), np.nextafter(c, np.float32(-np.inf))}
    best = None
    for x in cands:
        err = abs(Fraction(float(x)) - fr)
        even = (int(np.float32(x).view(np.uint32)) & 1) == 0
        if best is None or err < best[0] or (err == best[0] and even):
            best = (err, x)
    return np.float32(best[1])


def _key_exact(xq, yq, xi, yi) -> np.float32:
    ddx = _round_f32(Fraction(float(xq)) - Fraction(float(xi)))
    ddy = _round_f32(Fraction(float(yq)) - Fraction(float(yi)))
    p = _round_f32(Fraction(float(ddy)) ** 2)
    return _round_f32(Fraction(float(ddx)) ** 2 + Fraction(float(p)))


def test_key_is_the_defined_fp32_expression():
    rng = np.random.default_rng(9)
    n_unfused_differs = 0
    for _ in range(400):
        xq, yq, xi, yi = rng.uniform(0, 2000, 4).astype(np.float32)
        k = np.float32(oracle.knn_key(xq, yq, xi, yi))
        assert k == _key_exact(xq, yq, xi, yi)
        ddx, ddy = np.float32(xq - xi), np.float32(yq - yi)
        n_unfused_differs += k != np.float32(np.float32(ddx * ddx) + np.float32(ddy * ddy))
    assert n_unfused_differs > 0          # the test can tell fmaf from mul+add
    assert oracle.knn_key(3.0, 4.0, 0.0, 0.0) == 25.0


def test_node_coords_fmaf():
    g = oracle.geom(7, 5, 0.48828125, 0.1, 0.9765625, 0.3)
    xq, yq = oracle.node_coords(g)
    for I in range(5):
        for J in range(7):
            assert xq[I, J] == _round_f32(Fraction(J) * Fraction(float(np.float32(g.dx))) + Fraction(float(np.float32(g.x0))))
            assert yq[I, J] == _round_f32(Fraction(I) * Fraction(float(np.float32(g.dy))) + Fraction(float(np.float32(g.y0))))


def test_knn_ties_lowest_index():
    # 4 lattice points equidistant from the cell centre, k=2 -> the two lowest indices, in order
    x, y = np.array([1, 0, 1, 0], np.float32), np.array([1, 1, 0, 0], np.float32)
    idx, key = oracle.knn(x, y, 0.5, 0.5, 2)
    assert idx.tolist() == [0, 1] and key.tolist() == [0.5, 0.5]
    idx, _ = oracle.knn(x, y, 0.5, 0.5, 2, oracle.Buckets(x, y, 0.3))
    assert idx.tolist() == [0, 1]


def test_knn_brute_matches_exact_sort():
    rng = np.random.default_rng(10)
    x, y = rng.uniform(0, 50, 150).astype(np.float32), rng.uniform(0, 50, 150).astype(np.float32)
    x[40:45], y[40:45] = x[10], y[10] + np.float32(1.0)               # distinct points, many equal keys nearby
    for xq, yq in rng.uniform(-5, 55, (12, 2)).astype(np.float32):
        keys = np.array([_key_exact(xq, yq, a, b) for a, b in zip(x, y)], dtype=np.float32)
        order = np.lexsort((np.arange(150), keys))[:9]
        idx, key = oracle.knn(x, y, xq, yq, 9)
        assert idx.tolist() == order.tolist()
        assert key.tolist() == keys[order].tolist()


@pytest.mark.parametrize("cell", [0.7, 3.0, 40.0])
def test_knn_buckets_match_brute(cell):
    rng = np.random.default_rng(14)
    n = 4000
    x = np.concatenate([rng.uniform(0, 100, n // 2), rng.normal(50, 3, n // 2)]).astype(np.float32)   # uneven density
    y = np.concatenate([rng.uniform(0, 60, n // 2), rng.normal(20, 3, n // 2)]).astype(np.float32)
    # an exact lattice patch creates exact key ties
    x[:100], y[:100] = np.repeat(np.arange(10), 10) + 70, np.tile(np.arange(10), 10) + 40
    b = oracle.Buckets(x, y, cell)
    qs = np.vstack([rng.uniform(-20, 120, (150, 2)), [[74.5, 44.5], [75.0, 45.0], [0, 0], [100, 60]]]).astype(np.float32)
    for xq, yq in qs:
        for k in (1, 8, 33):
            i0, k0 = oracle.knn(x, y, xq, yq, k)
            i1, k1 = oracle.knn(x, y, xq, yq, k, b)
            assert i0.tolist() == i1.tolist() and k0.tolist() == k1.tolist()


# ------------------------------------------------------------------ full path (K1-K5)
def test_krige_constant_exact_at_data_sum_to_one():
    rng = np.random.default_rng(15)
    n = 300
    x, y = rng.uniform(0, 30, n).astype(np.float32), rng.uniform(0, 30, n).astype(np.float32)
    z = rng.normal(-5000, 10, n).astype(np.float32)
    xq, yq = rng.uniform(0, 30, 40).astype(np.float32), rng.uniform(0, 30, 40).astype(np.float32)
    for v in (oracle.vgm(SPH, 10, 100, 0), oracle.vgm(EXP, 10, 100, 1.0)):
        r = oracle.krige_points(x, y, np.full(n, -4321.5, np.float32), xq, yq, v, 8, want_lambda=True)
        np.testing.assert_allclose(r["zhat"], -4321.5, rtol=0, atol=1e-8)          # reproduces constants
        np.testing.assert_allclose(r["lam"].sum(axis=1), 1.0, atol=1e-11)
        assert r["failed"] == 0
        # exact interpolator at the data (nugget 0, and nugget > 0 under gamma(0) = 0)
        r = oracle.krige_points(x, y, z, x[:50], y[:50], v, 8, want_lambda=True)
        np.testing.assert_allclose(r["zhat"], z[:50].astype(np.float64), rtol=0, atol=1e-7)
        assert np.array_equal(r["nbr"][:, 0], np.arange(50))
        np.testing.assert_allclose(r["lam"][:, 0], 1.0, atol=1e-9)
        # the estimate is the weighted sum of the chosen neighbours (K5)
        r = oracle.krige_points(x, y, z, xq, yq, v, 8, want_lambda=True)
        np.testing.assert_allclose(r["zhat"], (r["lam"] * z[r["nbr"]]).sum(axis=1), rtol=0, atol=1e-8)
    # buckets and brute force give the same everything
    b = oracle.Buckets(x, y, 2.5)
    r0 = oracle.krige_points(x, y, z, xq, yq, v, 16)
    r1 = oracle.krige_points(x, y, z, xq, yq, v, 16, b)
    assert np.array_equal(r0["nbr"], r1["nbr"]) and np.array_equal(r0["zhat"], r1["zhat"])


def test_krige_duplicate_points_fail_as_nan():
    x = np.array([0, 0, 1, 2], np.float32)
    y = np.array([0, 0, 0, 1], np.float32)
    z = np.array([1, 2, 3, 4], np.float32)
    r = oracle.krige_points(x, y, z, [0.5], [0.5], oracle.vgm(EXP, 10, 1, 0.1), 4)
    assert r["failed"] == 1 and np.isnan(r["zhat"][0])


def test_krige_argument_errors():
    x = np.zeros(3, np.float32)
    for bad in (oracle.vgm(EXP, 0, 1, 0), oracle.vgm(EXP, 1, 0, 0), oracle.vgm(EXP, 1, 1, 2), oracle.vgm(7, 1, 1, 0)):
        with pytest.raises(ValueError):
            oracle.krige_points(x, x, x, [0.0], [0.0], bad, 2)
    with pytest.raises(ValueError):
        oracle.krige_points(x, x, x, [0.0], [0.0], oracle.vgm(EXP, 1, 1, 0), 4)     # k > n


# ---------------------------------------------------------------- NEXT-3: kriging variance; NEXT-4: Gaussian model

def test_variance_two_point_closed_form():
    """sigma^2 = sum lambda_i gamma_i0 + mu.  Two points: rows of the gamma form give gamma12 lambda2 + mu = gamma1,
    so mu = gamma1 - gamma12 lambda2 with lambda1 = 1/2 + (gamma2 - gamma1)/(2 gamma12) -- retyped here in numpy,
    and the value SURVEY.md 8(c) prints for (0,0),(4,0), query (1,0), exponential a=10, sill 1: 0.148703758152."""
    x, y, z = np.array([0, 4], np.float32), np.array([0, 0], np.float32), np.array([10, 20], np.float32)
    for model, gam in ((oracle.EXPONENTIAL, lambda h: 1 - np.exp(-h / 10.0)), (oracle.GAUSSIAN, lambda h: 1 - np.exp(-(h / 10.0) ** 2)),
                       (oracle.SPHERICAL, lambda h: 1.5 * h / 10 - 0.5 * (h / 10) ** 3)):
        g1, g2, g12 = gam(1.0), gam(3.0), gam(4.0)
        l1 = 0.5 + (g2 - g1) / (2 * g12)
        mu = g1 - g12 * (1 - l1)
        want = l1 * g1 + (1 - l1) * g2 + mu
        r = oracle.krige_points(x, y, z, [1.0], [0.0], oracle.vgm(model, 10.0, 1.0, 0.0), 2, want_var=True)
        assert abs(r["var"][0] - want) < 1e-13 and abs(r["zhat"][0] - (l1 * 10 + (1 - l1) * 20)) < 1e-12
        if model == oracle.EXPONENTIAL:
            assert abs(r["var"][0] - 0.148703758152) < 1e-11


def test_variance_zero_at_data_local_mean_and_scaling():
    rng = np.random.default_rng(5)
    x, y = rng.uniform(0, 50, 40).astype(np.float32), rng.uniform(0, 50, 40).astype(np.float32)
    z = rng.normal(-100, 3, 40).astype(np.float32)
    v = oracle.vgm(oracle.EXPONENTIAL, 15.0, 4.0, 0.4)
    r = oracle.krige_points(x, y, z, x[:5], y[:5], v, 8, want_var=True)
    assert np.abs(r["var"]).max() < 1e-12                         # gamma(0) = 0: no error at a datum
    r = oracle.krige_points(x, y, z, [3.3, 41.0], [7.7, 20.0], v, 8, want_var=True)
    assert (r["var"] > 0).all() and (r["var"] < 2 * 4.0).all()
    # sigma^2 scales with (sill, nugget) -> alpha (sill, nugget); the estimate does not
    r2 = oracle.krige_points(x, y, z, [3.3, 41.0], [7.7, 20.0], oracle.vgm(oracle.EXPONENTIAL, 15.0, 12.0, 1.2), 8, want_var=True)
    assert np.allclose(r2["var"], 3 * r["var"], rtol=1e-12) and np.allclose(r2["zhat"], r["zhat"], rtol=1e-13)
    # all k neighbours mutually and from the node beyond a spherical range: lambda = 1/k, mu = sill/k,
    # sigma^2 = sill (1 + 1/k)
    xs, ys = np.array([0, 100, 0, 100], np.float32), np.array([0, 0, 100, 100], np.float32)
    r = oracle.krige_points(xs, ys, np.array([1, 2, 3, 4], np.float32), [50.0], [50.0], oracle.vgm(oracle.SPHERICAL, 10.0, 2.0, 0.5), 4, want_var=True)
    assert abs(r["var"][0] - 2.0 * 1.25) < 1e-12 and abs(r["zhat"][0] - 2.5) < 1e-12


@pytest.mark.parametrize("model", [oracle.EXPONENTIAL, oracle.SPHERICAL, oracle.GAUSSIAN])
def test_variance_vs_c_form_lapack(model):
    """C-form with LAPACK: [C 1; 1^T 0][lambda; mu_C] = [c0; 1], sigma^2 = sill - lambda.c0 - mu_C."""
    rng = np.random.default_rng(17 + model)
    k = 6
    x, y = rng.uniform(0, 20, k).astype(np.float32), rng.uniform(0, 20, k).astype(np.float32)
    z = rng.normal(0, 1, k).astype(np.float32)
    sill, nug, a = 3.0, 0.3, 9.0
    v = oracle.vgm(model, a, sill, nug)
    xq, yq = np.float32(8.5), np.float32(11.25)
    r = oracle.krige_points(x, y, z, [xq], [yq], v, k, want_var=True)
    xd, yd = x.astype(np.float64), y.astype(np.float64)
    H = np.hypot(xd[:, None] - xd[None, :], yd[:, None] - yd[None, :])
    h0 = np.hypot(xd - float(xq), yd - float(yq))
    cov = lambda h: np.where(h == 0, sill, sill - oracle.variogram(v, h.ravel()).reshape(h.shape))
    A = np.zeros((k + 1, k + 1)); A[:k, :k] = cov(H); A[:k, k] = A[k, :k] = 1.0
    b = np.append(cov(h0), 1.0)
    sol = np.linalg.solve(A, b)
    want = sill - sol[:k] @ b[:k] - sol[k]
    assert abs(r["var"][0] - want) < 1e-10 and abs(r["zhat"][0] - sol[:k] @ z.astype(np.float64)) < 1e-10


def test_gaussian_variogram_values():
    v = oracle.vgm(oracle.GAUSSIAN, 8.0, 5.0, 1.0)
    g = oracle.variogram(v, [0.0, 8.0, 1e-300, 4.0, 1e6])
    assert g[0] == 0.0                                            # gamma(0) = 0 with a nugget
    assert abs(g[1] - (1.0 + 4.0 * (1 - np.exp(-1.0)))) < 1e-14   # gamma(a) = nugget + c_p (1 - 1/e)
    assert abs(g[2] - 1.0) < 1e-14 and abs(g[3] - (1.0 + 4.0 * (1 - np.exp(-0.25)))) < 1e-14
    assert abs(g[4] - 5.0) < 1e-14
