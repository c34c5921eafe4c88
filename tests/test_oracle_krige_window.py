"""Pins of oracle_krige_window (readings W1-W4)
against what the mathematics fixes: constants, symmetry (planes reproduced at the centre of a full window; equal
weights on the 4 axis neighbours), an independent LAPACK solve of the gamma-form system on the same points, the
bilinear fallback by hand, the (key, window order) tie rule, window clipping at the grid border."""
import numpy as np
import pytest

import oracle


def _lapack_ok(px, py, z, xq, yq, gam):
    k = len(px)
    A = np.zeros((k + 1, k + 1))
    H = np.hypot(np.subtract.outer(px, px), np.subtract.outer(py, py))
    A[:k, :k] = np.where(H == 0, 0.0, gam(H))
    A[:k, k] = A[k, :k] = 1.0
    b = np.append(gam(np.hypot(px - xq, py - yq)), 1.0)
    lam = np.linalg.solve(A, b)[:k]
    return float(lam @ z)


def test_constant_field_and_valid_cells_copied():
    rng = np.random.default_rng(1)
    z = np.full((12, 15), -4321.5, np.float32)
    holes = rng.random(z.shape) < 0.1
    z[holes] = np.nan
    r = oracle.krige_window(z, oracle.geom(15, 12, 3.0, -2.0, 2.0, 2.0), oracle.vgm(0, 9.0, 2.0, 0.0))
    assert r["failed"] == 0
    k = r["how"] != 255
    assert np.abs(r["out"][k] + 4321.5).max() < 1e-9          # weights sum to 1
    assert (r["how"][~holes] == 0).all() and (r["out"][~holes] == z[~holes]).all()


def test_single_hole_full_window_vs_lapack_and_plane():
    rng = np.random.default_rng(2)
    yy, xx = np.meshgrid(np.arange(9.0), np.arange(11.0), indexing="ij")
    z = (-100 + rng.normal(0, 3, (9, 11))).astype(np.float32)
    z[4, 5] = np.nan
    g = oracle.geom(11, 9, 10.0, 20.0, 1.5, 2.5)
    for model, gam in ((0, lambda h: 0.2 + 1.8 * (1 - np.exp(-h / 7.0))), (2, lambda h: 0.2 + 1.8 * (1 - np.exp(-(h / 7.0) ** 2)))):
        r = oracle.krige_window(z, g, oracle.vgm(model, 7.0, 2.0, 0.2))
        assert r["how"][4, 5] == 24
        ii, jj = np.meshgrid(np.arange(2, 7), np.arange(3, 8), indexing="ij")
        sel = ~((ii == 4) & (jj == 5))
        px, py = 10.0 + 1.5 * jj[sel], 20.0 + 2.5 * ii[sel]
        want = _lapack_ok(px, py, z[ii[sel], jj[sel]].astype(np.float64), 10.0 + 1.5 * 5, 20.0 + 2.5 * 4, gam)
        assert abs(r["out"][4, 5] - want) < 1e-9
    # a plane is reproduced at the centre of a full (symmetric) window: the weights are symmetric
    zp = (5.0 + 0.25 * xx - 0.75 * yy).astype(np.float32)
    truth = zp[4, 5]
    zp[4, 5] = np.nan
    r = oracle.krige_window(zp, g, oracle.vgm(0, 7.0, 2.0, 0.0))
    assert abs(r["out"][4, 5] - truth) < 1e-9


def test_nearest_n_and_the_tie_rule():
    rng = np.random.default_rng(3)
    z = rng.normal(50, 5, (7, 7)).astype(np.float32)
    z[3, 3] = np.nan
    g = oracle.geom(7, 7, 0.0, 0.0, 1.0, 1.0)
    v = oracle.vgm(0, 4.0, 1.0, 0.0)
    # n_max = 4: the four axis neighbours (key 1), equal weights by symmetry
    r = oracle.krige_window(z, g, v, n_max=4)
    assert r["how"][3, 3] == 4 and abs(r["out"][3, 3] - np.mean([z[2, 3], z[4, 3], z[3, 2], z[3, 4]], dtype=np.float64)) < 1e-9
    # one axis neighbour missing: three at key 1, then the FIRST diagonal in window order (-1,-1) among the four ties at key 2
    z2 = z.copy(); z2[3, 4] = np.nan
    r = oracle.krige_window(z2, g, v, n_max=4)
    pts = [(2, 2), (2, 3), (3, 2), (4, 3)]
    lam, _ = oracle.ok_weights([p[1] for p in pts], [p[0] for p in pts], 3.0, 3.0, v)
    assert r["how"][3, 3] == 4 and abs(r["out"][3, 3] - sum(l * float(z2[p]) for l, p in zip(lam, pts))) < 1e-12
    # non-square spacing: with dy = 3 dx the "nearest 2" are the left and right neighbours only
    r = oracle.krige_window(z, oracle.geom(7, 7, 0.0, 0.0, 1.0, 3.0), v, n_max=2, n_min=1)
    assert r["how"][3, 3] == 2 and abs(r["out"][3, 3] - 0.5 * (float(z[3, 2]) + float(z[3, 4]))) < 1e-9


def test_bilinear_fallback_by_hand_and_nan_rules():
    z = np.arange(49, dtype=np.float32).reshape(7, 7) ** 1.5
    g = oracle.geom(7, 7, 0.0, 0.0, 1.0, 1.0)
    v = oracle.vgm(0, 4.0, 1.0, 0.0)
    zz = z.copy(); zz[3, 3] = np.nan
    r = oracle.krige_window(zz, g, v, n_min=25)                # never enough: always the fallback
    want = 0.25 * (float(z[2, 2]) + float(z[2, 4]) + float(z[4, 2]) + float(z[4, 4]))
    assert r["how"][3, 3] == 255 and abs(r["out"][3, 3] - want) < 1e-12
    zz[2, 2] = np.nan                                          # a NaN corner: no fallback for bilinear (L182)
    r = oracle.krige_window(zz, g, v, n_min=25)
    assert np.isnan(r["out"][3, 3]) and np.isnan(r["out"][2, 2]) and r["how"][2, 2] == 255
    zz = z.copy(); zz[0, 3] = np.nan                           # on the border the rectangle leaves the grid
    r = oracle.krige_window(zz, g, v, n_min=25)
    assert np.isnan(r["out"][0, 3])
    # a hole whose whole window is empty falls back (and is NaN); its neighbours with >= n_min valid cells are kriged
    zz = z.copy(); zz[1:6, 1:6] = np.nan
    r = oracle.krige_window(zz, g, v, half=2, n_min=3)
    assert r["how"][3, 3] == 255 and np.isnan(r["out"][3, 3]) and 3 <= r["how"][1, 1] <= 24 and np.isfinite(r["out"][1, 1])


def test_window_is_clipped_at_the_border():
    rng = np.random.default_rng(5)
    z = rng.normal(0, 1, (6, 6)).astype(np.float32)
    z[0, 0] = np.nan
    g = oracle.geom(6, 6, 0.0, 0.0, 2.0, 2.0)
    v = oracle.vgm(1, 9.0, 3.0, 0.3)
    r = oracle.krige_window(z, g, v)
    pts = [(i, j) for i in range(3) for j in range(3) if (i, j) != (0, 0)]
    lam, _ = oracle.ok_weights([2.0 * p[1] for p in pts], [2.0 * p[0] for p in pts], 0.0, 0.0, v)
    assert r["how"][0, 0] == 8 and abs(r["out"][0, 0] - sum(l * float(z[p]) for l, p in zip(lam, pts))) < 1e-12


@pytest.mark.parametrize("half", [1, 2, 3])
def test_window_sizes(half):
    z = np.full((9, 9), 7.25, np.float32); z[4, 4] = np.nan
    r = oracle.krige_window(z, oracle.geom(9, 9, 0, 0, 1, 1), oracle.vgm(0, 5.0, 1.0, 0.0), half=half)
    assert r["how"][4, 4] == (2 * half + 1) ** 2 - 1 and abs(r["out"][4, 4] - 7.25) < 1e-10
