"""Seeded random geometries through the C ABI against the oracle: input sizes from 2 to a few tiles,
integer and non-integer spacing ratios (up- and down-sampling), shifted origins so that some output
nodes fall outside the input extent on any side, rectangular grids.  Bar: north_star's tolerances,
NaN patterns identical (tests/_util.max_abs_err)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_22675_b200 import workloads as W
from _util import ogeom, depth_range, max_abs_err

pytestmark = pytest.mark.gpu


def _field(rng, ny, nx):
    yy, xx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    z = -5000.0 + 0.4 * xx + 0.3 * yy + 30.0 * np.sin(xx / 7.0) * np.cos(yy / 5.0) + rng.normal(0, 0.5, (ny, nx))
    return z.astype(np.float32)


def _geoms(rng):
    nx, ny = int(rng.integers(2, 260)), int(rng.integers(2, 200))
    dxi, dyi = float(rng.choice([1.0, 0.5, 2.0, 1.25])), float(rng.choice([1.0, 0.5, 3.0]))
    gi = W.Geom(nx, ny, float(rng.uniform(-50, 50)), float(rng.uniform(-50, 50)), dxi, dyi)
    ratio_x = float(rng.choice([1.0, 0.5, 0.25, 1.0 / 3.0, 0.37, 0.8, 1.7, 4.0]))
    ratio_y = float(rng.choice([1.0, 0.5, 0.25, 0.2, 0.43, 1.3, 2.5]))
    dxo, dyo = dxi * ratio_x, dyi * ratio_y
    # output extent: the input extent shifted / stretched by up to 15 % on each side
    wx, wy = (nx - 1) * dxi, (ny - 1) * dyi
    x0 = gi.x0 + float(rng.uniform(-0.15, 0.10)) * wx
    y0 = gi.y0 + float(rng.uniform(-0.15, 0.10)) * wy
    nxo = int(min(max((wx * float(rng.uniform(0.6, 1.2))) / dxo, 1), 700)) + 1
    nyo = int(min(max((wy * float(rng.uniform(0.6, 1.2))) / dyo, 1), 500)) + 1
    return gi, W.Geom(nxo, nyo, x0, y0, dxo, dyo)


@pytest.mark.parametrize("seed", range(24))
def test_bilinear_and_spline_random_geometry(seed):
    import paper_2505_22675_b200 as b
    rng = np.random.default_rng(9100 + seed)
    gi, go = _geoms(rng)
    z = _field(rng, gi.ny, gi.nx)
    zt = torch.from_numpy(z).cuda()
    for name, fn, ofn in (("bilinear", b.interp_bilinear, oracle.bilinear), ("spline", b.interp_spline, oracle.spline)):
        ref = ofn(z, ogeom(gi), ogeom(go))
        got = fn(zt, gi, go).cpu().numpy()
        err = max_abs_err(got, ref)                                 # also asserts identical NaN patterns
        assert err <= 1e-5 * depth_range(ref), (name, seed, gi, go, err, depth_range(ref))


@pytest.mark.parametrize("seed", range(10))
def test_kriging_random_geometry(seed):
    import paper_2505_22675_b200 as b
    rng = np.random.default_rng(9300 + seed)
    n = int(rng.integers(40, 4000))
    span = float(rng.uniform(20, 300))
    xy = np.unique(rng.uniform(0, span, (n, 2)).astype(np.float32), axis=0)
    rng.shuffle(xy)
    x, y = np.ascontiguousarray(xy[:, 0]), np.ascontiguousarray(xy[:, 1])
    z = (-4000 + 0.2 * x - 0.1 * y + rng.normal(0, 2, x.size)).astype(np.float32)
    k = int(min(rng.choice([1, 4, 8, 12, 16, 24, 32, 48, 64]), x.size))
    model = int(rng.integers(0, 2))
    sill = W.sample_variance(z)
    nug = float(rng.choice([0.0, 0.01, 0.2])) * sill
    rng_a = float(rng.uniform(0.05, 0.6)) * span
    g = W.Geom(int(rng.integers(1, 70)), int(rng.integers(1, 50)), float(rng.uniform(-0.2, 0.3)) * span,
               float(rng.uniform(-0.2, 0.3)) * span, float(rng.uniform(0.002, 0.03)) * span, float(rng.uniform(0.002, 0.03)) * span)
    ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(model, rng_a, sill, nug), k)
    xt, yt, zt = (torch.from_numpy(a).cuda() for a in (x, y, z))
    idx = b.krige_build_index(xt, yt, zt)
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    got, nbr = b.krige_predict(idx, g, model, rng_a, sill, nug, k, want_nbr=True, failed=failed)
    idx.free()
    assert int(failed.item()) == 0 and ref["failed"] == 0
    assert np.array_equal(nbr.cpu().numpy(), ref["nbr"]), (seed, k, model)
    err = max_abs_err(got.cpu().numpy(), ref["zhat"])
    assert err <= 1e-4 * depth_range(ref["zhat"]), (seed, k, model, err, depth_range(ref["zhat"]))
