"""GPU parity, through the C ABI, of interp_catmull_rom against
the float64 oracle: max abs error <= 1e-5 x depth range, NaN patterns identical, the fallback to bilinear at
grid borders and next to NaN cells (the paper's Grid B workload: randomly removed cells)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_22675_b200 import workloads as W
from _util import ogeom, depth_range, max_abs_err

pytestmark = pytest.mark.gpu
TOL = 1e-5


def _run(z, gi, go):
    import paper_2505_22675_b200 as b
    return b.interp_catmull_rom(torch.from_numpy(np.ascontiguousarray(z)).cuda(), gi, go).cpu().numpy()


def _check(z, gi, go):
    ref = oracle.catmull_rom(z, ogeom(gi), ogeom(go))
    got = _run(z, gi, go)
    err = max_abs_err(got, ref)                                       # also: identical NaN patterns
    assert err <= TOL * depth_range(ref), (err, depth_range(ref))
    return got, ref


def test_config1_with_its_nan_cells():
    """Config 1 as generated: 10 % of the cells are NaN (Grid B style); x4 up-sampling."""
    w = W.grid_config(1)
    got, ref = _check(w.z, w.geom_in, w.geom_out)
    assert np.isnan(ref).any() and np.isfinite(ref).any()


@pytest.mark.parametrize("config,n_in,factor,nf,holes", [(2, 257, 4, 40, 0.0), (3, 600, 2, 200, 0.01), (3, 300, 3, 100, 0.05)])
def test_reduced_configs_with_holes(config, n_in, factor, nf, holes):
    w = W.grid_config(config, n_in=n_in, factor=factor, n_features=nf)
    z = w.z.copy()
    if holes:
        rng = np.random.default_rng(31)
        z.ravel()[rng.permutation(z.size)[: int(holes * z.size)]] = np.nan   # removal fractions of PAPER.md:L274, L299
    _check(z, w.geom_in, w.geom_out)


@pytest.mark.parametrize("seed", range(12))
def test_random_geometry(seed):
    rng = np.random.default_rng(9500 + seed)
    nx, ny = int(rng.integers(2, 200)), int(rng.integers(2, 150))
    gi = W.Geom(nx, ny, float(rng.uniform(-20, 20)), float(rng.uniform(-20, 20)), float(rng.choice([1.0, 0.5, 2.0])), float(rng.choice([1.0, 1.5])))
    rx, ry = float(rng.choice([1.0, 0.5, 0.25, 1 / 3, 0.37, 1.7, 4.0])), float(rng.choice([1.0, 0.5, 0.2, 0.43, 2.5]))
    wx, wy = (nx - 1) * gi.dx, (ny - 1) * gi.dy
    go = W.Geom(int(min(wx * 1.2 / (gi.dx * rx), 600)) + 1, int(min(wy * 1.2 / (gi.dy * ry), 400)) + 1,
                gi.x0 - 0.1 * wx, gi.y0 - 0.1 * wy, gi.dx * rx, gi.dy * ry)
    yy, xx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    z = (-5000 + 0.4 * xx + 0.3 * yy + 25 * np.sin(xx / 5.0) * np.cos(yy / 4.0) + rng.normal(0, 0.5, (ny, nx))).astype(np.float32)
    if seed % 2:
        z.ravel()[rng.permutation(z.size)[: max(1, z.size // 30)]] = np.nan
    _check(z, gi, go)


def test_quadratic_exact_and_knots():
    yy, xx = np.meshgrid(np.arange(40.0), np.arange(50.0), indexing="ij")
    z = (2.0 + 0.5 * xx - 0.25 * yy + 0.125 * xx * xx - 0.5 * xx * yy + 0.375 * yy * yy).astype(np.float32)
    gi, go = W.Geom(50, 40, 0, 0, 1, 1), W.Geom(4 * 47 + 1, 4 * 37 + 1, 1.0, 1.0, 0.25, 0.25)
    got = _run(z, gi, go)
    X, Y = 1.0 + 0.25 * np.arange(go.nx), 1.0 + 0.25 * np.arange(go.ny)
    want = 2.0 + 0.5 * X[None] - 0.25 * Y[:, None] + 0.125 * X[None] ** 2 - 0.5 * X[None] * Y[:, None] + 0.375 * Y[:, None] ** 2
    inside = (X[None] <= 47.0) & (Y[:, None] <= 37.0)
    assert np.abs(got - want)[inside].max() <= 2e-4                  # fp32 at |z| ~ 600
    assert np.array_equal(got[::4, ::4], z[1:39, 1:49][: got[::4, ::4].shape[0], : got[::4, ::4].shape[1]])   # knots bit-exact


# (full-size config 2 / config 3 parity on EVERY node: tests/test_gpu_full_size.py)
