"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times, on sampled
outputs the oracle can compute one by one:
  configs 2 and 3 (bilinear, spline): every node of a few output rows and of a few output columns
      (the oracle runs on strided sub-geometries whose nodes coincide exactly with full-grid nodes);
  configs 4 and 5 (kriging): seeded random nodes, neighbour lists bit-exact, depths within 1e-4 x range;
      config 5 through 64 tile calls as bench.py issues them.
Tolerances are north_star's (1e-5 / 1e-4 of the depth range)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_22675_b200 import workloads as W
from _util import ogeom

pytestmark = pytest.mark.gpu


def _bathy():
    import paper_2505_22675_b200 as b
    return b


@pytest.mark.parametrize("config", [2, 3])
def test_grid_configs_full_size_sampled_rows_and_columns(config):
    b = _bathy()
    w = W.grid_config(config)
    gi, go = w.geom_in, w.geom_out
    zt = torch.from_numpy(w.z).cuda()
    rng = np.random.default_rng(7000 + config)
    zrange = float(w.z.max() - w.z.min())
    for name, fn, ofn in (("bilinear", b.interp_bilinear, oracle.bilinear), ("spline", b.interp_spline, oracle.spline)):
        got = fn(zt, gi, go).cpu().numpy()
        assert np.isfinite(got).all()
        # rows: a regular sub-grid of 6 output rows (stride chosen so that first and last row are included)
        stride = (go.ny - 1) // 5
        rows = np.arange(6) * stride
        sub = W.Geom(go.nx, 6, go.x0, go.y0, go.dx, go.dy * stride)
        ref = ofn(w.z, ogeom(gi), ogeom(sub))
        err_r = float(np.abs(got[rows, :] - ref).max())
        # columns: 6 output columns at a random offset
        off = int(rng.integers(0, stride))
        cols = off + np.arange(6) * stride
        cols = cols[cols < go.nx]
        subc = W.Geom(len(cols), go.ny, go.x0 + off * go.dx, go.y0, go.dx * stride, go.dy)
        refc = ofn(w.z, ogeom(gi), ogeom(subc))
        err_c = float(np.abs(got[:, cols] - refc).max())
        assert max(err_r, err_c) <= 1e-5 * zrange, (name, err_r, err_c, zrange)


def _sampled_kriging(w, got, nbr_fn, n_samples, seed):
    g = w.geom_out
    rng = np.random.default_rng(seed)
    sel = np.unique(np.concatenate([rng.integers(0, g.n, n_samples), [0, g.nx - 1, g.n - g.nx, g.n - 1]]))
    xq, yq = oracle.node_coords(ogeom(g))
    v = oracle.vgm(w.model, w.range_, w.sill, w.nugget)
    ref = oracle.krige_points(w.x, w.y, w.z, xq.ravel()[sel], yq.ravel()[sel], v, w.k, oracle.Buckets(w.x, w.y, 4.0))
    assert ref["failed"] == 0
    zrange = float(w.z.max() - w.z.min())
    err = float(np.abs(got.ravel()[sel] - ref["zhat"]).max())
    assert err <= 1e-4 * zrange, (err, zrange)
    nb = nbr_fn(sel)
    if nb is not None:
        assert np.array_equal(nb, ref["nbr"])


def test_config4_full_size_sampled_nodes():
    b = _bathy()
    w = W.sounding_config(4)
    xt, yt, zt = (torch.from_numpy(a).cuda() for a in (w.x, w.y, w.z))
    idx = b.krige_build_index(xt, yt, zt)
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    got, nbr = b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, want_nbr=True, failed=failed)
    idx.free()
    assert int(failed.item()) == 0
    nbr = nbr.cpu().numpy().reshape(-1, w.k)
    _sampled_kriging(w, got.cpu().numpy(), lambda sel: nbr[sel], 3000, 7004)


def test_config5_full_size_tiles_sampled_nodes():
    b = _bathy()
    w = W.sounding_config(5)
    g = w.geom_out
    xt, yt, zt = (torch.from_numpy(a).cuda() for a in (w.x, w.y, w.z))
    idx = b.krige_build_index(xt, yt, zt)
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    out = torch.full(g.shape, float("nan"), dtype=torch.float32, device="cuda")
    for (i0, j0, ny, nx) in w.tiles:                       # 64 tiles of 512^2 in arrival order, as bench.py
        tile = b.krige_predict(idx, W.tile_geom(g, i0, j0, ny, nx), w.model, w.range_, w.sill, w.nugget, w.k, failed=failed)
        out[i0:i0 + ny, j0:j0 + nx] = tile
    idx.free()
    assert int(failed.item()) == 0
    got = out.cpu().numpy()
    assert np.isfinite(got).all()
    _sampled_kriging(w, got, lambda sel: None, 1500, 7005)
