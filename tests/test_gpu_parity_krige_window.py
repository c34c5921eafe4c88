"""GPU parity, through the C ABI, of interp_krige_window (PAPER.md:L163, L171, L179-L180,
L225-L234) against oracle_krige_window: the `how` map (copied / kriged from n neighbours / bilinear fallback)
bit-exact, NaN patterns identical, depths within 1e-4 x depth range (the kriging bar of north_star), valid cells
copied bit-exactly."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_22675_b200 import workloads as W
from _util import ogeom, depth_range, max_abs_err

pytestmark = pytest.mark.gpu
TOL = 1e-4


def _bathy():
    import paper_2505_22675_b200 as b
    return b


def _holed(config, n_in, nf, frac, seed):
    w = W.grid_config(config, n_in=n_in, factor=2, n_features=nf)
    z = np.where(np.isnan(w.z), np.float32(-5000.0), w.z).copy()
    rng = np.random.default_rng(seed)
    z[rng.random(z.shape) < frac] = np.nan                    # the paper's removal fractions: 0.01, 0.05, 0.1 (L274, L299)
    return z, w.geom_in


def _check(z, g, model, a, sill, nug, **kw):
    b = _bathy()
    ref = oracle.krige_window(z, ogeom(g), oracle.vgm(model, a, sill, nug), **kw)
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    out, how = b.interp_krige_window(torch.from_numpy(z).cuda(), g, model, a, sill, nug, want_how=True, failed=failed, **kw)
    out, how = out.cpu().numpy(), how.cpu().numpy()
    assert np.array_equal(how, ref["how"]), f"{int((how != ref['how']).sum())} cells with a different method/neighbour count"
    assert int(failed.item()) == ref["failed"]
    err = max_abs_err(out, ref["out"])                          # also: identical NaN patterns
    assert err <= TOL * depth_range(ref["out"]), (err, depth_range(ref["out"]))
    valid = ~np.isnan(z)
    assert np.array_equal(out[valid], z[valid])
    return out, how, ref


def test_config1_holes():
    """Config 1 as generated (64 x 64, 410 random NaN cells): 5 x 5 window, exponential variogram of PAPER.md:L157."""
    w = W.grid_config(1)
    sill = W.sample_variance(w.z[~np.isnan(w.z)])
    out, how, _ = _check(w.z, w.geom_in, 0, 10.0, sill, 0.0)
    assert (how[w.nan_mask] > 0).all() and np.isfinite(out).all()


@pytest.mark.parametrize("frac", [0.01, 0.05, 0.1])
@pytest.mark.parametrize("half,model", [(2, 0), (1, 1), (3, 0), (2, 2)])
def test_removal_fractions(frac, half, model):
    z, g = _holed(2, 300, 60, frac, 500 + int(frac * 100) + half)
    sill = W.sample_variance(z[~np.isnan(z)])
    _check(z, g, model, 12.0, sill, 0.02 * sill if model == 2 else 0.0, half=half)


@pytest.mark.parametrize("n_max,n_min", [(4, 1), (8, 3), (12, 12), (24, 25), (1, 1), (30, 5)])
def test_nearest_n_and_fallback(n_max, n_min):
    z, g = _holed(2, 200, 30, 0.3, 77)                          # 30 % holes: every neighbour count occurs
    sill = W.sample_variance(z[~np.isnan(z)])
    out, how, ref = _check(z, g, 0, 9.0, sill, 0.01 * sill, half=2, n_max=n_max, n_min=n_min)
    holes = np.isnan(z)
    if n_min > 24:
        assert (how[holes] == 255).all()
    else:
        assert (how[holes] == 255).any() or (how[holes] <= min(n_max, 24)).all()


def test_rectangular_spacing_borders_and_dense_holes():
    rng = np.random.default_rng(8)
    z = (-3000 + 40 * np.sin(np.arange(83)[None, :] / 6.0) + 25 * np.cos(np.arange(47)[:, None] / 4.0) + rng.normal(0, 0.5, (47, 83))).astype(np.float32)
    z[rng.random(z.shape) < 0.6] = np.nan
    z[0, :5] = np.nan; z[-1, -3:] = np.nan; z[:4, 0] = np.nan
    g = W.Geom(83, 47, 1000.0, -500.0, 2.5, 1.5)
    sill = W.sample_variance(z[~np.isnan(z)])
    out, how, ref = _check(z, g, 1, 15.0, sill, 0.0, half=2, n_min=3)
    assert np.isnan(out).any() and (how == 255).any()
    _check(z, g, 0, 15.0, sill, 0.05 * sill, half=3, n_max=20, n_min=2)


def test_all_valid_and_all_nan():
    b = _bathy()
    z = np.arange(30, dtype=np.float32).reshape(5, 6)
    g = W.Geom(6, 5, 0.0, 0.0, 1.0, 1.0)
    out, how = b.interp_krige_window(torch.from_numpy(z).cuda(), g, 0, 3.0, 1.0, 0.0, want_how=True)
    assert np.array_equal(out.cpu().numpy(), z) and (how.cpu().numpy() == 0).all()
    out, how = b.interp_krige_window(torch.full((5, 6), float("nan")).cuda(), g, 0, 3.0, 1.0, 0.0, want_how=True)
    assert torch.isnan(out).all() and (how.cpu().numpy() == 255).all()
    for kw, status in ((dict(half=0), -3), (dict(half=4), -3), (dict(n_min=0), -3), (dict(n_max=0), -3)):
        with pytest.raises(b.BathyError) as e:
            b.interp_krige_window(torch.from_numpy(z).cuda(), g, 0, 3.0, 1.0, 0.0, **kw)
        assert e.value.status == status


def test_full_size_4096_with_5_percent_holes():
    """The paper's Grid B workload at scale: 4096^2 grid, 5 % of the cells removed, 5 x 5 window."""
    w = W.grid_config(3)
    z = w.z.copy()
    rng = np.random.default_rng(4096)
    z[rng.random(z.shape) < 0.05] = np.nan
    sill = W.sample_variance(z[~np.isnan(z)][::97])
    out, how, ref = _check(z, w.geom_in, 0, 12.0, sill, 0.0)
    assert np.isfinite(out).all()
