"""GPU parity, through the C ABI, of krige_predict_aniso (reading Ani)
against oracle_krige_points_aniso: neighbour lists bit-exact (they do not depend on the anisotropy), depths within
1e-4 x depth range, kriging variance within 1e-4 x sill -- the bars of the isotropic kriging tests."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_22675_b200 import workloads as W
from _util import ogeom, depth_range, max_abs_err

pytestmark = pytest.mark.gpu


def _bathy():
    import paper_2505_22675_b200 as b
    return b


def _dev(*arrays):
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays)


@pytest.mark.parametrize("config,width,n_out,angle,ratio", [(4, 250.0, 160, 30.0, 0.4), (4, 250.0, 96, -72.0, 0.7),
                                                            (5, 300.0, 120, 115.0, 0.25), (5, 300.0, 64, 0.0, 0.5)])
def test_survey_like_configs(config, width, n_out, angle, ratio):
    """Reduced configs 4 (k = 32, exponential) and 5 (k = 64, spherical), same density and recipe as the full ones."""
    b = _bathy()
    w = W.sounding_config(config, width=width, n_target=int(width * width / 4), n_out=n_out)
    a = oracle.aniso(angle, ratio)
    ref = oracle.krige_grid(w.x, w.y, w.z, ogeom(w.geom_out), oracle.vgm(w.model, w.range_, w.sill, w.nugget), w.k,
                            oracle.Buckets(w.x, w.y, 4.0), a=a)
    iso = oracle.krige_grid(w.x, w.y, w.z, ogeom(w.geom_out), oracle.vgm(w.model, w.range_, w.sill, w.nugget), w.k,
                            oracle.Buckets(w.x, w.y, 4.0))
    idx = b.krige_build_index(*_dev(w.x, w.y, w.z))
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    got, nbr, var = b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, want_nbr=True, want_var=True,
                                    failed=failed, aniso=(angle, ratio))
    plain = b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, aniso=(angle, ratio))
    idx.free()
    assert int(failed.item()) == 0 and ref["failed"] == 0
    assert torch.equal(plain, got)
    assert np.array_equal(nbr.cpu().numpy(), ref["nbr"]) and np.array_equal(ref["nbr"], iso["nbr"])
    rng = depth_range(ref["zhat"])
    assert max_abs_err(got.cpu().numpy(), ref["zhat"]) <= 1e-4 * rng
    assert max_abs_err(var.cpu().numpy(), ref["var"]) <= 1e-4 * w.sill
    assert float(np.abs(ref["zhat"] - iso["zhat"]).max()) > 0.0                   # (the expected values are not the isotropic ones)
    print("aniso vs iso, max |dz| / tol:", float(np.abs(ref["zhat"] - iso["zhat"]).max()) / (1e-4 * rng))


@pytest.mark.parametrize("k,model", [(4, 2), (8, 0), (16, 1)])
def test_small_k_all_models_and_nodes_on_data(k, model):
    b = _bathy()
    rng = np.random.default_rng(1200 + k)
    xy = np.unique(rng.uniform(0, 100, (2500, 2)).astype(np.float32), axis=0)
    rng.shuffle(xy)
    x, y = np.ascontiguousarray(xy[:, 0]), np.ascontiguousarray(xy[:, 1])
    z = (-4000 + 3.0 * np.sin(x / 9.0) + 0.1 * y + rng.normal(0, 0.5, x.size)).astype(np.float32)
    sill = W.sample_variance(z)
    nug = 0.05 * sill if model == 2 else 0.0
    g = W.Geom(57, 41, -2.0, -1.0, 1.8, 2.5)
    a = oracle.aniso(52.0, 0.35)
    ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(model, 6.0, sill, nug), k, a=a)
    idx = b.krige_build_index(*_dev(x, y, z))
    got, nbr, var = b.krige_predict(idx, g, model, 6.0, sill, nug, k, want_nbr=True, want_var=True, aniso=(52.0, 0.35))
    # nodes that coincide with soundings: exact interpolation (no nugget), variance 0
    at = b.krige_predict(idx, W.Geom(1, 1, float(x[7]), float(y[7]), 1.0, 1.0), model, 6.0, sill, 0.0, k, aniso=(52.0, 0.35))
    idx.free()
    assert np.array_equal(nbr.cpu().numpy(), ref["nbr"])
    assert max_abs_err(got.cpu().numpy(), ref["zhat"]) <= 1e-4 * depth_range(ref["zhat"])
    assert max_abs_err(var.cpu().numpy(), ref["var"]) <= 1e-4 * sill
    assert abs(float(at[0, 0]) - float(z[7])) <= 1e-4 * depth_range(ref["zhat"])


def test_ratio_one_is_the_isotropic_call_and_bad_ratios_are_refused():
    b = _bathy()
    w = W.sounding_config(4, width=150.0, n_target=5600, n_out=96)
    idx = b.krige_build_index(*_dev(w.x, w.y, w.z))
    args = (w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k)
    iso = b.krige_predict(idx, *args)
    assert torch.equal(b.krige_predict(idx, *args, aniso=(0.0, 1.0)), iso)            # the identity map: bit for bit
    rot = b.krige_predict(idx, *args, aniso=(77.0, 1.0))                              # a pure rotation: the same lags up to rounding
    assert float((rot - iso).abs().max()) <= 1e-4 * float(iso.max() - iso.min())
    for ratio in (0.0, -1.0, 1.01, float("nan")):
        with pytest.raises(b.BathyError) as e:
            b.krige_predict(idx, *args, aniso=(10.0, ratio))
        assert e.value.status == -4                                                   # BATHY_ERR_VARIOGRAM
    with pytest.raises(b.BathyError):
        b.krige_predict(idx, *args, aniso=(float("inf"), 0.5))
    idx.free()
