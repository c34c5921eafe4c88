"""GPU parity, through the C ABI, of krige_build_index + krige_predict against the float64 oracle.
Bar (BASELINE.json north_star): neighbour indices bit-exact (ties broken by index), depths within
1e-4 x depth range of the oracle output."""
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


def _gpu(x, y, z, g, model, range_, sill, nugget, k, cell=0.0, want_nbr=True):
    b = _bathy()
    xt, yt, zt = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (x, y, z))
    idx = b.krige_build_index(xt, yt, zt, cell)
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    res = b.krige_predict(idx, g, model, range_, sill, nugget, k, want_nbr=want_nbr, failed=failed)
    torch.cuda.synchronize()
    info = idx.info()
    idx.free()
    if want_nbr:
        return res[0].cpu().numpy(), res[1].cpu().numpy(), int(failed.item()), info
    return res.cpu().numpy(), None, int(failed.item()), info


def _check(got, nbr, ref, k):
    assert np.array_equal(nbr, ref["nbr"]), f"{int((nbr != ref['nbr']).any(axis=-1).sum())} nodes with wrong neighbours"
    err = max_abs_err(got, ref["zhat"])
    assert err <= TOL * depth_range(ref["zhat"]), (err, depth_range(ref["zhat"]))


def test_config1_full():
    """64x64 grid with 10 % NaN, valid cells as scattered points (lattice: many exact key ties),
    k=8, spherical, range 10 m, sill = sample variance, nugget 0, onto the 253^2 grid."""
    w = W.grid_config(1)
    x, y, z = W.grid_to_scattered(w.z)
    sill = W.sample_variance(z)
    ref = oracle.krige_grid(x, y, z, ogeom(w.geom_out), oracle.vgm(oracle.SPHERICAL, 10.0, sill, 0.0), 8)
    got, nbr, failed, _ = _gpu(x, y, z, w.geom_out, 1, 10.0, sill, 0.0, 8)
    assert failed == 0 and ref["failed"] == 0
    _check(got, nbr, ref, 8)
    # exact interpolator at the data: every 4th node that sits on a valid cell returns its depth
    on = ~w.nan_mask
    assert np.abs(got[::4, ::4][on] - w.z[on]).max() <= 1e-3


def test_config1_pipeline_fill_then_upsample():
    """End to end on the GPU: kriging fills the NaN cells, then bilinear and spline upsample the
    filled grid; compared with the all-oracle pipeline under the kriging tolerance."""
    b = _bathy()
    w = W.grid_config(1)
    x, y, z = W.grid_to_scattered(w.z)
    sill = W.sample_variance(z)
    v = oracle.vgm(oracle.SPHERICAL, 10.0, sill, 0.0)
    ii, jj = np.nonzero(w.nan_mask)
    fill_ref = oracle.krige_points(x, y, z, jj.astype(np.float32), ii.astype(np.float32), v, 8)["zhat"]
    filled_ref = w.z.copy()
    filled_ref[ii, jj] = fill_ref.astype(np.float32)
    got64, _, failed, _ = _gpu(x, y, z, w.geom_in, 1, 10.0, sill, 0.0, 8, want_nbr=False)
    assert failed == 0
    filled_gpu = np.where(w.nan_mask, got64, w.z).astype(np.float32)
    zt = torch.from_numpy(filled_gpu).cuda()
    for name, fn, ofn in (("bilinear", b.interp_bilinear, oracle.bilinear), ("spline", b.interp_spline, oracle.spline)):
        ref = ofn(filled_ref, ogeom(w.geom_in), ogeom(w.geom_out))
        got = fn(zt, w.geom_in, w.geom_out).cpu().numpy()
        assert max_abs_err(got, ref) <= TOL * depth_range(ref), name


@pytest.mark.parametrize("config,width,n_out", [(4, 250.0, 200), (5, 300.0, 160)])
def test_reduced_configs_4_5(config, width, n_out):
    """Same swath generator and density (0.25 /m^2), reduced area; k=32 exponential / k=64 spherical."""
    w = W.sounding_config(config, width=width, n_target=int(width * width / 4), n_out=n_out)
    v = oracle.vgm(w.model, w.range_, w.sill, w.nugget)
    buckets = oracle.Buckets(w.x, w.y, 4.0)
    ref = oracle.krige_grid(w.x, w.y, w.z, ogeom(w.geom_out), v, w.k, buckets)
    got, nbr, failed, info = _gpu(w.x, w.y, w.z, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k)
    assert failed == 0 and ref["failed"] == 0
    _check(got, nbr, ref, w.k)
    # tiles (sub-geometries) reproduce the monolithic output bit for bit (per-node independence)
    b = _bathy()
    xt, yt, zt = (torch.from_numpy(a).cuda() for a in (w.x, w.y, w.z))
    idx = b.krige_build_index(xt, yt, zt)
    tiled = np.full_like(got, np.nan)
    for (i0, j0, ny, nx) in W.boustrophedon_tiles(n_out, 64):
        tg = W.tile_geom(w.geom_out, i0, j0, ny, nx)
        tiled[i0:i0 + ny, j0:j0 + nx] = b.krige_predict(idx, tg, w.model, w.range_, w.sill, w.nugget, w.k).cpu().numpy()
    idx.free()
    # dx = width/n_out (1.25, 1.875) and x0 = dx/2 are exact in binary, as in configs 4-5, so a tile's
    # nodes are bit-identical to the monolithic grid's nodes and so must the depths be
    assert np.array_equal(tiled, got)
    # another cell size gives the same neighbours and the same depths
    got2, nbr2, _, info2 = _gpu(w.x, w.y, w.z, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, cell=info["cell_size"] * 0.37)
    assert info2["ncx"] > info["ncx"]
    assert np.array_equal(nbr2, nbr)
    assert np.abs(got2 - got).max() <= 1e-3


@pytest.mark.parametrize("k", [1, 2, 3, 5, 8, 9, 16, 17, 31, 33, 64])
def test_all_k(k):
    rng = np.random.default_rng(100 + k)
    n = 700
    x, y = rng.uniform(0, 60, n).astype(np.float32), rng.uniform(0, 40, n).astype(np.float32)
    z = (-4000 + 2.0 * x + rng.normal(0, 3, n)).astype(np.float32)
    g = W.Geom(47, 31, -3.0, -2.0, 1.4, 1.45)                    # includes nodes outside the bounding box
    for model, nug in ((0, 0.05), (1, 0.0)):
        sill = W.sample_variance(z)
        ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(model, 15.0, sill, nug * sill), k)
        got, nbr, failed, _ = _gpu(x, y, z, g, model, 15.0, sill, nug * sill, k)
        assert failed == 0
        _check(got, nbr, ref, k)


def test_k_equals_n_and_tiny_inputs():
    rng = np.random.default_rng(31)
    for n in (1, 2, 5, 64):
        x, y = rng.uniform(0, 10, n).astype(np.float32), rng.uniform(0, 10, n).astype(np.float32)
        z = rng.normal(-100, 5, n).astype(np.float32)
        g = W.Geom(9, 7, 0.0, 0.0, 1.25, 1.5)
        ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(0, 8.0, 25.0, 0.25), n)
        got, nbr, failed, _ = _gpu(x, y, z, g, 0, 8.0, 25.0, 0.25, n)
        assert failed == 0
        _check(got, nbr, ref, n)


def test_constant_field_and_exact_at_data():
    rng = np.random.default_rng(32)
    n = 2000
    x, y = rng.uniform(0, 100, n).astype(np.float32), rng.uniform(0, 100, n).astype(np.float32)
    g = W.Geom(64, 64, 0.5, 0.5, 1.5, 1.5)
    got, _, failed, _ = _gpu(x, y, np.full(n, -4321.5, np.float32), g, 0, 20.0, 1.0, 0.01, 32, want_nbr=False)
    assert failed == 0 and np.abs(got + 4321.5).max() <= 1e-3      # weights sum to 1
    # nodes that coincide with soundings return the sounding (nugget 0 and nugget > 0 under gamma(0) = 0)
    xs, ys = np.meshgrid(np.arange(40, dtype=np.float32), np.arange(30, dtype=np.float32))
    z = rng.normal(-5000, 20, xs.size).astype(np.float32)
    gl = W.Geom(40, 30, 0.0, 0.0, 1.0, 1.0)
    for nug in (0.0, 40.0):
        got, nbr, failed, _ = _gpu(xs.ravel(), ys.ravel(), z, gl, 1, 6.0, 400.0, nug, 8)
        assert failed == 0
        assert np.array_equal(nbr[..., 0].ravel(), np.arange(xs.size))
        assert np.abs(got.ravel() - z).max() <= 2e-3


def test_duplicates_fail_as_nan_and_are_counted():
    x = np.array([0, 0, 1, 2, 3, 5], np.float32)
    y = np.array([0, 0, 0, 1, 2, 1], np.float32)
    z = np.array([1, 2, 3, 4, 5, 6], np.float32)
    g = W.Geom(3, 2, 0.25, 0.25, 0.5, 0.5)
    got, _, failed, _ = _gpu(x, y, z, g, 0, 10.0, 1.0, 0.1, 6, want_nbr=False)
    assert failed == 6 and np.isnan(got).all()


def test_argument_errors():
    b = _bathy()
    x = torch.zeros(10, device="cuda")
    idx = b.krige_build_index(torch.arange(10, dtype=torch.float32, device="cuda"), x, x)
    g = W.Geom(4, 4, 0, 0, 1, 1)
    for kw, status in ((dict(model=0, range_=0.0, sill=1, nugget=0, k=4), -4),
                       (dict(model=0, range_=1.0, sill=0.0, nugget=0, k=4), -4),
                       (dict(model=0, range_=1.0, sill=1.0, nugget=2.0, k=4), -4),
                       (dict(model=3, range_=1.0, sill=1.0, nugget=0.0, k=4), -4),
                       (dict(model=0, range_=1.0, sill=1.0, nugget=0.0, k=0), -3),
                       (dict(model=0, range_=1.0, sill=1.0, nugget=0.0, k=11), -3),
                       (dict(model=0, range_=1.0, sill=1.0, nugget=0.0, k=65), -3)):
        with pytest.raises(b.BathyError) as e:
            b.krige_predict(idx, g, **kw)
        assert e.value.status == status
    idx.free()
    # (non-finite soundings are found on the device: tests/test_gpu_streaming_and_boundary.py)


def test_host_form():
    b = _bathy()
    w = W.sounding_config(4, width=150.0, n_target=5600, n_out=96)
    dev, _, _, _ = _gpu(w.x, w.y, w.z, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, want_nbr=False)
    host, failed = b.krige_host(w.x, w.y, w.z, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k)
    assert failed == 0 and np.array_equal(dev, host)


def test_large_coordinates_and_clustered_density():
    """Search bounds under stress: UTM-like coordinates (fp32 ulp 0.03 m) and a density that varies by
    three orders of magnitude (forces the block search to split down to single nodes)."""
    rng = np.random.default_rng(77)
    # (a) large offsets
    x = (500000.0 + rng.uniform(0, 120, 3000)).astype(np.float32)
    y = (4200000.0 + rng.uniform(0, 90, 3000)).astype(np.float32)
    xy = np.unique(np.stack([x, y], 1), axis=0)
    rng.shuffle(xy)
    x, y = np.ascontiguousarray(xy[:, 0]), np.ascontiguousarray(xy[:, 1])
    z = (-3000 + 0.05 * (x - 500000.0) + rng.normal(0, 2, x.size)).astype(np.float32)
    g = W.Geom(50, 38, 499990.0, 4199990.0, 3.0, 3.0)
    for k, model in ((16, 0), (32, 1)):
        sill = W.sample_variance(z)
        ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(model, 40.0, sill, 0.02 * sill), k)
        got, nbr, failed, _ = _gpu(x, y, z, g, model, 40.0, sill, 0.02 * sill, k)
        assert failed == 0 and ref["failed"] == 0
        _check(got, nbr, ref, k)
    # (b) a dense clump inside a sparse field
    xs = np.concatenate([rng.uniform(0, 200, 1500), 100 + rng.uniform(0, 4, 6000)])
    ys = np.concatenate([rng.uniform(0, 200, 1500), 100 + rng.uniform(0, 4, 6000)])
    xy = np.unique(np.stack([xs.astype(np.float32), ys.astype(np.float32)], 1), axis=0)
    rng.shuffle(xy)
    x, y = np.ascontiguousarray(xy[:, 0]), np.ascontiguousarray(xy[:, 1])
    z = (-4000 + 0.3 * x + rng.normal(0, 1, x.size)).astype(np.float32)
    g = W.Geom(64, 48, 70.0, 80.0, 1.0, 1.0)
    sill = W.sample_variance(z)
    ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(0, 30.0, sill, 0.05 * sill), 32)
    got, nbr, failed, _ = _gpu(x, y, z, g, 0, 30.0, sill, 0.05 * sill, 32)
    assert failed == 0 and ref["failed"] == 0
    assert np.array_equal(nbr, ref["nbr"])
    # in the clump neighbours are centimetres apart under a 30 m range; the depth bar holds there too
    assert max_abs_err(got, ref["zhat"]) <= TOL * depth_range(ref["zhat"])


def test_stream_ordered_release_and_rebuild():
    """krige_free_index_async: build -> predict -> release -> build again on the same stream, no host
    synchronisation in between; results are bit-identical from call to call."""
    b = _bathy()
    w = W.sounding_config(4, width=120.0, n_target=3600, n_out=64)
    xt, yt, zt = (torch.from_numpy(a).cuda() for a in (w.x, w.y, w.z))
    outs = []
    for _ in range(4):
        idx = b.krige_build_index(xt, yt, zt)
        outs.append(b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k))
        idx.free_async()
        assert idx.handle is None
    torch.cuda.synchronize()
    for o in outs[1:]:
        assert torch.equal(o, outs[0])
    assert torch.isfinite(outs[0]).all()


def test_async_host_forms_on_three_streams():
    # the enqueue-only host forms (include/bathy.h): three methods on three streams, results
    # defined after the streams are synchronised, bit-identical to the device-pointer forms
    b = _bathy()
    w = W.sounding_config(4, width=150.0, n_target=5600, n_out=96)
    gw = W.grid_config(2, n_in=129, factor=4, n_features=10)
    dev_k, _, _, _ = _gpu(w.x, w.y, w.z, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, want_nbr=False)
    zt = torch.from_numpy(gw.z).cuda()
    dev_b = b.interp_bilinear(zt, gw.geom_in, gw.geom_out).cpu().numpy()
    dev_s = b.interp_spline(zt, gw.geom_in, gw.geom_out).cpu().numpy()
    hx, hy, hz = (torch.from_numpy(a).pin_memory() for a in (w.x, w.y, w.z))
    hg = torch.from_numpy(gw.z).pin_memory()
    ok = torch.full(w.geom_out.shape, -1.0, dtype=torch.float32).pin_memory()
    ob = torch.full(gw.geom_out.shape, -1.0, dtype=torch.float32).pin_memory()
    os_ = torch.full(gw.geom_out.shape, -1.0, dtype=torch.float32).pin_memory()
    failed = torch.full((1,), -1, dtype=torch.int64).pin_memory()
    sk, sb, ss = (torch.cuda.Stream() for _ in range(3))
    for _ in range(3):                                   # repeated: scratch comes from and returns to the stream pool
        b.krige_host_async(hx, hy, hz, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, out=ok, failed=failed, stream=sk)
        b.interp_bilinear_host_async(hg, gw.geom_in, gw.geom_out, out=ob, stream=sb)
        b.interp_spline_host_async(hg, gw.geom_in, gw.geom_out, out=os_, stream=ss)
        for s_ in (sk, sb, ss):
            s_.synchronize()
        assert int(failed[0]) == 0
        assert np.array_equal(ok.numpy(), dev_k) and np.array_equal(ob.numpy(), dev_b) and np.array_equal(os_.numpy(), dev_s)
        ok.fill_(-1.0); ob.fill_(-1.0); os_.fill_(-1.0)
    with pytest.raises(TypeError):
        b.interp_bilinear_host_async(torch.from_numpy(gw.z), gw.geom_in, gw.geom_out, out=ob)      # not pinned


@pytest.mark.parametrize("k,model", [(8, 1), (32, 0), (64, 1)])
def test_repeated_launches_are_bit_identical(k, model):
    """Stands in for racecheck (closed on the pool, profiles/r2_sanitizer_refusal.md): a data race in the
    __syncwarp-ordered shared-memory buffers of the solve would make the result timing dependent; 12 launches, with
    another stream keeping the SMs busy, give bit-identical depths and variances."""
    b = _bathy()
    w = W.sounding_config(4, width=200.0, n_target=10000, n_out=160)
    xt, yt, zt = (torch.from_numpy(a).cuda() for a in (w.x, w.y, w.z))
    idx = b.krige_build_index(xt, yt, zt)
    side = torch.cuda.Stream()
    noise = torch.randn(2048, 2048, device="cuda")
    first = None
    for it in range(12):
        with torch.cuda.stream(side):
            for _ in range(it % 4):
                noise = torch.tanh(noise @ noise * 1e-3)
        z, var = b.krige_predict(idx, w.geom_out, model, 60.0, w.sill, w.nugget, k, want_var=True)
        if first is None:
            first = (z.clone(), var.clone())
        else:
            assert torch.equal(z, first[0]) and torch.equal(var, first[1])
    torch.cuda.synchronize()
    idx.free()
    assert torch.isfinite(first[0]).all()
