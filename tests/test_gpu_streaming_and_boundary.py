"""GPU tests of the boundary conventions (every device-pointer call only enqueues) and of the
SURVEY.md 8(f) NEXT-3 / NEXT-4 rows: appendable index (krige_index_create / krige_index_append), kriging
variance and ill-conditioning counter (krige_predict_ex), Gaussian variogram -- each against the float64 oracle."""
import threading
import time

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


def test_device_pointer_calls_only_enqueue():
    """No exported device-pointer call blocks the host: each returns while a long kernel queued ahead of it on
    the same stream is still running (checked by an event query), krige_build_index included."""
    b = _bathy()
    w = W.sounding_config(4, width=150.0, n_target=5600, n_out=96)
    gw = W.grid_config(2, n_in=129, factor=4, n_features=10)
    xt, yt, zt = _dev(w.x, w.y, w.z)
    gz, = _dev(gw.z)
    st = torch.cuda.Stream()
    ref_idx = b.krige_build_index(xt, yt, zt)
    ref_k = b.krige_predict(ref_idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k)
    ref_b = b.interp_bilinear(gz, gw.geom_in, gw.geom_out)
    ref_s = b.interp_spline(gz, gw.geom_in, gw.geom_out)
    ref_c = b.interp_catmull_rom(gz, gw.geom_in, gw.geom_out)
    torch.cuda.synchronize()
    ws = torch.empty(b.interp_spline_workspace_bytes(gw.geom_in, gw.geom_out), dtype=torch.uint8, device="cuda")
    outs = [torch.empty_like(ref_b) for _ in range(3)]
    out_k = torch.empty_like(ref_k)
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    with torch.cuda.stream(st):
        torch.cuda._sleep(int(1.5e9))                      # ~0.7 s of spinning ahead of everything below
        blocker = torch.cuda.Event()
        blocker.record(st)
        t0 = time.perf_counter()
        idx = b.krige_build_index(xt, yt, zt, stream=st)
        b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, out=out_k, failed=failed, stream=st)
        idx2 = b.krige_index_create(0.0, 150.0, 0.0, 150.0, capacity=w.x.size, stream=st)
        b.krige_index_append(idx2, xt, yt, zt, stream=st)
        b.interp_bilinear(gz, gw.geom_in, gw.geom_out, out=outs[0], stream=st)
        b.interp_spline(gz, gw.geom_in, gw.geom_out, out=outs[1], workspace=ws, stream=st)
        b.interp_catmull_rom(gz, gw.geom_in, gw.geom_out, out=outs[2], stream=st)
        idx.free_async(stream=st)
        idx2.free_async(stream=st)
        dt = time.perf_counter() - t0
        still_running = not blocker.query()
    assert still_running, f"a call blocked the host until the queued kernel finished ({dt:.3f} s)"
    st.synchronize()
    assert int(failed.item()) == 0
    assert torch.equal(out_k, ref_k) and torch.equal(outs[0], ref_b) and torch.equal(outs[1], ref_s)
    assert torch.equal(outs[2], ref_c)
    ref_idx.free()


def test_non_finite_soundings_are_reported_on_the_device():
    b = _bathy()
    x = torch.tensor([0.0, float("nan"), 2.0, 3.0], device="cuda")
    y = torch.zeros(4, device="cuda")
    idx = b.krige_build_index(x, y, y)
    with pytest.raises(b.BathyError) as e:
        idx.info()
    assert e.value.status == -2
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    got = b.krige_predict(idx, W.Geom(5, 3, 0, 0, 1, 1), 0, 1.0, 1.0, 0.0, 2, failed=failed)
    assert torch.isnan(got).all() and int(failed.item()) == 15
    idx.free()


def test_append_equals_one_shot_and_the_oracle():
    """create + append(A) + append(B) == create + append(A|B) bit for bit; after append(A) alone the estimate is
    the oracle's on A alone (streaming: predict with the data so far); neighbours bit-exact throughout."""
    b = _bathy()
    w = W.sounding_config(4, width=200.0, n_target=10000, n_out=128)
    n = w.x.size
    cut = int(0.55 * n)                                   # survey order: the first lines, then the rest
    xt, yt, zt = _dev(w.x, w.y, w.z)
    g = w.geom_out
    v = oracle.vgm(w.model, w.range_, w.sill, w.nugget)

    def predict(idx):
        failed = torch.zeros(1, dtype=torch.int64, device="cuda")
        z, nb = b.krige_predict(idx, g, w.model, w.range_, w.sill, w.nugget, w.k, want_nbr=True, failed=failed)
        assert int(failed.item()) == 0
        return z.cpu().numpy(), nb.cpu().numpy()

    changed = torch.zeros(4, device="cuda")
    two = b.krige_index_create(0.0, 200.0, 0.0, 200.0, capacity=n)
    b.krige_index_append(two, xt[:cut], yt[:cut], zt[:cut], changed=changed)
    assert two.info()["n"] == cut
    zA, nA = predict(two)
    refA = oracle.krige_grid(w.x[:cut], w.y[:cut], w.z[:cut], ogeom(g), v, w.k)
    assert np.array_equal(nA, refA["nbr"])
    assert max_abs_err(zA, refA["zhat"]) <= 1e-4 * depth_range(refA["zhat"])
    b.krige_index_append(two, xt[cut:], yt[cut:], zt[cut:], changed=changed)
    assert two.info()["n"] == n
    ch = changed.cpu().numpy()
    assert np.allclose(ch, [w.x[cut:].min(), w.x[cut:].max(), w.y[cut:].min(), w.y[cut:].max()], rtol=0, atol=0)
    z2, n2 = predict(two)

    one = b.krige_index_create(0.0, 200.0, 0.0, 200.0, capacity=n)
    b.krige_index_append(one, xt, yt, zt)
    z1, n1 = predict(one)
    assert np.array_equal(n1, n2) and np.array_equal(z1, z2), "append(A) + append(B) differs from append(A|B)"
    assert one.info() == two.info()

    ref = oracle.krige_grid(w.x, w.y, w.z, ogeom(g), v, w.k)
    assert np.array_equal(n2, ref["nbr"])
    assert max_abs_err(z2, ref["zhat"]) <= 1e-4 * depth_range(ref["zhat"])
    # nodes farther from every new sounding than their k-th neighbour are untouched by the append
    same = (nA == n2).all(axis=-1)
    assert same.any() and np.array_equal(zA[same], z2[same])
    # the one-shot index over the bounding box finds the same neighbours
    shot = b.krige_build_index(xt, yt, zt)
    z3, n3 = predict(shot)
    assert np.array_equal(n3, n2) and np.abs(z3 - z2).max() <= 1e-3
    # capacity is enforced, and a one-shot index is not appendable
    with pytest.raises(b.BathyError) as e:
        b.krige_index_append(two, xt[:1], yt[:1], zt[:1])
    assert e.value.status == -7
    with pytest.raises(b.BathyError) as e:
        b.krige_index_append(shot, xt[:1], yt[:1], zt[:1])
    assert e.value.status == -8
    for i in (one, two, shot):
        i.free()


def test_append_many_small_batches_and_points_outside_the_extent():
    b = _bathy()
    rng = np.random.default_rng(41)
    n = 3000
    xy = np.unique(rng.uniform(-20, 120, (n, 2)).astype(np.float32), axis=0)      # extent is [0,100]^2: some outside
    rng.shuffle(xy)
    x, y = np.ascontiguousarray(xy[:, 0]), np.ascontiguousarray(xy[:, 1])
    z = (-3000 + 0.1 * x + rng.normal(0, 1, x.size)).astype(np.float32)
    xt, yt, zt = _dev(x, y, z)
    idx = b.krige_index_create(0.0, 100.0, 0.0, 100.0, capacity=x.size)
    edges = np.linspace(0, x.size, 12).astype(int)
    for a, e in zip(edges[:-1], edges[1:]):
        b.krige_index_append(idx, xt[a:e], yt[a:e], zt[a:e])
    g = W.Geom(40, 33, -25.0, -22.0, 3.7, 4.4)                                     # nodes inside and outside the extent
    sill = W.sample_variance(z)
    got, nbr = b.krige_predict(idx, g, 1, 30.0, sill, 0.02 * sill, 12, want_nbr=True)
    idx.free()
    ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(1, 30.0, sill, 0.02 * sill), 12)
    assert np.array_equal(nbr.cpu().numpy(), ref["nbr"])
    assert max_abs_err(got.cpu().numpy(), ref["zhat"]) <= 1e-4 * depth_range(ref["zhat"])


@pytest.mark.parametrize("config,width,n_out", [(4, 250.0, 160), (5, 300.0, 120)])
def test_kriging_variance_parity(config, width, n_out):
    """sigma^2 of krige_predict_ex against the oracle's sum lambda gamma0 + mu: within 1e-4 x sill."""
    b = _bathy()
    w = W.sounding_config(config, width=width, n_target=int(width * width / 4), n_out=n_out)
    xt, yt, zt = _dev(w.x, w.y, w.z)
    idx = b.krige_build_index(xt, yt, zt)
    ill = torch.zeros(1, dtype=torch.int64, device="cuda")
    got, var = b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, want_var=True, illcond=ill)
    plain = b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k)
    idx.free()
    ref = oracle.krige_grid(w.x, w.y, w.z, ogeom(w.geom_out), oracle.vgm(w.model, w.range_, w.sill, w.nugget), w.k,
                            oracle.Buckets(w.x, w.y, 4.0), want_var=True)
    assert torch.equal(plain, got)                        # the extra outputs do not change the estimate
    assert max_abs_err(got.cpu().numpy(), ref["zhat"]) <= 1e-4 * depth_range(ref["zhat"])
    assert max_abs_err(var.cpu().numpy(), ref["var"]) <= 1e-4 * w.sill
    assert int(ill.item()) == 0                           # survey-like density: no node flagged


def test_variance_zero_at_data_and_sill_far_away():
    b = _bathy()
    xs, ys = np.meshgrid(np.arange(30, dtype=np.float32), np.arange(20, dtype=np.float32))
    rng = np.random.default_rng(3)
    z = rng.normal(-5000, 20, xs.size).astype(np.float32)
    xt, yt, zt = _dev(xs.ravel(), ys.ravel(), z)
    idx = b.krige_build_index(xt, yt, zt)
    _, var = b.krige_predict(idx, W.Geom(30, 20, 0.0, 0.0, 1.0, 1.0), 1, 6.0, 400.0, 40.0, 8, want_var=True)
    assert float(var.abs().max()) <= 1e-4 * 400.0         # every node sits on a datum
    # one far node: all neighbours beyond the spherical range of the node -> sigma^2 ~ sill + mu > sill
    _, var = b.krige_predict(idx, W.Geom(1, 1, 500.0, 500.0, 1.0, 1.0), 1, 6.0, 400.0, 40.0, 8, want_var=True)
    ref = oracle.krige_points(xs.ravel(), ys.ravel(), z, [500.0], [500.0], oracle.vgm(1, 6.0, 400.0, 40.0), 8, want_var=True)
    idx.free()
    assert abs(float(var.item()) - ref["var"][0]) <= 1e-4 * 400.0 and float(var.item()) > 400.0


@pytest.mark.parametrize("k", [4, 16, 32])
def test_gaussian_variogram_parity(k):
    b = _bathy()
    rng = np.random.default_rng(900 + k)
    n = 2500
    xy = np.unique(rng.uniform(0, 100, (n, 2)).astype(np.float32), axis=0)
    rng.shuffle(xy)
    x, y = np.ascontiguousarray(xy[:, 0]), np.ascontiguousarray(xy[:, 1])
    z = (-4000 + 3.0 * np.sin(x / 9.0) + 0.1 * y + rng.normal(0, 0.5, x.size)).astype(np.float32)
    sill = W.sample_variance(z)
    g = W.Geom(57, 41, -2.0, -1.0, 1.8, 2.5)
    v = oracle.vgm(oracle.GAUSSIAN, 4.0, sill, 0.05 * sill)
    ref = oracle.krige_grid(x, y, z, ogeom(g), v, k, want_var=True)
    xt, yt, zt = _dev(x, y, z)
    idx = b.krige_build_index(xt, yt, zt)
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    got, nbr, var = b.krige_predict(idx, g, b.GAUSSIAN, 4.0, sill, 0.05 * sill, k, want_nbr=True, want_var=True, failed=failed)
    idx.free()
    assert int(failed.item()) == 0 and ref["failed"] == 0
    assert np.array_equal(nbr.cpu().numpy(), ref["nbr"])
    assert max_abs_err(got.cpu().numpy(), ref["zhat"]) <= 1e-4 * depth_range(ref["zhat"])
    assert max_abs_err(var.cpu().numpy(), ref["var"]) <= 1e-4 * sill


def test_ill_conditioned_nodes_are_counted():
    """Reading K-cond: neighbours centimetres apart under a 30 m range and NO nugget make
    the covariance matrix nearly singular (pivots < 1e-3 of the sill) and the fp32 factorisation loses accuracy;
    the library flags such nodes through d_illcond (smallest pivot < BATHY_ILLCOND_PIVOT), and every node that
    misses the 1e-4 x range bar is among the flagged ones.  With a 5 % nugget nothing is flagged."""
    b = _bathy()
    rng = np.random.default_rng(77)
    xs = np.concatenate([rng.uniform(0, 200, 1500), 100 + rng.uniform(0, 4, 6000)])
    ys = np.concatenate([rng.uniform(0, 200, 1500), 100 + rng.uniform(0, 4, 6000)])
    xy = np.unique(np.stack([xs.astype(np.float32), ys.astype(np.float32)], 1), axis=0)
    rng.shuffle(xy)
    x, y = np.ascontiguousarray(xy[:, 0]), np.ascontiguousarray(xy[:, 1])
    z = (-4000 + 0.3 * x + rng.normal(0, 1, x.size)).astype(np.float32)
    g = W.Geom(64, 48, 70.0, 80.0, 1.0, 1.0)
    sill = W.sample_variance(z)
    ref = oracle.krige_grid(x, y, z, ogeom(g), oracle.vgm(0, 30.0, sill, 0.0), 32)
    xt, yt, zt = _dev(x, y, z)
    idx = b.krige_build_index(xt, yt, zt)
    ill = torch.zeros(1, dtype=torch.int64, device="cuda")
    got = b.krige_predict(idx, g, 0, 30.0, sill, 0.0, 32, illcond=ill)
    err = np.abs(got.cpu().numpy() - ref["zhat"])
    over = int((err > 1e-4 * depth_range(ref["zhat"])).sum())
    assert 0 < int(ill.item()) < g.n and over <= int(ill.item())
    ill.zero_()
    b.krige_predict(idx, g, 0, 30.0, sill, 0.05 * sill, 32, illcond=ill)
    idx.free()
    assert int(ill.item()) == 0


def test_catmull_rom_host_forms():
    b = _bathy()
    gw = W.grid_config(1)
    dev = b.interp_catmull_rom(torch.from_numpy(gw.z).cuda(), gw.geom_in, gw.geom_out).cpu().numpy()
    host = b.interp_catmull_rom_host(gw.z, gw.geom_in, gw.geom_out)
    assert np.array_equal(dev, host, equal_nan=True)
    hz = torch.from_numpy(gw.z).pin_memory()
    out = torch.full(gw.geom_out.shape, -1.0, dtype=torch.float32).pin_memory()
    st = torch.cuda.Stream()
    b.interp_catmull_rom_host_async(hz, gw.geom_in, gw.geom_out, out=out, stream=st)
    st.synchronize()
    assert np.array_equal(out.numpy(), dev, equal_nan=True)
    with pytest.raises(TypeError):
        b.interp_bilinear_host(gw.z, gw.geom_in, gw.geom_out, out=np.empty(gw.geom_out.shape, dtype=np.float64))


def test_two_threads_first_calls_on_distinct_streams():
    """Calls on distinct streams are thread-safe, first calls included (per-device one-time setup)."""
    b = _bathy()
    w = W.sounding_config(5, width=150.0, n_target=5600, n_out=64)
    gw = W.grid_config(3, n_in=300, factor=2, n_features=30)
    xt, yt, zt = _dev(w.x, w.y, w.z)
    gz, = _dev(gw.z)
    res, errs = {}, []

    def work(tag):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for _ in range(3):
                    idx = b.krige_build_index(xt, yt, zt, stream=st)
                    k_ = b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k, stream=st)
                    idx.free_async(stream=st)
                    s_ = b.interp_spline(gz, gw.geom_in, gw.geom_out, stream=st)
                    c_ = b.interp_catmull_rom(gz, gw.geom_in, gw.geom_out, stream=st)
                    b_ = b.interp_bilinear(gz, gw.geom_in, gw.geom_out, stream=st)
            st.synchronize()
            res[tag] = [t.cpu() for t in (k_, s_, c_, b_)]
        except Exception as e:                                # noqa: BLE001
            errs.append(e)

    ts = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errs, errs
    for a, c in zip(res[0], res[1]):
        assert torch.equal(a, c)


def test_free_right_after_a_predict_on_another_stream():
    """krige_free_index is safe right after a krige_predict that went to a stream other than the build's: the
    library notices the foreign stream and waits for the device before the index memory returns to the pool
    (with only the build stream awaited, the next stream-ordered allocation could be handed the blocks
    the running kernel still reads).  The memory is recycled at once by a second build plus a fill of the pool."""
    b = _bathy()
    w = W.sounding_config(4, width=400.0, n_target=40000, n_out=512)
    xt, yt, zt = _dev(w.x, w.y, w.z)
    args = (w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k)
    idx = b.krige_build_index(xt, yt, zt)
    want = b.krige_predict(idx, *args).clone()
    torch.cuda.synchronize()
    idx.free()
    other = torch.cuda.Stream()
    junk = (xt + 3.0e5, yt - 3.0e5, torch.full_like(zt, 123.0))   # other soundings of the same count
    for _ in range(3):
        idx = b.krige_build_index(xt, yt, zt)                  # built on the current stream ...
        other.wait_stream(torch.cuda.current_stream())
        got = torch.empty_like(want)
        b.krige_predict(idx, *args, out=got, stream=other)     # ... read on another one (a few ms of work)
        idx.free()                                             # must not let go of the memory early
        idx2 = b.krige_build_index(*junk)                      # same sizes: the pool hands the freed blocks straight back
        torch.cuda.synchronize()
        idx2.free()
        assert torch.equal(got, want)


@pytest.mark.skipif(torch.cuda.is_available() and torch.cuda.device_count() < 2, reason="needs two visible devices")
def test_index_of_another_device_is_refused():
    b = _bathy()
    w = W.sounding_config(4, width=120.0, n_target=3600, n_out=64)
    torch.cuda.set_device(0)
    idx = b.krige_build_index(*_dev(w.x, w.y, w.z))
    try:
        torch.cuda.set_device(1)
        with pytest.raises(b.BathyError) as e:
            b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k,
                            out=torch.empty((w.geom_out.ny, w.geom_out.nx), dtype=torch.float32, device="cuda:1"))
        assert e.value.status == -8                            # BATHY_ERR_INDEX, not a sticky illegal-address error
        with pytest.raises(b.BathyError):
            idx.info()
    finally:
        torch.cuda.set_device(0)
    assert idx.info()["n"] == w.x.size
    idx.free()


@pytest.mark.skipif(torch.cuda.is_available() and torch.cuda.device_count() < 2, reason="needs two visible devices")
def test_second_device_after_the_first_in_one_process():
    b = _bathy()
    gw = W.grid_config(3, n_in=700, factor=2, n_features=50)      # footprint > 48 KB of shared memory per tile
    w = W.sounding_config(4, width=120.0, n_target=3600, n_out=64)
    outs = []
    for dev in (0, 1):
        torch.cuda.set_device(dev)
        z = torch.from_numpy(gw.z).to(f"cuda:{dev}")
        xt, yt, zt = (torch.from_numpy(a).to(f"cuda:{dev}") for a in (w.x, w.y, w.z))
        idx = b.krige_build_index(xt, yt, zt)
        outs.append([t.cpu() for t in (b.interp_bilinear(z, gw.geom_in, gw.geom_out), b.interp_spline(z, gw.geom_in, gw.geom_out),
                                       b.interp_catmull_rom(z, gw.geom_in, gw.geom_out),
                                       b.krige_predict(idx, w.geom_out, w.model, w.range_, w.sill, w.nugget, w.k))])
        idx.free()
    torch.cuda.set_device(0)
    for a, c in zip(*outs):
        assert torch.equal(a, c)


def test_tma_tensor_load_probe():
    """cp.async.bulk.tensor.2d (TMA) works on the box: one 88 x 54 box load, interior and clipped by the tensor edge
    (out-of-tensor elements arrive as zeros).  The committed reproduction behind DESIGN.md's TMA paragraph: the
    load works whenever the box's first COLUMN is a multiple of 4 floats (16 bytes), rows are free; a first column
    that is not 16-byte aligned raises "illegal instruction" (profiles/r2_tma_probe.md) -- which is what round 1 hit."""
    b = _bathy()
    rng = np.random.default_rng(12)
    z = rng.normal(size=(300, 512)).astype(np.float32)
    zt = torch.from_numpy(z).cuda()
    for x0, y0 in ((0, 0), (16, 33), (124, 200), (-12, -7), (468, 281), (-88, 3)):
        got = b.probe_tma(zt, x0, y0).cpu().numpy()
        want = np.zeros((54, 88), np.float32)
        ys, xs = np.arange(y0, y0 + 54), np.arange(x0, x0 + 88)
        oky, okx = (ys >= 0) & (ys < 300), (xs >= 0) & (xs < 512)
        want[np.ix_(oky, okx)] = z[np.ix_(ys[oky], xs[okx])]
        assert np.array_equal(got, want), (x0, y0)
