"""GPU parity, through the C ABI, of interp_bilinear and interp_spline against the float64 oracle.
Tolerance (BASELINE.json north_star): max abs error <= 1e-5 x depth range of the oracle output."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_22675_b200 import workloads as W
from _util import ogeom, depth_range, max_abs_err

pytestmark = pytest.mark.gpu
TOL = 1e-5


def _bathy():
    import paper_2505_22675_b200 as b
    return b


def _run(method, z, gi, go):
    b = _bathy()
    zt = torch.from_numpy(np.ascontiguousarray(z)).cuda()
    fn = {"bilinear": b.interp_bilinear, "spline": b.interp_spline, "catmull_rom": b.interp_catmull_rom}[method]
    out = fn(zt, gi, go)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _ref(method, z, gi, go):
    return {"bilinear": oracle.bilinear, "spline": oracle.spline, "catmull_rom": oracle.catmull_rom}[method](z, ogeom(gi), ogeom(go))


def _filled_config1():
    """Config 1 grid with its NaN cells filled by the ORACLE's kriging (isolates the method)."""
    w = W.grid_config(1)
    x, y, z = W.grid_to_scattered(w.z)
    v = oracle.vgm(oracle.SPHERICAL, 10.0, W.sample_variance(z), 0.0)
    ii, jj = np.nonzero(w.nan_mask)
    r = oracle.krige_points(x, y, z, jj.astype(np.float32), ii.astype(np.float32), v, 8)
    filled = w.z.copy()
    filled[ii, jj] = r["zhat"].astype(np.float32)
    assert not np.isnan(filled).any()
    return w, filled


@pytest.mark.parametrize("method", ["bilinear", "spline"])
def test_config1(method):
    w, filled = _filled_config1()
    ref = _ref(method, filled, w.geom_in, w.geom_out)
    got = _run(method, filled, w.geom_in, w.geom_out)
    err = max_abs_err(got, ref)
    assert err <= TOL * depth_range(ref), (err, depth_range(ref))
    if method == "bilinear":
        assert np.array_equal(got[::4, ::4], filled)            # knots bit-exact


@pytest.mark.parametrize("method", ["bilinear", "spline"])
@pytest.mark.parametrize("config,n_in,factor,nf", [(2, 257, 4, 40), (3, 600, 2, 200)])
def test_reduced_configs_2_3(method, config, n_in, factor, nf):
    # same generator, reduced size: several tiles in both directions and a ragged tail
    w = W.grid_config(config, n_in=n_in, factor=factor, n_features=nf)
    ref = _ref(method, w.z, w.geom_in, w.geom_out)
    got = _run(method, w.z, w.geom_in, w.geom_out)
    err = max_abs_err(got, ref)
    assert err <= TOL * depth_range(ref), (err, depth_range(ref))


@pytest.mark.parametrize("method", ["bilinear", "spline"])
def test_general_geometry_and_out_of_extent(method):
    rng = np.random.default_rng(21)
    z = (rng.normal(-3000, 40, (37, 53))).astype(np.float32)
    gi = W.Geom(53, 37, 10.0, -5.0, 2.0, 3.0)
    # non-integer ratio, shifted origin, nodes outside on all four sides
    go = W.Geom(301, 173, 4.0, -9.5, 0.37, 0.71)
    ref = _ref(method, z, gi, go)
    got = _run(method, z, gi, go)
    assert np.isnan(ref).any() and np.isfinite(ref).any()
    err = max_abs_err(got, ref)
    assert err <= TOL * depth_range(ref), (err, depth_range(ref))
    # down-sampling (footprint larger than a tile: gather path)
    z2 = rng.normal(-3000, 40, (400, 900)).astype(np.float32)
    gi2 = W.Geom(900, 400, 0.0, 0.0, 1.0, 1.0)
    go2 = W.Geom(40, 30, 0.5, 0.25, 22.0, 13.0)
    ref2 = _ref(method, z2, gi2, go2)
    got2 = _run(method, z2, gi2, go2)
    assert max_abs_err(got2, ref2) <= TOL * depth_range(ref2)


@pytest.mark.parametrize("method", ["bilinear", "spline"])
def test_degenerate_sizes(method):
    rng = np.random.default_rng(22)
    for (ny, nx), (oy, ox) in [((2, 2), (5, 7)), ((2, 9), (1, 33)), ((9, 2), (17, 1)), ((3, 3), (1, 1))]:
        z = rng.normal(-100, 5, (ny, nx)).astype(np.float32)
        gi = W.Geom(nx, ny, 0.0, 0.0, 1.0, 1.0)
        go = W.Geom(ox, oy, 0.0, 0.0, (nx - 1) / max(ox - 1, 1), (ny - 1) / max(oy - 1, 1))
        ref = _ref(method, z, gi, go)
        got = _run(method, z, gi, go)
        # (a single output node has depth range 0: the bar then is 1e-5 m absolute, DESIGN.md section 2 reading Tol)
        assert max_abs_err(got, ref) <= TOL * max(depth_range(ref), 1.0)


def test_bilinear_nan_propagation():
    w = W.grid_config(1)                                          # 10 % NaN cells, not filled
    ref = oracle.bilinear(w.z, ogeom(w.geom_in), ogeom(w.geom_out))
    got = _run("bilinear", w.z, w.geom_in, w.geom_out)
    assert np.isnan(ref).sum() > 0
    err = max_abs_err(got, ref)                                   # also checks the NaN pattern (B4)
    assert err <= TOL * depth_range(ref)


def test_plane_and_constant_exactness():
    # linear fields are reproduced by both methods (all second derivatives vanish)
    X, Y = np.meshgrid(np.arange(70, dtype=np.float64), np.arange(50, dtype=np.float64))
    z = (-5000 + 0.5 * X + 0.25 * Y).astype(np.float32)
    gi, go = W.Geom(70, 50, 0, 0, 1, 1), W.Geom(277, 197, 0, 0, 0.25, 0.25)
    Xo, Yo = np.meshgrid(np.arange(277) * 0.25, np.arange(197) * 0.25)
    exact = -5000 + 0.5 * Xo + 0.25 * Yo
    for method in ("bilinear", "spline"):
        got = _run(method, z, gi, go)
        assert np.abs(got - exact).max() <= 1e-3, method             # ~2 ulp at 5000 m


def test_argument_errors_and_workspace():
    b = _bathy()
    z = torch.zeros((4, 4), device="cuda")
    with pytest.raises(b.BathyError) as e:
        b.interp_bilinear(z, W.Geom(4, 4, 0, 0, 0.0, 1), W.Geom(4, 4, 0, 0, 1, 1))
    assert e.value.status == -2
    with pytest.raises(b.BathyError):
        b.interp_bilinear(torch.zeros((1, 16), device="cuda"), W.Geom(16, 1, 0, 0, 1, 1), W.Geom(4, 4, 0, 0, 1, 1))
    need = b.interp_spline_workspace_bytes(W.Geom(4, 4, 0, 0, 1, 1), W.Geom(7, 7, 0, 0, .5, .5))
    assert need > 0
    with pytest.raises(b.BathyError) as e:
        b.interp_spline(z, W.Geom(4, 4, 0, 0, 1, 1), W.Geom(7, 7, 0, 0, .5, .5),
                        workspace=torch.empty(max(need - 256, 1), dtype=torch.uint8, device="cuda"))
    assert e.value.status == -5


def test_host_forms_match_device_forms():
    b = _bathy()
    w = W.grid_config(2, n_in=129, factor=4, n_features=10)
    for method, hostfn in (("bilinear", b.interp_bilinear_host), ("spline", b.interp_spline_host)):
        dev = _run(method, w.z, w.geom_in, w.geom_out)
        host = hostfn(w.z, w.geom_in, w.geom_out)
        assert np.array_equal(dev, host)


# ---------------------------------------------------------------------------------- spline paths
# interp_spline has two implementations (include/bathy.h, bathy_set_spline_path): the fused tile
# kernel (windowed Thomas solves) and the global-solve path.

@pytest.fixture
def spline_path():
    b = _bathy()
    yield b.set_spline_path
    b.set_spline_path(0)


@pytest.mark.parametrize("path", [1, 2])
@pytest.mark.parametrize("n_in,factor", [(89, 2), (57, 4), (90, 3), (130, 2), (41, 4), (193, 1)])
def test_spline_both_paths_match_oracle(spline_path, path, n_in, factor):
    # sizes at and just above one solve window, tiles with a single cell in the last row/column
    w = W.grid_config(2, n_in=n_in, factor=factor, n_features=12, seed=500 + n_in)
    ref = _ref("spline", w.z, w.geom_in, w.geom_out)
    spline_path(path)
    got = _run("spline", w.z, w.geom_in, w.geom_out)
    err = max_abs_err(got, ref)
    assert err <= TOL * depth_range(ref), (path, err, depth_range(ref))


def test_spline_fused_rectangular_shifted_noninteger(spline_path):
    rng = np.random.default_rng(77)
    z = rng.normal(-4200, 25, (150, 260)).astype(np.float32)
    gi = W.Geom(260, 150, 100.0, -50.0, 2.0, 3.0)
    go = W.Geom(1500, 700, 95.0, -57.0, 0.353, 0.671)            # out-of-extent nodes on all four sides
    ref = _ref("spline", z, gi, go)
    assert np.isnan(ref).any()
    for path in (1, 2):
        spline_path(path)
        got = _run("spline", z, gi, go)
        assert max_abs_err(got, ref) <= TOL * depth_range(ref), path


def test_spline_fused_worst_case_data(spline_path):
    # white noise and a checkerboard: the largest second derivatives a given depth range allows,
    # i.e. the worst case of the window bound
    rng = np.random.default_rng(78)
    ii, jj = np.meshgrid(np.arange(200), np.arange(300), indexing="ij")
    for z in (rng.uniform(-6000, -5000, (200, 300)), -5500.0 + 500.0 * ((ii + jj) % 2)):
        z = z.astype(np.float32)
        gi, go = W.Geom(300, 200, 0, 0, 1, 1), W.Geom(1197, 797, 0, 0, 0.25, 0.25)
        ref = _ref("spline", z, gi, go)
        spline_path(1)
        got = _run("spline", z, gi, go)
        assert max_abs_err(got, ref) <= TOL * depth_range(ref)


@pytest.mark.parametrize("nx,ny,fy", [(100, 60, 60), (40, 40, 50), (120, 70, 45)])
def test_spline_fused_long_bands(spline_path, nx, ny, fy):
    # up-sampling factors in y so large that a warp's band of output rows is longer than its
    # shared-memory row table (it is then walked in chunks)
    rng = np.random.default_rng(79 + fy)
    yy, xx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    z = (-3000.0 + 20.0 * np.sin(xx / 3.0) * np.cos(yy / 4.0) + rng.normal(0, 1.0, (ny, nx))).astype(np.float32)
    gi = W.Geom(nx, ny, 0.0, 0.0, 1.0, 1.0)
    go = W.Geom(2 * nx + 3, (ny - 1) * fy + 7, -1.0, -3.0 / fy, 0.5, 1.0 / fy)     # a few nodes outside on each side
    ref = _ref("spline", z, gi, go)
    assert np.isnan(ref).any()
    spline_path(1)
    got = _run("spline", z, gi, go)
    assert max_abs_err(got, ref) <= TOL * depth_range(ref)


def test_spline_fused_path_refuses_what_it_cannot_serve(spline_path):
    b = _bathy()
    spline_path(1)
    z = torch.zeros((20, 20), device="cuda")
    with pytest.raises(b.BathyError):                             # smaller than a solve window
        b.interp_spline(z, W.Geom(20, 20, 0, 0, 1, 1), W.Geom(39, 39, 0, 0, .5, .5))
    spline_path(0)
    b.interp_spline(z, W.Geom(20, 20, 0, 0, 1, 1), W.Geom(39, 39, 0, 0, .5, .5))   # automatic: global path


@pytest.mark.parametrize("ny,nx", [(600, 777), (257, 1025), (513, 33), (40, 300)])
def test_spline_global_path_segments_worst_case(spline_path, ny, nx):
    """The global-solve path cuts every system into 256-knot segments solved on windows with a 32-knot halo
    (0.268^32 = 5e-19: below fp32 rounding): sizes with several ragged segments per direction, on full-amplitude
    white noise (the largest second derivatives a depth range allows), down- and up-sampling, TMA and cp.async paths."""
    rng = np.random.default_rng(1000 + nx)
    z = rng.uniform(-6000, -5000, (ny, nx)).astype(np.float32)
    gi = W.Geom(nx, ny, 0.0, 0.0, 1.0, 1.0)
    for go in (W.Geom(2 * nx - 1, 2 * ny - 1, 0.0, 0.0, 0.5, 0.5), W.Geom(nx // 2, ny // 3, 0.3, 0.7, 1.9, 2.7)):
        ref = _ref("spline", z, gi, go)
        spline_path(2)
        got = _run("spline", z, gi, go)
        assert max_abs_err(got, ref) <= TOL * depth_range(ref), (ny, nx, go)
    if nx >= 87 and ny >= 54:
        go = W.Geom(2 * nx - 1, 2 * ny - 1, 0.0, 0.0, 0.5, 0.5)
        ref = _ref("spline", z, gi, go)
        for path in (1, 3):
            spline_path(path)
            assert max_abs_err(_run("spline", z, gi, go), ref) <= TOL * depth_range(ref), path


@pytest.mark.parametrize("method", ["bilinear", "spline", "catmull_rom"])
def test_small_depth_range_at_5km(method):
    """A call whose whole depth range is ~32 m at 5 km depth: 1e-5 x range = 3.2e-4 m is 0.65 ulp of the float32
    OUTPUT (ulp(5000) = 4.9e-4 m).  The kernels compute on differences to a reference depth and add it last, so the
    only rounding at full magnitude is the final one (0.5 ulp) and the bar holds; below ~25 m of range the float32
    output format itself exceeds 1e-5 x range (reading "fp32 output")."""
    b = _bathy()
    rng = np.random.default_rng(31)
    ny, nx = 70, 131
    yy, xx = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    z = (-5000.0 + 0.17 * xx + 0.12 * yy + 3.0 * np.sin(xx / 9.0) * np.cos(yy / 7.0) + rng.normal(0, 0.3, (ny, nx))).astype(np.float32)
    gi = W.Geom(nx, ny, 0.0, 0.0, 1.0, 1.0)
    for go in (W.Geom(4 * nx - 3, 4 * ny - 3, 0.0, 0.0, 0.25, 0.25), W.Geom(300, 171, 1.3, 0.7, 0.41, 0.37)):
        ref = _ref(method, z, gi, go)
        assert 28.0 < depth_range(ref) < 42.0
        got = _run(method, z, gi, go)
        assert max_abs_err(got, ref) <= TOL * depth_range(ref), (method, depth_range(ref))
