"""interp_krige_window_noalloc -- hole filling for callers that may not allocate device memory while they run.

The vehicle's mapping loop hands out its whole device-memory budget before the dive; after that a call that asks
the driver for memory can fail, and cudaMalloc / cudaFree stall every stream of the device.  The same goes for a
host program whose own allocator has reserved the GPU.  interp_krige_window takes its scratch (the hole list and
its counter) from the stream's memory pool on every call; interp_krige_window_noalloc runs the same two kernels
with that scratch in a fixed 16 MiB array inside the library's device image (include/bathy.h,
BATHY_NOALLOC_MAX_CELLS = 2048 x 2048 cells).

What is checked here, through the C ABI on a GPU:
  - the new entry point gives what the existing one gives -- the `how` map bit for bit, the same NaN pattern, the
    depths within the 1e-4 x depth range the kriging parity tests use -- on two calls in a row;
  - the second call is a different, smaller grid with fewer holes: the array still holds the first call's list
    (and its counter), so a counter that is not reset or a stale list entry being read would show up here;
  - a third call repeats the first one and must reproduce it bit for bit (the array is reused, not used up);
  - a grid over the limit is refused with BATHY_ERR_SCRATCH and nothing is written.

This file is named so that pytest collects it after every other test file: `pytest -x` stops at the first failure,
and a failure here must not hide the parity tests.  It makes no assumption about what ran before it: it passes
as the only test of a fresh process (its first call then does the once-per-device set-up) and after the rest of
the suite."""
import numpy as np
import pytest
import torch

from paper_2505_22675_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-4                                                     # x depth range: the bar of tests/test_gpu_parity_krige_window.py


def _holed(n_in, n_features, frac, seed):
    w = W.grid_config(2, n_in=n_in, factor=2, n_features=n_features)
    z = np.where(np.isnan(w.z), np.float32(-5000.0), w.z).copy()
    z[np.random.default_rng(seed).random(z.shape) < frac] = np.nan
    return z, w.geom_in


def _both_paths(b, z, g, **kw):
    """(existing path, new entry point) on the same input; outputs of the new one are pre-filled with a sentinel."""
    sill = W.sample_variance(z[~np.isnan(z)])
    zt = torch.from_numpy(z).cuda()
    f_old = torch.zeros(1, dtype=torch.int64, device="cuda")
    f_new = torch.zeros(1, dtype=torch.int64, device="cuda")
    out_old, how_old = b.interp_krige_window(zt, g, b.EXPONENTIAL, 12.0, sill, 0.0, want_how=True, failed=f_old, **kw)
    out_new = torch.full(z.shape, -7.0, dtype=torch.float32, device="cuda")
    how_new = torch.full(z.shape, 77, dtype=torch.uint8, device="cuda")
    b.interp_krige_window_noalloc(zt, g, b.EXPONENTIAL, 12.0, sill, 0.0, out=out_new, how=how_new, failed=f_new, **kw)
    torch.cuda.synchronize()
    return (out_old.cpu().numpy(), how_old.cpu().numpy(), int(f_old.item())), (out_new.cpu().numpy(), how_new.cpu().numpy(), int(f_new.item()))


def _assert_same(old, new, z):
    (o_out, o_how, o_failed), (n_out, n_how, n_failed) = old, new
    assert np.array_equal(n_how, o_how), f"{int((n_how != o_how).sum())} cells filled by a different method"
    assert n_failed == o_failed
    assert np.array_equal(np.isnan(n_out), np.isnan(o_out))
    fin = ~np.isnan(o_out)
    rng = float(o_out[fin].max() - o_out[fin].min())
    err = float(np.abs(n_out[fin].astype(np.float64) - o_out[fin].astype(np.float64)).max())
    assert err <= TOL * rng, (err, rng)
    valid = ~np.isnan(z)
    assert np.array_equal(n_out[valid], z[valid])              # valid cells are copied, the sentinel is gone everywhere
    assert (n_how[~valid] != 0).all() and (n_how[valid] == 0).all()


def test_noalloc_matches_the_allocating_path_on_two_calls_in_a_row():
    import paper_2505_22675_b200 as b
    z1, g1 = _holed(300, 60, 0.10, 901)                         # 90 000 cells, ~9 000 holes: several batches per warp, ragged tail
    z2, g2 = _holed(173, 30, 0.02, 902)                         # second call: smaller grid, ~600 holes, 7 x 7 window
    old1, new1 = _both_paths(b, z1, g1)
    _assert_same(old1, new1, z1)
    old2, new2 = _both_paths(b, z2, g2, half=3, n_min=2)
    _assert_same(old2, new2, z2)
    assert int(np.isnan(z2).sum()) < int(np.isnan(z1).sum())   # (the stale tail of call 1's list was really there to be misread)
    _, new3 = _both_paths(b, z1, g1)                            # the array is shared and reused: call 1 again, same bits
    assert np.array_equal(new3[0], new1[0], equal_nan=True) and np.array_equal(new3[1], new1[1])


def test_noalloc_refuses_a_grid_over_its_limit():
    import paper_2505_22675_b200 as b
    nx, ny = 2048, 2049                                         # one row over BATHY_NOALLOC_MAX_CELLS
    assert nx * ny > b.NOALLOC_MAX_CELLS
    z = torch.zeros((ny, nx), dtype=torch.float32, device="cuda")
    out = torch.full((ny, nx), -7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(b.BathyError) as e:
        b.interp_krige_window_noalloc(z, W.Geom(nx, ny, 0.0, 0.0, 1.0, 1.0), b.EXPONENTIAL, 12.0, 1.0, 0.0, out=out)
    assert e.value.status == -9 and "4194304" in str(e.value)   # BATHY_ERR_SCRATCH, and the message names the limit
    torch.cuda.synchronize()
    assert bool((out == -7.0).all())                            # nothing was enqueued
    ok = torch.full((2048, 2048), -7.0, dtype=torch.float32, device="cuda")   # exactly at the limit: accepted
    zin = torch.zeros((2048, 2048), dtype=torch.float32, device="cuda")
    zin[5, 7] = float("nan"); zin[2047, 2047] = float("nan")
    b.interp_krige_window_noalloc(zin, W.Geom(2048, 2048, 0.0, 0.0, 1.0, 1.0), b.EXPONENTIAL, 12.0, 1.0, 0.0, out=ok)
    torch.cuda.synchronize()
    assert float(ok[5, 7]) == 0.0 and float(ok[2047, 2047]) == 0.0 and bool((ok == 0.0).all())
