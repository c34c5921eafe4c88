"""Shared helpers of the parity tests (no method arithmetic)."""
import numpy as np

import oracle


def ogeom(g):
    return oracle.geom(g.nx, g.ny, g.x0, g.y0, g.dx, g.dy)


def depth_range(ref):
    f = ref[np.isfinite(ref)]
    return float(f.max() - f.min()) if f.size else 1.0


def max_abs_err(got, ref):
    """Max |got - ref| over nodes finite in the reference; NaN patterns must agree."""
    got = np.asarray(got, dtype=np.float64)
    assert got.shape == ref.shape
    nan_ref, nan_got = np.isnan(ref), np.isnan(got)
    assert np.array_equal(nan_ref, nan_got), f"NaN pattern differs at {int((nan_ref != nan_got).sum())} nodes"
    if nan_ref.all():
        return 0.0
    return float(np.abs(got - ref)[~nan_ref].max())
