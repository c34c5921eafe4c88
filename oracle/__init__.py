"""ctypes front end of oracle/oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this package.  It never imports paper_2505_22675_b200 and the CUDA path never imports it.
All arithmetic lives in oracle.c (float64, written from PAPER.md); this file only marshals.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (no CUDA, no third-party code)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Geom(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("x0", C.c_float), ("y0", C.c_float),
                ("dx", C.c_float), ("dy", C.c_float)]


class Vgm(C.Structure):
    _fields_ = [("model", C.c_int32), ("range", C.c_double), ("sill", C.c_double), ("nugget", C.c_double)]


class Aniso(C.Structure):
    """Geometric anisotropy of the variogram (oracle.c, oracle_aniso_lag): direction of greatest continuity in degrees
    counter-clockwise from +x, ratio = range across / range along in (0, 1]."""
    _fields_ = [("angle_deg", C.c_double), ("ratio", C.c_double)]


EXPONENTIAL, SPHERICAL, GAUSSIAN = 0, 1, 2
_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        fp, dp, ip = C.POINTER(C.c_float), C.POINTER(C.c_double), C.POINTER(C.c_int32)
        gp, vp = C.POINTER(Geom), C.POINTER(Vgm)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_num_threads.argtypes = [C.c_int]
        L.oracle_bilinear.argtypes = [fp, gp, gp, dp]
        L.oracle_spline.argtypes = [fp, gp, gp, dp]
        L.oracle_catmull_rom.argtypes = [fp, gp, gp, dp]
        L.oracle_spline1d.argtypes = [dp, C.c_int, C.c_double, dp, C.c_int, dp, dp]
        L.oracle_node_coords.argtypes = [gp, fp, fp]
        L.oracle_node_coords.restype = None
        L.oracle_knn_key.argtypes = [C.c_float] * 4
        L.oracle_knn_key.restype = C.c_float
        L.oracle_knn_brute.argtypes = [fp, fp, C.c_int64, C.c_float, C.c_float, C.c_int, ip, fp]
        L.oracle_buckets_build.argtypes = [fp, fp, C.c_int64, C.c_double]
        L.oracle_buckets_build.restype = C.c_void_p
        L.oracle_buckets_free.argtypes = [C.c_void_p]
        L.oracle_buckets_free.restype = None
        L.oracle_knn_buckets.argtypes = [C.c_void_p, fp, fp, C.c_float, C.c_float, C.c_int, ip, fp]
        L.oracle_variogram.argtypes = [vp, C.c_double]
        L.oracle_variogram.restype = C.c_double
        L.oracle_lu_solve.argtypes = [dp, dp, C.c_int, C.c_double]
        L.oracle_ok_weights.argtypes = [dp, dp, C.c_int, C.c_double, C.c_double, vp, dp, dp]
        L.oracle_krige_points.argtypes = [fp, fp, fp, C.c_int64, C.c_void_p, fp, fp, C.c_int64, vp,
                                          C.c_int, dp, ip, dp]
        L.oracle_krige_points.restype = C.c_int64
        L.oracle_krige_points_var.argtypes = [fp, fp, fp, C.c_int64, C.c_void_p, fp, fp, C.c_int64, vp,
                                              C.c_int, dp, dp, ip]
        L.oracle_krige_points_var.restype = C.c_int64
        ap = C.POINTER(Aniso)
        L.oracle_aniso_lag.argtypes = [ap, C.c_double, C.c_double]
        L.oracle_aniso_lag.restype = C.c_double
        L.oracle_ok_weights_aniso.argtypes = [dp, dp, C.c_int, C.c_double, C.c_double, vp, ap, dp, dp]
        L.oracle_krige_points_aniso.argtypes = [fp, fp, fp, C.c_int64, C.c_void_p, fp, fp, C.c_int64, vp, ap,
                                                C.c_int, dp, dp, ip, dp]
        L.oracle_krige_points_aniso.restype = C.c_int64
        L.oracle_krige_window.argtypes = [fp, gp, C.c_int, C.c_int, C.c_int, vp, dp, C.POINTER(C.c_uint8)]
        L.oracle_krige_window.restype = C.c_int64
        _lib = L
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def geom(nx, ny, x0, y0, dx, dy) -> Geom:
    return Geom(int(nx), int(ny), float(x0), float(y0), float(dx), float(dy))


def vgm(model, range_, sill, nugget) -> Vgm:
    return Vgm(int(model), float(range_), float(sill), float(nugget))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def bilinear(z, gi: Geom, go: Geom) -> np.ndarray:
    """PAPER.md:L132.  z fp32 [ny_in, nx_in] -> float64 [ny_out, nx_out]."""
    z = _f32(z)
    assert z.shape == (gi.ny, gi.nx)
    out = np.empty((go.ny, go.nx), dtype=np.float64)
    rc = lib().oracle_bilinear(_p(z, C.c_float), C.byref(gi), C.byref(go), _p(out, C.c_double))
    if rc:
        raise ValueError(f"oracle_bilinear: {rc}")
    return out


def catmull_rom(z, gi: Geom, go: Geom) -> np.ndarray:
    """4x4 Catmull-Rom cubic, x on 4 rows then y; bilinear fallback when one of the 16
    neighbours is outside the grid or NaN."""
    z = _f32(z)
    assert z.shape == (gi.ny, gi.nx)
    out = np.empty((go.ny, go.nx), dtype=np.float64)
    rc = lib().oracle_catmull_rom(_p(z, C.c_float), C.byref(gi), C.byref(go), _p(out, C.c_double))
    if rc:
        raise ValueError(f"oracle_catmull_rom: {rc}")
    return out


def spline(z, gi: Geom, go: Geom) -> np.ndarray:
    """Separable natural bicubic spline (reading D1/S1-S3)."""
    z = _f32(z)
    assert z.shape == (gi.ny, gi.nx)
    out = np.empty((go.ny, go.nx), dtype=np.float64)
    rc = lib().oracle_spline(_p(z, C.c_float), C.byref(gi), C.byref(go), _p(out, C.c_double))
    if rc:
        raise ValueError(f"oracle_spline: {rc}")
    return out


def spline1d(z, h, u):
    """Natural cubic spline through knots 0,h,2h,.. with values z, evaluated at u (knot units).
    Returns (values, M)."""
    z, u = _f64(z), _f64(np.atleast_1d(u))
    out, M = np.empty(u.shape[0]), np.empty(z.shape[0])
    rc = lib().oracle_spline1d(_p(z, C.c_double), z.shape[0], float(h), _p(u, C.c_double), u.shape[0],
                               _p(out, C.c_double), _p(M, C.c_double))
    if rc:
        raise ValueError(f"oracle_spline1d: {rc}")
    return out, M


def node_coords(g: Geom):
    """K1: fp32 node coordinates fmaf(J, dx, x0), fmaf(I, dy, y0), each [ny, nx]."""
    xq = np.empty((g.ny, g.nx), dtype=np.float32)
    yq = np.empty((g.ny, g.nx), dtype=np.float32)
    lib().oracle_node_coords(C.byref(g), _p(xq, C.c_float), _p(yq, C.c_float))
    return xq, yq


def knn_key(xq, yq, xi, yi) -> float:
    return float(lib().oracle_knn_key(float(xq), float(yq), float(xi), float(yi)))


class Buckets:
    """Independent float64 bucket grid used to search large sounding sets (validated against
    brute force in tests/test_oracle_kriging.py)."""

    def __init__(self, x, y, cell: float):
        self.x, self.y = _f32(x), _f32(y)
        self.h = lib().oracle_buckets_build(_p(self.x, C.c_float), _p(self.y, C.c_float),
                                            self.x.shape[0], float(cell))
        if not self.h:
            raise ValueError("oracle_buckets_build failed")

    def __del__(self):
        try:
            if getattr(self, "h", None):
                lib().oracle_buckets_free(self.h)
                self.h = None
        except Exception:          # interpreter shutdown
            pass


def knn(x, y, xq, yq, k, buckets: Buckets | None = None):
    """K2: indices (ascending (key, index)) and fp32 keys of the k nearest soundings."""
    x, y = _f32(x), _f32(y)
    idx = np.empty(k, dtype=np.int32)
    key = np.empty(k, dtype=np.float32)
    if buckets is None:
        rc = lib().oracle_knn_brute(_p(x, C.c_float), _p(y, C.c_float), x.shape[0], float(xq), float(yq),
                                    int(k), _p(idx, C.c_int32), _p(key, C.c_float))
    else:
        rc = lib().oracle_knn_buckets(buckets.h, _p(x, C.c_float), _p(y, C.c_float), float(xq), float(yq),
                                      int(k), _p(idx, C.c_int32), _p(key, C.c_float))
    if rc:
        raise ValueError(f"oracle_knn: {rc}")
    return idx, key


def variogram(v: Vgm, h) -> np.ndarray:
    h = np.atleast_1d(np.asarray(h, dtype=np.float64))
    return np.array([lib().oracle_variogram(C.byref(v), float(t)) for t in h])


def lu_solve(A, b):
    A, b = _f64(A).copy(), _f64(b).copy()
    rc = lib().oracle_lu_solve(_p(A, C.c_double), _p(b, C.c_double), b.shape[0], 0.0)
    if rc:
        raise ValueError("singular")
    return b


def aniso(angle_deg: float, ratio: float) -> Aniso:
    return Aniso(float(angle_deg), float(ratio))


def aniso_lag(a: Aniso | None, dx: float, dy: float) -> float:
    return float(lib().oracle_aniso_lag(C.byref(a) if a is not None else None, float(dx), float(dy)))


def ok_weights(px, py, xq, yq, v: Vgm, a: Aniso | None = None):
    """K4: (lambda[k], mu) of the gamma-form ordinary-kriging system, dense LU (a: anisotropic lags, NEXT-4)."""
    px, py = _f64(px), _f64(py)
    k = px.shape[0]
    lam = np.empty(k)
    mu = C.c_double(0.0)
    if a is not None:
        rc = lib().oracle_ok_weights_aniso(_p(px, C.c_double), _p(py, C.c_double), k, float(xq), float(yq),
                                           C.byref(v), C.byref(a), _p(lam, C.c_double), C.byref(mu))
    else:
        rc = lib().oracle_ok_weights(_p(px, C.c_double), _p(py, C.c_double), k, float(xq), float(yq),
                                     C.byref(v), _p(lam, C.c_double), C.byref(mu))
    if rc:
        raise ValueError("singular kriging system")
    return lam, mu.value


def krige_points(x, y, z, xq, yq, v: Vgm, k: int, buckets: Buckets | None = None,
                 want_nbr: bool = True, want_lambda: bool = False, want_var: bool = False, a: Aniso | None = None):
    """K1-K5 at fp32 query points.  Returns dict(zhat float64 [nq], nbr int32 [nq,k], lam, failed[, var]).
    a: geometric anisotropy of the variogram (NEXT-4; neighbours stay the k nearest by plain distance)."""
    if a is not None:
        return _krige_points_aniso(x, y, z, xq, yq, v, a, k, buckets, want_nbr, want_lambda)
    if want_var:
        return _krige_points_var(x, y, z, xq, yq, v, k, buckets, want_nbr)
    x, y, z = _f32(x), _f32(y), _f32(z)
    xq, yq = _f32(np.ravel(xq)), _f32(np.ravel(yq))
    nq = xq.shape[0]
    zhat = np.empty(nq, dtype=np.float64)
    nbr = np.empty((nq, k), dtype=np.int32) if want_nbr else None
    lam = np.empty((nq, k), dtype=np.float64) if want_lambda else None
    failed = lib().oracle_krige_points(
        _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float), x.shape[0],
        buckets.h if buckets is not None else None,
        _p(xq, C.c_float), _p(yq, C.c_float), nq, C.byref(v), int(k),
        _p(zhat, C.c_double), _p(nbr, C.c_int32) if want_nbr else None,
        _p(lam, C.c_double) if want_lambda else None)
    if failed < 0:
        raise ValueError(f"oracle_krige_points: {failed}")
    return {"zhat": zhat, "nbr": nbr, "lam": lam, "failed": int(failed)}


def _krige_points_aniso(x, y, z, xq, yq, v, a, k, buckets, want_nbr, want_lambda):
    x, y, z = _f32(x), _f32(y), _f32(z)
    xq, yq = _f32(np.ravel(xq)), _f32(np.ravel(yq))
    nq = xq.shape[0]
    zhat, var = np.empty(nq, dtype=np.float64), np.empty(nq, dtype=np.float64)
    nbr = np.empty((nq, k), dtype=np.int32) if want_nbr else None
    lam = np.empty((nq, k), dtype=np.float64) if want_lambda else None
    failed = lib().oracle_krige_points_aniso(
        _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float), x.shape[0],
        buckets.h if buckets is not None else None,
        _p(xq, C.c_float), _p(yq, C.c_float), nq, C.byref(v), C.byref(a), int(k),
        _p(zhat, C.c_double), _p(var, C.c_double), _p(nbr, C.c_int32) if want_nbr else None,
        _p(lam, C.c_double) if want_lambda else None)
    if failed < 0:
        raise ValueError(f"oracle_krige_points_aniso: {failed}")
    return {"zhat": zhat, "var": var, "nbr": nbr, "lam": lam, "failed": int(failed)}


def _krige_points_var(x, y, z, xq, yq, v, k, buckets, want_nbr):
    x, y, z = _f32(x), _f32(y), _f32(z)
    xq, yq = _f32(np.ravel(xq)), _f32(np.ravel(yq))
    nq = xq.shape[0]
    zhat = np.empty(nq, dtype=np.float64)
    var = np.empty(nq, dtype=np.float64)
    nbr = np.empty((nq, k), dtype=np.int32) if want_nbr else None
    failed = lib().oracle_krige_points_var(
        _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float), x.shape[0],
        buckets.h if buckets is not None else None,
        _p(xq, C.c_float), _p(yq, C.c_float), nq, C.byref(v), int(k),
        _p(zhat, C.c_double), _p(var, C.c_double), _p(nbr, C.c_int32) if want_nbr else None)
    if failed < 0:
        raise ValueError(f"oracle_krige_points_var: {failed}")
    return {"zhat": zhat, "var": var, "nbr": nbr, "lam": None, "failed": int(failed)}


def krige_grid(x, y, z, g: Geom, v: Vgm, k: int, buckets: Buckets | None = None, **kw):
    """Kriging onto every node of grid g (node coordinates per K1)."""
    xq, yq = node_coords(g)
    r = krige_points(x, y, z, xq, yq, v, k, buckets, **kw)
    r["zhat"] = r["zhat"].reshape(g.ny, g.nx)
    if r.get("var") is not None:
        r["var"] = r["var"].reshape(g.ny, g.nx)
    if r["nbr"] is not None:
        r["nbr"] = r["nbr"].reshape(g.ny, g.nx, k)
    return r


def krige_window(z, g: Geom, v: Vgm, half: int = 2, n_max: int | None = None, n_min: int = 3):
    """NEXT-2: holes (NaN) of a regular grid filled by ordinary kriging from the valid
    cells of the (2 half + 1)^2 window, bilinear fallback below n_min neighbours.  Returns dict(out float64 [ny, nx],
    how uint8 [ny, nx], failed)."""
    z = _f32(z)
    assert z.shape == (g.ny, g.nx)
    if n_max is None:
        n_max = (2 * half + 1) ** 2 - 1
    out = np.empty((g.ny, g.nx), dtype=np.float64)
    how = np.empty((g.ny, g.nx), dtype=np.uint8)
    failed = lib().oracle_krige_window(_p(z, C.c_float), C.byref(g), int(half), int(n_max), int(n_min), C.byref(v),
                                       _p(out, C.c_double), _p(how, C.c_uint8))
    if failed < 0:
        raise ValueError(f"oracle_krige_window: {failed}")
    return {"out": out, "how": how, "failed": int(failed)}
