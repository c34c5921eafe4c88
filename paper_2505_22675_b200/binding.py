"""Thin Python binding of libbathy.so (include/bathy.h): argument marshalling only.

Same names as the C ABI.  torch is used for device memory and streams; every step of the path
runs in the library's CUDA kernels.  There is no CPU fallback: if the shared library is missing
or cannot be loaded, importing a symbol raises, and compute calls without a CUDA device fail
with BATHY_ERR_CUDA.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from .workloads import Geom

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbathy.so")

EXPONENTIAL, SPHERICAL, GAUSSIAN = 0, 1, 2
MAX_K = 64

SYMBOLS = ["interp_bilinear", "interp_catmull_rom", "interp_spline_workspace_bytes", "interp_spline", "krige_build_index",
           "krige_predict", "krige_free_index", "krige_free_index_async", "krige_index_info", "interp_bilinear_host",
           "interp_spline_host", "krige_host", "interp_bilinear_host_async", "interp_spline_host_async",
           "krige_host_async", "bathy_strerror", "bathy_launch_count", "bathy_set_spline_path",
           "krige_predict_ex", "krige_index_create", "krige_index_append", "interp_catmull_rom_host",
           "interp_catmull_rom_host_async", "bathy_probe_fp32", "interp_krige_window", "bathy_probe_tma",
           "interp_krige_window_noalloc", "krige_predict_aniso"]


class GridGeom(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("x0", C.c_float), ("y0", C.c_float),
                ("dx", C.c_float), ("dy", C.c_float)]


class Variogram(C.Structure):
    _fields_ = [("model", C.c_int32), ("range", C.c_float), ("sill", C.c_float), ("nugget", C.c_float)]


class KrigeOutputs(C.Structure):
    _fields_ = [("d_var", C.c_void_p), ("d_nbr", C.c_void_p), ("d_failed", C.c_void_p), ("d_illcond", C.c_void_p)]


class KrigeAniso(C.Structure):
    _fields_ = [("angle_deg", C.c_float), ("ratio", C.c_float)]


class KrigeWindow(C.Structure):
    _fields_ = [("half", C.c_int32), ("n_max", C.c_int32), ("n_min", C.c_int32)]


class BathyError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {lib().bathy_strerror(status).decode()} ({status})")


_lib = None


def lib():
    """Loads libbathy.so (build it with `python -m paper_2505_22675_b200.build`); fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build the CUDA extension first "
                              "(python -m paper_2505_22675_b200.build); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.interp_bilinear.argtypes = [vp, GridGeom, vp, GridGeom, vp]
        L.interp_catmull_rom.argtypes = [vp, GridGeom, vp, GridGeom, vp]
        L.interp_spline_workspace_bytes.argtypes = [GridGeom, GridGeom]
        L.interp_spline_workspace_bytes.restype = C.c_size_t
        L.interp_spline.argtypes = [vp, GridGeom, vp, GridGeom, vp, C.c_size_t, vp]
        L.krige_build_index.argtypes = [vp, vp, vp, C.c_int64, C.c_float, vp, C.POINTER(vp)]
        L.krige_predict.argtypes = [vp, GridGeom, Variogram, C.c_int32, vp, vp, vp, vp]
        L.krige_predict_ex.argtypes = [vp, GridGeom, Variogram, C.c_int32, vp, C.POINTER(KrigeOutputs), vp]
        L.krige_predict_aniso.argtypes = [vp, GridGeom, Variogram, KrigeAniso, C.c_int32, vp, C.POINTER(KrigeOutputs), vp]
        L.krige_index_create.argtypes = [C.c_float] * 5 + [C.c_int64, vp, C.POINTER(vp)]
        L.krige_index_append.argtypes = [vp, vp, vp, vp, C.c_int64, vp, vp]
        L.interp_krige_window.argtypes = [vp, GridGeom, KrigeWindow, Variogram, vp, vp, vp, vp]
        L.interp_krige_window_noalloc.argtypes = L.interp_krige_window.argtypes
        L.krige_free_index.argtypes = [vp]
        L.krige_free_index.restype = None
        L.krige_free_index_async.argtypes = [vp, vp]
        L.krige_free_index_async.restype = None
        L.krige_index_info.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_float),
                                       C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.interp_bilinear_host.argtypes = [vp, GridGeom, vp, GridGeom, vp]
        L.interp_spline_host.argtypes = [vp, GridGeom, vp, GridGeom, vp]
        L.krige_host.argtypes = [vp, vp, vp, C.c_int64, C.c_float, GridGeom, Variogram, C.c_int32, vp, vp, vp]
        L.interp_catmull_rom_host.argtypes = L.interp_bilinear_host.argtypes
        L.interp_catmull_rom_host_async.argtypes = L.interp_bilinear_host.argtypes
        L.interp_bilinear_host_async.argtypes = L.interp_bilinear_host.argtypes
        L.interp_spline_host_async.argtypes = L.interp_spline_host.argtypes
        L.krige_host_async.argtypes = L.krige_host.argtypes
        L.bathy_strerror.argtypes = [C.c_int]
        L.bathy_strerror.restype = C.c_char_p
        L.bathy_launch_count.restype = C.c_int64
        L.bathy_set_spline_path.argtypes = [C.c_int]
        L.bathy_probe_tma.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp]
        L.bathy_probe_fp32.argtypes = [C.c_int32, C.c_int64, C.c_int32, vp, C.POINTER(C.c_double), vp]
        _lib = L
    return _lib


def _geom(g) -> GridGeom:
    if isinstance(g, GridGeom):
        return g
    return GridGeom(int(g.nx), int(g.ny), float(g.x0), float(g.y0), float(g.dx), float(g.dy))


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _check(rc: int, where: str):
    if rc != 0:
        raise BathyError(rc, where)


def _dev_f32(t: torch.Tensor, name: str) -> torch.Tensor:
    if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous float32 CUDA tensor")
    return t


def launch_count() -> int:
    return int(lib().bathy_launch_count())


def probe_fp32(packed: bool, iters: int, ctas_per_sm: int = 2, stream=None) -> float:
    """Enqueues the FMA-chain probe (include/bathy.h) and returns the flop it retires; time it with CUDA events."""
    sink = torch.zeros(1, dtype=torch.float32, device=torch.device("cuda", torch.cuda.current_device()))
    flop = C.c_double(0.0)
    _check(lib().bathy_probe_fp32(int(bool(packed)), int(iters), int(ctas_per_sm), sink.data_ptr(), C.byref(flop),
                                  _stream(stream)), "bathy_probe_fp32")
    return float(flop.value)


def probe_tma(z: torch.Tensor, x0: int, y0: int, stream=None) -> torch.Tensor:
    """One cp.async.bulk.tensor.2d load of the 88 x 54 box at (x0, y0) of z [ny, nx] (include/bathy.h)."""
    _dev_f32(z, "z")
    out = torch.empty((54, 88), dtype=torch.float32, device=z.device)
    _check(lib().bathy_probe_tma(z.data_ptr(), int(z.shape[1]), int(z.shape[0]), int(x0), int(y0), out.data_ptr(),
                                 _stream(stream)), "bathy_probe_tma")
    return out


def set_spline_path(path: int) -> None:
    """0 = automatic, 1 = fused tile kernel only, 2 = global-solve path only (include/bathy.h)."""
    _check(lib().bathy_set_spline_path(int(path)), "bathy_set_spline_path")


def interp_bilinear(z: torch.Tensor, gin, gout, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """PAPER.md:L115-L134.  z [ny_in, nx_in] fp32 on the GPU -> [ny_out, nx_out]."""
    gi, go = _geom(gin), _geom(gout)
    _dev_f32(z, "z")
    assert z.numel() == gi.nx * gi.ny
    if out is None:
        out = torch.empty((go.ny, go.nx), dtype=torch.float32, device=z.device)
    _dev_f32(out, "out")
    assert out.numel() == go.nx * go.ny
    _check(lib().interp_bilinear(z.data_ptr(), gi, out.data_ptr(), go, _stream(stream)), "interp_bilinear")
    return out


def interp_catmull_rom(z: torch.Tensor, gin, gout, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """PAPER.md:L136-L144 (the paper's own cubic): 4x4 Catmull-Rom, bilinear fallback where one of the 16
    neighbours is missing.  z [ny_in, nx_in] fp32 on the GPU -> [ny_out, nx_out]."""
    gi, go = _geom(gin), _geom(gout)
    _dev_f32(z, "z")
    assert z.numel() == gi.nx * gi.ny
    if out is None:
        out = torch.empty((go.ny, go.nx), dtype=torch.float32, device=z.device)
    _dev_f32(out, "out")
    assert out.numel() == go.nx * go.ny
    _check(lib().interp_catmull_rom(z.data_ptr(), gi, out.data_ptr(), go, _stream(stream)), "interp_catmull_rom")
    return out


def interp_spline_workspace_bytes(gin, gout) -> int:
    return int(lib().interp_spline_workspace_bytes(_geom(gin), _geom(gout)))


def interp_spline(z: torch.Tensor, gin, gout, out: torch.Tensor | None = None,
                  workspace: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """Separable natural bicubic spline (reading D1)."""
    gi, go = _geom(gin), _geom(gout)
    _dev_f32(z, "z")
    assert z.numel() == gi.nx * gi.ny
    if out is None:
        out = torch.empty((go.ny, go.nx), dtype=torch.float32, device=z.device)
    _dev_f32(out, "out")
    assert out.numel() == go.nx * go.ny
    need = interp_spline_workspace_bytes(gi, go)
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=z.device)
        if stream is not None and hasattr(workspace, "record_stream") and hasattr(stream, "cuda_stream"):
            workspace.record_stream(stream)            # the temporary outlives this call on `stream`
    _check(lib().interp_spline(z.data_ptr(), gi, out.data_ptr(), go, workspace.data_ptr(),
                               workspace.numel() * workspace.element_size(), _stream(stream)), "interp_spline")
    return out


class KrigeIndex:
    """Owner of an opaque krige_index_t*."""

    def __init__(self, handle: int):
        self.handle = handle

    def info(self) -> dict:
        n, c, ncx, ncy = C.c_int64(), C.c_float(), C.c_int32(), C.c_int32()
        _check(lib().krige_index_info(self.handle, C.byref(n), C.byref(c), C.byref(ncx), C.byref(ncy)), "krige_index_info")
        return {"n": n.value, "cell_size": c.value, "ncx": ncx.value, "ncy": ncy.value}

    def free(self):
        if self.handle:
            lib().krige_free_index(self.handle)
            self.handle = None

    def free_async(self, stream=None):
        """Stream-ordered release (krige_free_index_async): no host synchronisation."""
        if self.handle:
            lib().krige_free_index_async(self.handle, _stream(stream))
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def krige_build_index(x: torch.Tensor, y: torch.Tensor, z: torch.Tensor, cell_size: float = 0.0,
                      stream=None) -> KrigeIndex:
    for t, nm in ((x, "x"), (y, "y"), (z, "z")):
        _dev_f32(t, nm)
    assert x.numel() == y.numel() == z.numel()
    h = C.c_void_p()
    _check(lib().krige_build_index(x.data_ptr(), y.data_ptr(), z.data_ptr(), x.numel(), float(cell_size),
                                   _stream(stream), C.byref(h)), "krige_build_index")
    return KrigeIndex(h.value)


def _counter(t, name):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.int64 and t.numel() == 1):
        raise TypeError(f"{name} must be an int64 CUDA tensor of one element")
    return t.data_ptr()


def krige_predict(index: KrigeIndex, gout, model: int, range_: float, sill: float, nugget: float, k: int,
                  out: torch.Tensor | None = None, want_nbr: bool = False, failed: torch.Tensor | None = None,
                  stream=None, want_var: bool = False, var: torch.Tensor | None = None,
                  illcond: torch.Tensor | None = None, aniso: tuple | None = None):
    """PAPER.md:L146-L171.  Returns zhat [ny, nx]; with want_nbr also nbr [ny, nx, k] int32; with want_var (or
    `var`) also the kriging variance [ny, nx] (krige_predict_ex): (zhat[, nbr][, var]).  aniso = (angle_deg, ratio):
    geometrically anisotropic variogram (krige_predict_aniso)."""
    go = _geom(gout)
    dev = torch.device("cuda", torch.cuda.current_device())
    if out is None:
        out = torch.empty((go.ny, go.nx), dtype=torch.float32, device=dev)
    _dev_f32(out, "out")
    if out.numel() != go.nx * go.ny:
        raise ValueError("out has the wrong number of elements")
    nbr = torch.empty((go.ny, go.nx, int(k)), dtype=torch.int32, device=dev) if want_nbr else None
    if var is None and want_var:
        var = torch.empty((go.ny, go.nx), dtype=torch.float32, device=dev)
    if var is not None:
        _dev_f32(var, "var")
        if var.numel() != go.nx * go.ny:
            raise ValueError("var has the wrong number of elements")
    if stream is not None and hasattr(stream, "cuda_stream"):
        for t in (nbr, var):
            if t is not None:
                t.record_stream(stream)
    vg = Variogram(int(model), float(range_), float(sill), float(nugget))
    fp, ip = _counter(failed, "failed"), _counter(illcond, "illcond")
    if aniso is not None:
        outs = KrigeOutputs(var.data_ptr() if var is not None else None, nbr.data_ptr() if nbr is not None else None, fp, ip)
        _check(lib().krige_predict_aniso(index.handle, go, vg, KrigeAniso(float(aniso[0]), float(aniso[1])), int(k),
                                         out.data_ptr(), C.byref(outs), _stream(stream)), "krige_predict_aniso")
    elif var is None and ip is None:
        _check(lib().krige_predict(index.handle, go, vg, int(k), out.data_ptr(),
                                   nbr.data_ptr() if nbr is not None else None, fp, _stream(stream)), "krige_predict")
    else:
        outs = KrigeOutputs(var.data_ptr() if var is not None else None, nbr.data_ptr() if nbr is not None else None, fp, ip)
        _check(lib().krige_predict_ex(index.handle, go, vg, int(k), out.data_ptr(), C.byref(outs), _stream(stream)),
               "krige_predict_ex")
    res = (out,) + ((nbr,) if want_nbr else ()) + ((var,) if var is not None else ())
    return res if len(res) > 1 else out


def interp_krige_window(z: torch.Tensor, geom, model: int, range_: float, sill: float, nugget: float, half: int = 2,
                        n_max: int | None = None, n_min: int = 3, out: torch.Tensor | None = None, want_how: bool = False,
                        failed: torch.Tensor | None = None, stream=None):
    """fills the NaN cells of a regular grid by ordinary kriging
    over the (2 half + 1)^2 window of grid cells, bilinear fallback below n_min valid neighbours.  Returns out
    (and how, uint8 [ny, nx], when want_how)."""
    g = _geom(geom)
    _dev_f32(z, "z")
    assert z.numel() == g.nx * g.ny
    if out is None:
        out = torch.empty((g.ny, g.nx), dtype=torch.float32, device=z.device)
    _dev_f32(out, "out")
    assert out.numel() == g.nx * g.ny and out.data_ptr() != z.data_ptr()
    how = torch.empty((g.ny, g.nx), dtype=torch.uint8, device=z.device) if want_how else None
    if n_max is None:
        n_max = (2 * int(half) + 1) ** 2 - 1
    vg = Variogram(int(model), float(range_), float(sill), float(nugget))
    _check(lib().interp_krige_window(z.data_ptr(), g, KrigeWindow(int(half), int(n_max), int(n_min)), vg, out.data_ptr(),
                                     how.data_ptr() if how is not None else None, _counter(failed, "failed"),
                                     _stream(stream)), "interp_krige_window")
    return (out, how) if want_how else out


NOALLOC_MAX_CELLS = 4194304          # BATHY_NOALLOC_MAX_CELLS of include/bathy.h


def interp_krige_window_noalloc(z: torch.Tensor, geom, model: int, range_: float, sill: float, nugget: float, half: int = 2,
                                n_max: int | None = None, n_min: int = 3, *, out: torch.Tensor, how: torch.Tensor | None = None,
                                failed: torch.Tensor | None = None, stream=None):
    """interp_krige_window for callers that may not allocate device memory while they run -- a real-time loop
    whose memory budget was handed out at start-up, or a program whose own allocator owns the GPU.  The library
    call behind it allocates nothing: its scratch is a fixed 16 MiB array inside libbathy.so's device image, one
    per GPU, shared by every call (so calls that can overlap on the GPU race -- keep them on one stream).  This
    wrapper allocates nothing either, which is why `out` (float32 [ny, nx]) is required and `how` (uint8 [ny, nx],
    optional) is passed in instead of being created here.  Grids above NOALLOC_MAX_CELLS cells raise BathyError
    (BATHY_ERR_SCRATCH).  Make the first call on each device at start-up, outside of any stream capture: it looks
    up the array's device address once.  Returns `out`."""
    g = _geom(geom)
    _dev_f32(z, "z")
    _dev_f32(out, "out")
    assert z.numel() == g.nx * g.ny and out.numel() == g.nx * g.ny and out.data_ptr() != z.data_ptr()
    if how is not None:
        assert how.is_cuda and how.dtype == torch.uint8 and how.is_contiguous() and how.numel() == g.nx * g.ny
    if n_max is None:
        n_max = (2 * int(half) + 1) ** 2 - 1
    vg = Variogram(int(model), float(range_), float(sill), float(nugget))
    _check(lib().interp_krige_window_noalloc(z.data_ptr(), g, KrigeWindow(int(half), int(n_max), int(n_min)), vg,
                                             out.data_ptr(), how.data_ptr() if how is not None else None,
                                             _counter(failed, "failed"), _stream(stream)), "interp_krige_window_noalloc")
    return out


def krige_index_create(xmin: float, xmax: float, ymin: float, ymax: float, capacity: int, cell_size: float = 0.0,
                       stream=None) -> KrigeIndex:
    """an empty, appendable index over the planned survey extent (include/bathy.h)."""
    h = C.c_void_p()
    _check(lib().krige_index_create(float(xmin), float(xmax), float(ymin), float(ymax), float(cell_size), int(capacity),
                                    _stream(stream), C.byref(h)), "krige_index_create")
    return KrigeIndex(h.value)


def krige_index_append(index: KrigeIndex, x: torch.Tensor, y: torch.Tensor, z: torch.Tensor,
                       changed: torch.Tensor | None = None, stream=None) -> None:
    """Merges a batch of soundings into an appendable index; `changed` (4 floats on the GPU) receives the
    batch's bounding box xmin, xmax, ymin, ymax."""
    for t, nm in ((x, "x"), (y, "y"), (z, "z")):
        _dev_f32(t, nm)
    assert x.numel() == y.numel() == z.numel()
    if changed is not None:
        _dev_f32(changed, "changed")
        assert changed.numel() == 4
    _check(lib().krige_index_append(index.handle, x.data_ptr(), y.data_ptr(), z.data_ptr(), x.numel(),
                                    changed.data_ptr() if changed is not None else None, _stream(stream)), "krige_index_append")


def krige_free_index(index: KrigeIndex) -> None:
    index.free()


# ---- host-buffer forms (numpy in, numpy out; copies happen inside the C call)

def _host_f32(a, name):
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous():
            raise TypeError(f"{name} must be a contiguous float32 host tensor")
        return a, a.data_ptr()
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data


def _host_out_f32(a, go):
    """A caller-supplied host OUTPUT must be written in place: contiguous float32 of the right size."""
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous() or a.numel() != go.nx * go.ny:
            raise TypeError("out must be a contiguous float32 host tensor with ny*nx elements")
        return a, a.data_ptr()
    if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags["C_CONTIGUOUS"] and a.size == go.nx * go.ny):
        raise TypeError("out must be a C-contiguous float32 numpy array with ny*nx elements")
    return a, a.ctypes.data


def interp_bilinear_host(z, gin, gout, out=None, stream=None):
    gi, go = _geom(gin), _geom(gout)
    z, zp = _host_f32(z, "z")
    if out is None:
        out = np.empty((go.ny, go.nx), dtype=np.float32)
    out, op = _host_out_f32(out, go)
    _check(lib().interp_bilinear_host(zp, gi, op, go, _stream(stream)), "interp_bilinear_host")
    return out


def interp_catmull_rom_host(z, gin, gout, out=None, stream=None):
    gi, go = _geom(gin), _geom(gout)
    z, zp = _host_f32(z, "z")
    if out is None:
        out = np.empty((go.ny, go.nx), dtype=np.float32)
    out, op = _host_out_f32(out, go)
    _check(lib().interp_catmull_rom_host(zp, gi, op, go, _stream(stream)), "interp_catmull_rom_host")
    return out


def interp_spline_host(z, gin, gout, out=None, stream=None):
    gi, go = _geom(gin), _geom(gout)
    z, zp = _host_f32(z, "z")
    if out is None:
        out = np.empty((go.ny, go.nx), dtype=np.float32)
    out, op = _host_out_f32(out, go)
    _check(lib().interp_spline_host(zp, gi, op, go, _stream(stream)), "interp_spline_host")
    return out


def _pinned_f32(a, name):
    if not isinstance(a, torch.Tensor) or a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous() or not a.is_pinned():
        raise TypeError(f"{name} must be a contiguous pinned float32 host tensor (torch.Tensor.pin_memory())")
    return a.data_ptr()


def interp_bilinear_host_async(z, gin, gout, out, stream=None):
    """Enqueue only (include/bathy.h): `out` is defined after the caller synchronises `stream`."""
    _check(lib().interp_bilinear_host_async(_pinned_f32(z, "z"), _geom(gin), _pinned_f32(out, "out"), _geom(gout),
                                            _stream(stream)), "interp_bilinear_host_async")
    return out


def interp_catmull_rom_host_async(z, gin, gout, out, stream=None):
    """Enqueue only (include/bathy.h): `out` is defined after the caller synchronises `stream`."""
    _check(lib().interp_catmull_rom_host_async(_pinned_f32(z, "z"), _geom(gin), _pinned_f32(out, "out"), _geom(gout),
                                               _stream(stream)), "interp_catmull_rom_host_async")
    return out


def interp_spline_host_async(z, gin, gout, out, stream=None):
    """Enqueue only (include/bathy.h): `out` is defined after the caller synchronises `stream`."""
    _check(lib().interp_spline_host_async(_pinned_f32(z, "z"), _geom(gin), _pinned_f32(out, "out"), _geom(gout),
                                          _stream(stream)), "interp_spline_host_async")
    return out


def krige_host_async(x, y, z, gout, model, range_, sill, nugget, k, out, failed, cell_size: float = 0.0, stream=None):
    """Enqueue only (include/bathy.h): `out` and `failed` (a pinned int64 tensor of one element) are
    defined after the caller synchronises `stream`."""
    if not isinstance(failed, torch.Tensor) or failed.dtype != torch.int64 or failed.numel() != 1 or not failed.is_pinned():
        raise TypeError("failed must be a pinned int64 host tensor of one element")
    vg = Variogram(int(model), float(range_), float(sill), float(nugget))
    _check(lib().krige_host_async(_pinned_f32(x, "x"), _pinned_f32(y, "y"), _pinned_f32(z, "z"), x.numel(), float(cell_size),
                                  _geom(gout), vg, int(k), _pinned_f32(out, "out"), failed.data_ptr(), _stream(stream)),
           "krige_host_async")
    return out, failed


def krige_host(x, y, z, gout, model, range_, sill, nugget, k, cell_size: float = 0.0, out=None, stream=None):
    go = _geom(gout)
    x, xp = _host_f32(x, "x")
    y, yp = _host_f32(y, "y")
    z, zp = _host_f32(z, "z")
    if out is None:
        out = np.empty((go.ny, go.nx), dtype=np.float32)
    out, op = _host_out_f32(out, go)
    failed = C.c_int64(0)
    vg = Variogram(int(model), float(range_), float(sill), float(nugget))
    n = x.numel() if isinstance(x, torch.Tensor) else x.shape[0]
    _check(lib().krige_host(xp, yp, zp, n, float(cell_size), go, vg, int(k), op, C.addressof(failed),
                            _stream(stream)), "krige_host")
    return out, failed.value
