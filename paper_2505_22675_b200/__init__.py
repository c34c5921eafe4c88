"""bathy-b200: B200-native (sm_100a) bilinear / natural-bicubic-spline / ordinary-kriging
interpolation of sonar soundings onto a grid -- the data-parallel hot path of arxiv 2505.22675.

Public API = the C ABI of include/bathy.h, re-exported by `binding` under the same names.
"""
from .binding import (EXPONENTIAL, SPHERICAL, GAUSSIAN, MAX_K, krige_index_create, krige_index_append, probe_fp32, probe_tma, interp_krige_window,
                      interp_krige_window_noalloc, NOALLOC_MAX_CELLS,
                      interp_catmull_rom_host, interp_catmull_rom_host_async, BathyError, KrigeIndex, interp_bilinear,  # noqa: F401
                      interp_bilinear_host, interp_bilinear_host_async, interp_catmull_rom, interp_spline, interp_spline_host,
                      interp_spline_host_async, interp_spline_workspace_bytes, krige_host_async,
                      krige_build_index, krige_free_index, krige_host, krige_predict, launch_count, lib,
                      set_spline_path)
from .workloads import Geom  # noqa: F401
