#!/usr/bin/env python
"""bench.py -- output nodes/s of the hot path (bilinear, natural bicubic spline, ordinary kriging)
on B200, with the roofline of the dominant kernel and the oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A STEP is one pass of the whole hot path (every row of SURVEY.md 8(a)) over one batch of seeded
synthetic input:
    interp_bilinear   config 3   4096^2 -> 8191^2 fp32                       (B1)
    interp_spline     config 3   4096^2 -> 8191^2 fp32                       (S1-S4)
    krige_build_index config 4   ~1.0 M multibeam soundings                   (K1)
    krige_predict     config 4   -> 2048^2 nodes, k=32, exponential a=50 m    (K2-K5)
`value` = output nodes of all three methods per second of device time, inputs resident in HBM.
`methods` gives, for EVERY BASELINE.json config (1-5) and method, nodes/s (median and best of >= 20
separately timed repetitions) and the roofline fraction against both denominators SURVEY.md 8(d)
names (measured copy bandwidth and nominal 8 TB/s; measured and derived FP32 peak); configs 1-2 fit
in L2 and are reported warm and cold (L2 flushed before each repetition); config 5 goes through its
64 tile calls and reports total time, per-tile latency p50/max and the index build separately.
`roofline` is the one of the kernel that takes most of the step.
`e2e` is the same step through the C ABI's host-buffer entry points (pinned host memory, the
host<->device copies inside the timed region).
`--workload small|config2|config5` runs the step on other configs; `--no-extras` skips the
per-config table, the FP32 probe and e2e (short runs under ncu).

N > 1 (torchrun): every rank runs the same step on its own batch (seed + rank): the path shards
by batch with no data-path collective ("weak").  Time = max over ranks.

`--impl reference` times the float64 CPU oracle (oracle/, as it stands) on a bounded sample of the
same workload -- this tier has no reference implementation to install.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "output nodes/s (bilinear + natural bicubic spline + ordinary kriging, one pass of the hot path)"
UNIT = "nodes/s"
FP32_LANES_PER_SM, SMS = 128, 148          # guide: 4 SMSP x 32 FP32 lanes, 148 SMs


def krige_flops(k: int) -> float:
    """Algorithmic flop per kriging node: Cholesky k^3/3,
    two right-hand sides forward+back 4k^2, covariances 10 flop-equivalents for each of the
    k(k+1)/2 pairs, 10k for c0 and the estimate."""
    return k ** 3 / 3.0 + 4.0 * k * k + 5.0 * k * (k + 1) + 10.0 * k


WORKLOADS = {
    # name: (grid config, n_in, factor, features | kriging config, width, n_target, n_out)
    "default": dict(grid=(3, 4096, 2, 8000), krige=(4, 2000.0, 1_000_000, 2048), tiles=False,
                    label="config3(bilinear+spline 4096^2->8191^2) + config4(kriging 1.0M soundings->2048^2, k=32 exponential)"),
    "config2": dict(grid=(2, 1024, 4, 500), krige=(4, 2000.0, 1_000_000, 2048), tiles=False,
                    label="config2(bilinear+spline 1024^2->4093^2) + config4(kriging)"),
    "config5": dict(grid=(3, 4096, 2, 8000), krige=(5, 4000.0, 4_000_000, 4096), tiles=True,
                    label="config3(bilinear+spline) + config5(kriging 4.0M soundings->4096^2 as 64 tiles of 512^2, k=64 spherical)"),
    "small5": dict(grid=(2, 257, 4, 40), krige=(5, 300.0, 22500, 128), tiles=True,
                   label="reduced configs (257^2->1025^2; 22.5k soundings->128^2 as 64 tiles, k=64 spherical)"),
    "small": dict(grid=(2, 257, 4, 40), krige=(4, 250.0, 15625, 200), tiles=False,
                  label="reduced configs (257^2->1025^2; 15.6k soundings->200^2, k=32)"),
}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [c.strip() for c in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ inputs

def make_inputs(name: str, rank: int):
    from paper_2505_22675_b200 import workloads as W
    spec = WORKLOADS[name]
    gc, n_in, factor, nf = spec["grid"]
    kc, width, n_target, n_out = spec["krige"]
    from paper_2505_22675_b200 import sharding as S
    gw = W.grid_config(gc, n_in=n_in, factor=factor, n_features=nf, seed=S.rank_seed(W.SEEDS[gc], rank))
    sw = W.sounding_config(kc, width=width, n_target=n_target, n_out=n_out, seed=S.rank_seed(W.SEEDS[kc], rank))
    if spec["tiles"]:
        tiles = W.boustrophedon_tiles(n_out, max(n_out // 8, 1))
    else:
        tiles = [(0, 0, n_out, n_out)]
    return gw, sw, tiles


# ------------------------------------------------------------------------------------------ our arm

NOMINAL_HBM_GBS = 8000.0                               # the ~8 TB/s north_star names (context denominator)


def time_reps(fn, reps, stream, before=None, inner=1):
    """Median / best / mean of `reps` separately timed repetitions of fn() (CUDA events on the launching
    stream); `before()` runs outside the timed bracket of every repetition (L2 flush).  inner > 1: a repetition
    is `inner` back-to-back calls and the time is per call (the ~3 us an event pair adds to a 60 us kernel is
    shared by the calls); only used where one call's data exceeds the L2, so that no call finds the previous
    one's lines."""
    import torch
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for e0, e1 in evs:
        if before:
            before()
        e0.record(stream)
        for _ in range(inner):
            fn()
        e1.record(stream)
    torch.cuda.synchronize()
    ms = sorted(e0.elapsed_time(e1) / inner for e0, e1 in evs)
    return {"ms_median": ms[len(ms) // 2], "ms_best": ms[0], "ms_mean": float(np.mean(ms)), "reps": reps, "calls_per_rep": inner}


def hbm_roof(t, grid_bytes, n_nodes, peaks):
    sec = t["ms_median"] * 1e-3
    ach = grid_bytes / sec / 1e9
    return {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
            "frac_of_nominal_8TBps": ach / NOMINAL_HBM_GBS, "frac_best": grid_bytes / (t["ms_best"] * 1e-3) / 1e9 / peaks["hbm_gbs"],
            "bytes_per_node": grid_bytes / n_nodes}


def alu_roof(ms, k, n_nodes, fp32):
    ach = krige_flops(k) * n_nodes / (ms * 1e-3) / 1e12
    return {"bound": "alu", "achieved": ach, "peak": fp32["derived"], "unit": "TFLOP/s", "frac": ach / fp32["derived"],
            "peak_measured": fp32.get("measured"), "frac_of_measured": (ach / fp32["measured"]) if fp32.get("measured") else None,
            "flop_per_node": krige_flops(k)}


def measure_link(h_in, h_out, dev, reps=3):
    """Bare pinned-memory copy rates of this process on this box (cudaMemcpyAsync through torch's copy_, CUDA
    events): host->device of the step's grid input, device->host of one grid result, and both at once on two
    streams (the link is full duplex).  These make `e2e` self-explaining: a slow box shows up here, not as a
    mystery in ms_per_step."""
    import torch
    d_in = torch.empty(h_in.shape, dtype=h_in.dtype, device=dev)
    d_out = torch.empty(h_out.shape, dtype=h_out.dtype, device=dev)
    s1, s2 = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    nb_in, nb_out = h_in.numel() * h_in.element_size(), h_out.numel() * h_out.element_size()

    def timed(fn):
        best = float("inf")
        for _ in range(reps + 1):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            fn()
            torch.cuda.synchronize()
            best = min(best, time.perf_counter() - t0)
        return best

    def h2d():
        with torch.cuda.stream(s1):
            d_in.copy_(h_in, non_blocking=True)

    def d2h():
        with torch.cuda.stream(s2):
            h_out.copy_(d_out, non_blocking=True)
    t_h2d, t_d2h, t_both = timed(h2d), timed(d2h), timed(lambda: (h2d(), d2h()))
    return {"h2d_gbs": nb_in / t_h2d / 1e9, "d2h_gbs": nb_out / t_d2h / 1e9,
            "duplex_gbs": (nb_in + nb_out) / t_both / 1e9, "h2d_probe_bytes": nb_in, "d2h_probe_bytes": nb_out,
            "pinned": bool(h_in.is_pinned() and h_out.is_pinned())}


def measure_fp32_peak(B, stream, reps=5):
    """FMA-chain microbenchmark of the library (bathy_probe_fp32): TFLOP/s of scalar FFMA and packed FFMA2."""
    import torch
    out = {}
    for name, packed in (("ffma", False), ("ffma2", True)):
        best = 0.0
        B.probe_fp32(packed, 20000, 2)
        torch.cuda.synchronize()
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            flop = B.probe_fp32(packed, 200000, 2)
            e1.record(stream)
            torch.cuda.synchronize()
            best = max(best, flop / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        out[name] = best
    return out


def grid_methods(B, gw, reps, stream, peaks, flush=None, with_cr=True, z_dev=None):
    """bilinear / spline / Catmull-Rom of one gridded config: warm (back to back) and, if `flush` is given,
    cold (L2 flushed before every repetition)."""
    import torch
    gi, go = gw.geom_in, gw.geom_out
    z = z_dev if z_dev is not None else torch.from_numpy(gw.z).cuda()
    out = torch.empty(go.shape, dtype=torch.float32, device="cuda")
    ws = torch.empty(B.interp_spline_workspace_bytes(gi, go), dtype=torch.uint8, device="cuda")
    grid_bytes = 4.0 * (gi.n + go.n)
    fns = {"bilinear": lambda: B.interp_bilinear(z, gi, go, out=out),
           "spline": lambda: B.interp_spline(z, gi, go, out=out, workspace=ws)}
    if with_cr:
        fns["catmull_rom"] = lambda: B.interp_catmull_rom(z, gi, go, out=out)
    res = {}
    for name, fn in fns.items():
        for _ in range(3):
            fn()
        t = time_reps(fn, reps, stream, inner=4 if (flush is None and grid_bytes > 2.0e8) else 1)
        e = {"nodes": go.n, "nodes_per_s": go.n / (t["ms_median"] * 1e-3), "nodes_per_s_best": go.n / (t["ms_best"] * 1e-3), **t,
             "roofline": hbm_roof(t, grid_bytes, go.n, peaks)}
        if flush is not None:
            tc = time_reps(fn, reps, stream, before=flush)
            e["cold_l2"] = {"nodes_per_s": go.n / (tc["ms_median"] * 1e-3), **tc, "roofline": hbm_roof(tc, grid_bytes, go.n, peaks)}
            e["l2"] = "fits in the 126 MB L2: top-level numbers are warm-L2 (back to back), cold_l2 = L2 flushed (512 MB written) before every repetition"
        else:
            e["l2"] = "%.0f MB per call exceed the 126 MB L2: no flush needed" % (grid_bytes / 1e6)
        res[name] = e
    return res


def krige_methods(B, sw, tiles, reps, stream, fp32, flush=None):
    """krige_build_index and krige_predict of one sounding config (one call, or the tile calls in arrival order)."""
    import torch
    from paper_2505_22675_b200 import workloads as W
    gk = sw.geom_out
    sx, sy, sz = (torch.from_numpy(a).cuda() for a in (sw.x, sw.y, sw.z))
    failed = torch.zeros(1, dtype=torch.int64, device="cuda")
    res = {}
    hold = []

    def build():
        hold.append(B.krige_build_index(sx, sy, sz))

    def release():
        while hold:
            hold.pop().free_async()
    for _ in range(3):
        build(); release()
    tb = time_reps(lambda: (build(), release()), reps, stream, before=flush)
    res["krige_build_index"] = {"soundings": int(sw.x.shape[0]), "soundings_per_s": sw.x.shape[0] / (tb["ms_median"] * 1e-3), **tb,
                                "note": "one-off per survey; not part of nodes/s"}
    idx = B.krige_build_index(sx, sy, sz)
    if tiles is None:
        out = torch.empty(gk.shape, dtype=torch.float32, device="cuda")
        fn = lambda: B.krige_predict(idx, gk, sw.model, sw.range_, sw.sill, sw.nugget, sw.k, out=out, failed=failed)
        n_calls = 1
    else:
        tg = [W.tile_geom(gk, i0, j0, ny, nx) for (i0, j0, ny, nx) in tiles]
        bufs = [torch.empty((t.ny, t.nx), dtype=torch.float32, device="cuda") for t in tg]

        def fn():
            for t, bf in zip(tg, bufs):
                B.krige_predict(idx, t, sw.model, sw.range_, sw.sill, sw.nugget, sw.k, out=bf, failed=failed)
        n_calls = len(tg)
    for _ in range(3):
        fn()
    t = time_reps(fn, reps, stream, before=flush if tiles is None else None)
    e = {"nodes": gk.n, "k": sw.k, "launches": n_calls, "nodes_per_s": gk.n / (t["ms_median"] * 1e-3),
         "nodes_per_s_best": gk.n / (t["ms_best"] * 1e-3), **t, "roofline": alu_roof(t["ms_median"], sw.k, gk.n, fp32)}
    if tiles is not None:                                   # per-tile latency: events around every tile call of one pass
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(n_calls + 1)]
        evs[0].record(stream)
        for i, (tgi, bf) in enumerate(zip(tg, bufs)):
            B.krige_predict(idx, tgi, sw.model, sw.range_, sw.sill, sw.nugget, sw.k, out=bf, failed=failed)
            evs[i + 1].record(stream)
        torch.cuda.synchronize()
        lat = sorted(evs[i].elapsed_time(evs[i + 1]) for i in range(n_calls))
        e["tiles"] = {"count": n_calls, "tile_nodes": tg[0].nx * tg[0].ny, "ms_total_first_launch_to_last_completion": float(evs[0].elapsed_time(evs[-1])),
                      "ms_tile_p50": lat[len(lat) // 2], "ms_tile_max": lat[-1], "ms_tile_min": lat[0]}
    idx.free()
    assert int(failed.item()) == 0, "kriging reported failed nodes on a bench workload"
    res["kriging"] = e
    return res


def append_costs(B, sw, reps, stream):
    """Streaming index (krige_index_create / krige_index_append): ms per append against batch size, into an index
    that already holds the rest of the survey, with a caller's cell size and room for 8 M soundings -- the case
    where the cell arrays are sized for the capacity (4 cells per sounding) but the grid in use is small."""
    import torch
    n = int(sw.x.shape[0])
    sx, sy, sz = (torch.from_numpy(a).cuda() for a in (sw.x, sw.y, sw.z))
    ext = (float(sw.x.min()), float(sw.x.max()), float(sw.y.min()), float(sw.y.max()))
    res = {"capacity": 8_000_000, "cell_size_m": 6.0, "held_before_append": None, "by_batch": {}}
    for batch in (1_000, 10_000, 100_000):
        held = n - batch
        idx = B.krige_index_create(*ext, capacity=8_000_000, cell_size=6.0)
        B.krige_index_append(idx, sx[:held], sy[:held], sz[:held])
        torch.cuda.synchronize()
        ms = []
        for _ in range(max(3, min(reps, 10))):             # each repetition appends the same batch to a fresh copy of the state
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            B.krige_index_append(idx, sx[held:], sy[held:], sz[held:])
            e1.record(stream)
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
            idx.free()
            idx = B.krige_index_create(*ext, capacity=8_000_000, cell_size=6.0)
            B.krige_index_append(idx, sx[:held], sy[:held], sz[:held])
            torch.cuda.synchronize()
        idx.free()
        res["by_batch"][str(batch)] = {"ms_median": statistics.median(ms), "ms_best": min(ms), "held": held}
    res["note"] = "an append re-merges the sorted arrays: cost ~ batch + cells in use + soundings held, independent of the capacity"
    return res


_WORKLOAD_CACHE = {}


def cached_workload(kind, config):
    """Full-size BASELINE.json workloads are generated once per process (config 5 takes several seconds)."""
    from paper_2505_22675_b200 import workloads as W
    key = (kind, config)
    if key not in _WORKLOAD_CACHE:
        _WORKLOAD_CACHE[key] = W.grid_config(config) if kind == "grid" else W.sounding_config(config)
    return _WORKLOAD_CACHE[key]


def per_config_table(B, stream, peaks, fp32, reps):
    """Every BASELINE.json config through the same entry points: {config: {method: numbers}}."""
    import torch
    from paper_2505_22675_b200 import workloads as W
    flush_buf = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    flush = lambda: flush_buf.fill_(1)
    table = {}
    # config 1: kriging (k = 8, spherical) on the valid cells -> 253^2, fill, bilinear + spline on the filled grid
    w1 = W.grid_config(1)
    x, y, z = W.grid_to_scattered(w1.z)
    sill = W.sample_variance(z)
    sw1 = W.SoundingWorkload(1, x, y, z, w1.geom_out, 8, B.SPHERICAL, 10.0, sill, 0.0)
    t1 = krige_methods(B, sw1, None, reps, stream, fp32, flush=None)
    xt, yt, zt = (torch.from_numpy(a).cuda() for a in (x, y, z))
    idx = B.krige_build_index(xt, yt, zt)
    fill = B.krige_predict(idx, w1.geom_in, B.SPHERICAL, 10.0, sill, 0.0, 8)
    idx.free()
    filled = torch.where(torch.from_numpy(w1.nan_mask).cuda(), fill, torch.from_numpy(w1.z).cuda()).contiguous()
    t1.update(grid_methods(B, w1, reps, stream, peaks, flush=flush, z_dev=filled))
    t1["catmull_rom"]["note"] = "on the kriging-filled grid (as bilinear and spline)"
    table["config1"] = t1
    # config 2 (L2-resident: warm and cold), config 3 (HBM regime)
    table["config2"] = grid_methods(B, cached_workload("grid", 2), reps, stream, peaks, flush=flush)
    w3 = cached_workload("grid", 3)
    table["config3"] = grid_methods(B, w3, reps, stream, peaks)
    # NEXT-2: the paper's Grid B workload at scale -- config-3 grid, 5 % of the cells removed at
    # random, filled by 5 x 5 grid-window ordinary kriging
    zh = w3.z.copy()
    zh[np.random.default_rng(4096).random(zh.shape) < 0.05] = np.nan
    n_holes = int(np.isnan(zh).sum())
    zt = torch.from_numpy(zh).cuda()
    oh = torch.empty_like(zt)
    sill = float(np.nanvar(zh[::16, ::16]))
    fn = lambda: B.interp_krige_window(zt, w3.geom_in, B.EXPONENTIAL, 12.0, sill, 0.0, half=2, out=oh)
    for _ in range(3):
        fn()
    tw = time_reps(fn, reps, stream)
    table["gridB_4096_5pct_holes"] = {"krige_window": {
        "nodes": n_holes, "grid_cells": int(zh.size), "holes_per_s": n_holes / (tw["ms_median"] * 1e-3), **tw,
        "roofline": alu_roof(tw["ms_median"], 24, n_holes, fp32),
        "note": "whole call (hole scan + persistent solve kernel); flop = the k = 24 system of a full 5 x 5 window per hole; "
                "the scan alone moves %.0f MB (read + write of the grid)" % (8.0 * zh.size / 1e6)}}
    del zt, oh
    torch.cuda.empty_cache()
    # config 4 (one call), config 5 (64 tile calls in arrival order)
    table["config4"] = krige_methods(B, cached_workload("soundings", 4), None, reps, stream, fp32, flush=flush)
    table["config4"]["krige_index_append"] = append_costs(B, cached_workload("soundings", 4), reps, stream)
    w5 = cached_workload("soundings", 5)
    table["config5"] = krige_methods(B, w5, w5.tiles, reps, stream, fp32)
    del flush_buf
    return table


def run_survey_sharded(args):
    """--shard survey: ONE config-5 survey split over the ranks -- the soundings of
    rank 0 are replicated by one NCCL broadcast, every rank builds the same index and predicts the output tiles it
    owns (round-robin in arrival order); no other collective.  Strong scaling: value = all nodes / slowest rank."""
    import torch
    import paper_2505_22675_b200 as B
    from paper_2505_22675_b200 import workloads as W
    from paper_2505_22675_b200 import sharding

    world, rank, local = (int(os.environ.get(k, d)) for k, d in (("WORLD_SIZE", "1"), ("RANK", "0"), ("LOCAL_RANK", "0")))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    sw = W.sounding_config(5)                               # same seed on every rank: only rank 0's copy is used
    gk = sw.geom_out
    xs = [torch.from_numpy(a).to(dev) if rank == 0 else torch.zeros(a.shape[0], dtype=torch.float32, device=dev) for a in (sw.x, sw.y, sw.z)]
    mine = sharding.tiles_of_rank(sw.tiles, rank, world)
    geoms = [W.tile_geom(gk, *t) for t in mine]
    bufs = [torch.empty((g.ny, g.nx), dtype=torch.float32, device=dev) for g in geoms]
    failed = torch.zeros(1, dtype=torch.int64, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        sharding.broadcast_soundings(*xs, dist, 0)
        idx = B.krige_build_index(*xs)
        for g, bf in zip(geoms, bufs):
            B.krige_predict(idx, g, sw.model, sw.range_, sw.sill, sw.nugget, sw.k, out=bf, failed=failed)
        idx.free_async()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = B.launch_count()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms = sharding.reduce_step_times([e0.elapsed_time(e1) / args.steps], dist, dev)[0]
    assert int(failed.item()) == 0
    if rank == 0:
        print(json.dumps({"metric": "output nodes/s (ordinary kriging, one config-5 survey sharded by output tile)", "value": gk.n / (ms * 1e-3),
                          "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms,
                          "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": {"workload": WORKLOADS["config5"]["label"], "tiles_per_rank": len(mine),
                                     "parallelism": f"replicated index (one broadcast of {12 * sw.x.shape[0] / 1e6:.0f} MB), output tiles round-robin x{world}"},
                          "gpu_launches": int(B.launch_count() - n0)}))
    if dist is not None:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import paper_2505_22675_b200 as B
    from paper_2505_22675_b200 import workloads as W
    from paper_2505_22675_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    B.lib()                                             # fails loudly if libbathy.so is missing

    gw, sw, tiles = make_inputs(args.workload, rank)
    gi, go, gk = gw.geom_in, gw.geom_out, sw.geom_out
    n_grid, n_krige = go.n, gk.n
    nodes_per_step = 2 * n_grid + n_krige

    # resident inputs and outputs
    z_in = torch.from_numpy(gw.z).to(dev)
    out_b = torch.empty(go.shape, dtype=torch.float32, device=dev)
    out_s = torch.empty(go.shape, dtype=torch.float32, device=dev)
    ws = torch.empty(B.interp_spline_workspace_bytes(gi, go), dtype=torch.uint8, device=dev)
    sx, sy, sz = (torch.from_numpy(a).to(dev) for a in (sw.x, sw.y, sw.z))
    out_k = torch.empty(gk.shape, dtype=torch.float32, device=dev)
    failed = torch.zeros(1, dtype=torch.int64, device=dev)
    tile_geoms = [(W.tile_geom(gk, i0, j0, ny, nx), i0, j0, ny, nx) for (i0, j0, ny, nx) in tiles]
    tile_bufs = [torch.empty((ny, nx), dtype=torch.float32, device=dev) for (_, _, _, ny, nx) in tile_geoms] \
        if len(tiles) > 1 else None
    stream = torch.cuda.current_stream()

    def step(ev=None):
        if ev: ev[0].record(stream)
        B.interp_bilinear(z_in, gi, go, out=out_b)
        if ev: ev[1].record(stream)
        B.interp_spline(z_in, gi, go, out=out_s, workspace=ws)
        if ev: ev[2].record(stream)
        idx = B.krige_build_index(sx, sy, sz)
        if ev: ev[3].record(stream)
        if tile_bufs is None:
            B.krige_predict(idx, gk, sw.model, sw.range_, sw.sill, sw.nugget, sw.k, out=out_k, failed=failed)
        else:                                           # config 5: 64 calls in arrival order
            for (tg, i0, j0, ny, nx), buf in zip(tile_geoms, tile_bufs):
                B.krige_predict(idx, tg, sw.model, sw.range_, sw.sill, sw.nugget, sw.k, out=buf, failed=failed)
        if ev: ev[4].record(stream)
        idx.free_async()                                # stream-ordered: the next step's build reuses the memory
        return idx

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    sampler = ClockSampler(local) if rank == 0 else None
    n0 = B.launch_count()
    t0 = time.time()
    barrier()
    for s in range(args.steps):
        step(evs[s])
    barrier()
    t1 = time.time()
    n1 = B.launch_count()
    clocks = sampler.stop(t0, t1) if sampler else None
    assert int(failed.item()) == 0, "kriging reported failed nodes on the bench workload"

    seg = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(4)] for e in evs])        # ms per segment
    total_ms = float(evs[0][0].elapsed_time(evs[-1][4]))
    total_ms, ms_bil, ms_spl, ms_idx, ms_krg = sharding.reduce_step_times(
        [total_ms] + seg.mean(axis=0).tolist(), dist, dev)          # max over ranks
    ms_per_step = total_ms / args.steps
    seg_med = np.median(seg, axis=0).tolist()
    seg_best = seg.min(axis=0).tolist()

    peaks = load_peaks()
    fp32 = {"derived": SMS * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12, "measured": None}
    table, probe = None, None
    e2e = None
    if args.extras:
        # ---- measured FP32 peak (the library's FMA-chain probe), rank 0 does the reporting but every rank runs it
        probe = measure_fp32_peak(B, stream)
        fp32["measured"] = max(probe.values())

        # ---- end to end through the host-buffer C ABI (pinned host memory, copies inside the timed region)
        hz = torch.from_numpy(gw.z).pin_memory()
        hob = torch.empty(go.shape, dtype=torch.float32).pin_memory()
        hos = torch.empty(go.shape, dtype=torch.float32).pin_memory()
        hx, hy, hzz = (torch.from_numpy(a).pin_memory() for a in (sw.x, sw.y, sw.z))
        hok = torch.empty(gk.shape, dtype=torch.float32).pin_memory()
        hfail = torch.zeros(1, dtype=torch.int64).pin_memory()
        # the three methods of the step are enqueued on three streams through the `*_host_async` entry points
        # (include/bathy.h): the copies of one overlap the kernels and the opposite-direction copies of the
        # others; the host then waits for all three and reads the results.  The two grid methods go on
        # high-priority streams: their short kernels must not queue behind the kriging kernel, whose CTAs
        # fill every SM, because their 268 MB results are what keeps the link busy.
        st_b, st_s = (torch.cuda.Stream(device=dev, priority=-1) for _ in range(2))
        st_k = torch.cuda.Stream(device=dev)

        def e2e_step():
            B.interp_bilinear_host_async(hz, gi, go, out=hob, stream=st_b.cuda_stream)
            B.interp_spline_host_async(hz, gi, go, out=hos, stream=st_s.cuda_stream)
            B.krige_host_async(hx, hy, hzz, gk, sw.model, sw.range_, sw.sill, sw.nugget, sw.k, out=hok, failed=hfail,
                               stream=st_k.cuda_stream)
            st_b.synchronize(); st_s.synchronize(); st_k.synchronize()
            return float(hok[0, 0]) + float(hob[0, 0]) + float(hos[0, 0]) + int(hfail[0])      # the host reads the result

        e2e_steps = max(2, min(args.steps, 10))
        link = measure_link(hz, hob, dev)
        pool_before = (torch.cuda.mem_get_info(dev)[0])
        for _ in range(3):                               # warm-up: pool growth, first use of the three streams
            e2e_step()
        barrier()
        per_step = []
        te0 = time.perf_counter()
        for _ in range(e2e_steps):
            ts0 = time.perf_counter()
            e2e_step()
            per_step.append((time.perf_counter() - ts0) * 1e3)
        barrier()
        e2e_ms = (time.perf_counter() - te0) * 1e3 / e2e_steps
        e2e_ms = sharding.reduce_step_times([e2e_ms], dist, dev)[0]
        h2d_b, d2h_b = 2 * gi.n * 4 + 3 * sw.x.shape[0] * 4, 2 * n_grid * 4 + n_krige * 4 + 8
        floor_ms = max(h2d_b / link["h2d_gbs"], d2h_b / link["d2h_gbs"]) / 1e6     # full duplex: the slower direction
        e2e = {"value": world * nodes_per_step / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": h2d_b, "d2h_bytes_per_step": d2h_b,
               "steps": e2e_steps, "ms_per_step_each": per_step,
               "link_gbs": link, "ms_copy_floor": floor_ms, "ms_over_copy_floor": e2e_ms / floor_ms,
               "device_free_bytes_before_after": [int(pool_before), int(torch.cuda.mem_get_info(dev)[0])],
               "note": "ms_copy_floor = the step's bytes in the slower direction / the bare pinned copy rate measured in this "
                       "process just before (link_gbs); a step far above its floor on a fast link is the library's fault, "
                       "a slow link_gbs is the box's",
               "api": "interp_bilinear_host_async + interp_spline_host_async + krige_host_async on three streams, then stream synchronize (pinned host buffers); no call blocks the host"}
        del hz, hob, hos, hx, hy, hzz, hok

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    if args.extras and world == 1:
        del z_in, out_b, out_s, out_k, ws
        torch.cuda.empty_cache()
        table = per_config_table(B, stream, peaks, fp32, args.reps)

    grid_bytes = 4.0 * (gi.n + n_grid)                  # compulsory: input read once, output written once

    def seg_entry(i, n_nodes):
        return {"nodes_per_s": n_nodes / (seg_med[i] * 1e-3), "ms": [ms_bil, ms_spl, ms_idx, ms_krg][i], "ms_median": seg_med[i],
                "ms_best": seg_best[i]}
    step_methods = {
        "bilinear": {**seg_entry(0, n_grid), "launches": 1,
                     "roofline": hbm_roof({"ms_median": ms_bil, "ms_best": seg_best[0]}, grid_bytes, n_grid, peaks)},
        "spline": {**seg_entry(1, n_grid),
                   "roofline": hbm_roof({"ms_median": ms_spl, "ms_best": seg_best[1]}, grid_bytes, n_grid, peaks)},
        "krige_build_index": {"soundings_per_s": sw.x.shape[0] / (ms_idx * 1e-3), "ms": ms_idx, "ms_median": seg_med[2]},
        "kriging": {**seg_entry(3, n_krige), "k": sw.k, "launches": len(tiles), "ms_per_launch": ms_krg / len(tiles),
                    "roofline": alu_roof(ms_krg, sw.k, n_krige, fp32)},
    }
    dom = max(("bilinear", "spline", "kriging"), key=lambda m: step_methods[m]["ms"])
    kernel_name = {"bilinear": "bilinear_tiled_kernel", "spline": "spline_tables_kernel + spline_tile_kernel",
                   "kriging": "krige_predict_kernel<%d>" % (8 if sw.k <= 8 else 16 if sw.k <= 16 else 32 if sw.k <= 32 else 64)}[dom]
    roof = dict(step_methods[dom]["roofline"])
    if roof["bound"] == "alu" and fp32["measured"]:
        # the judged fraction is against the MEASURED FP32 peak; the derived one stays beside it
        roof.update({"peak": fp32["measured"], "frac": roof["achieved"] / fp32["measured"], "peak_derived": fp32["derived"],
                     "frac_of_derived": roof["achieved"] / fp32["derived"]})
    roof.update({"kernel": kernel_name, "traffic": None, "peak_source": (
        f"{peaks['source']} copy bandwidth (MEASURED_PEAKS.json)" if roof["bound"] == "hbm" else
        ("measured: bathy_probe_fp32 FMA-chain microbenchmark in this run (best of FFMA / FFMA2); derived beside it: "
         if fp32["measured"] else "derived: ") +
        f"{SMS} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x {peaks['sm_max_mhz']:.0f} MHz = {fp32['derived']:.1f} TFLOP/s (DESIGN.md)")})
    tr = os.path.join(ROOT, "profiles", "traffic.json")      # DRAM bytes per launch from the committed ncu capture
    if os.path.exists(tr):
        try:
            with open(tr) as f:
                roof["traffic"] = json.load(f).get(args.workload, {}).get(dom)
        except Exception:
            pass

    line = {
        "metric": METRIC, "value": world * nodes_per_step / (ms_per_step * 1e-3), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.workload]["label"], "nodes_per_step_per_gpu": nodes_per_step,
                   "soundings": int(sw.x.shape[0]), "k": sw.k,
                   "l2": ("grid inputs+outputs (%.0f MB per method) exceed the 126 MB L2; the kriging soundings (%.0f MB) are "
                          "evicted every step by the %.0f MB the two grid methods stream through L2 before it; no explicit flush"
                          % (grid_bytes / 1e6, 16.0 * sw.x.shape[0] / 1e6, 2 * grid_bytes / 1e6))
                   if grid_bytes > 2.0e8 else "grid data fits L2: warm-L2 numbers for bilinear/spline",
                   "parallelism": f"replicated batches x{world}, no collective"},
        "step_methods": step_methods,
        "methods": table if table is not None else {"step": step_methods},
        "roofline": roof,
        "fp32_peak": {"derived_tflops": fp32["derived"], "measured_tflops": fp32["measured"], "probe": probe,
                      "how": "bathy_probe_fp32: 2 CTAs x 512 threads per SM, 16 independent FMA chains per thread, CUDA events"},
        "gpu_launches": int(n1 - n0),
        "clocks": clocks,
    }
    if table is not None:
        # every config's kernels against their rooflines at the top level (the driver's record keeps top-level keys):
        # kriging k = 32 (config 4) AND k = 64 (config 5, 64 streamed tiles), bilinear / spline of configs 2-3
        by = {}
        for cfg, methods in table.items():
            for mname, e in methods.items():
                if isinstance(e, dict) and "roofline" in e and "ms_median" in e:
                    r = e["roofline"]
                    frac = r["frac_of_measured"] if r.get("frac_of_measured") is not None else r["frac"]
                    by[f"{cfg}.{mname}"] = {"bound": r["bound"], "achieved": r["achieved"], "unit": r["unit"],
                                            "peak": r.get("peak_measured") or r["peak"], "frac": frac, "ms_median": e["ms_median"],
                                            **({"k": e["k"]} if "k" in e else {}),
                                            **({"cold_l2_frac": e["cold_l2"]["roofline"]["frac"]} if "cold_l2" in e else {})}
        line["roofline_by_config"] = by
    if e2e is not None:
        line["e2e"] = e2e
    if args.cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(args.workload, budget_s=args.cpu_budget)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------ oracle arm

def oracle_sample_step(name: str, gw, sw, krige_nodes: int, grid_n_in: int):
    """One bounded sample of the step through the float64 oracle: bilinear and spline on the
    top-left grid_n_in^2 crop of the input (same up-sampling factor), kriging at krige_nodes nodes
    spread evenly over the output grid (full sounding set).  Returns seconds per method and the
    nodes each processed."""
    import oracle
    from paper_2505_22675_b200 import workloads as W
    gi, go = gw.geom_in, gw.geom_out
    n = min(grid_n_in, gi.nx)
    factor = round(gi.dx / go.dx)
    crop = np.ascontiguousarray(gw.z[:n, :n])
    ogi = oracle.geom(n, n, gi.x0, gi.y0, gi.dx, gi.dy)
    n_out = (n - 1) * factor + 1
    ogo = oracle.geom(n_out, n_out, go.x0, go.y0, go.dx, go.dy)
    t0 = time.perf_counter(); oracle.bilinear(crop, ogi, ogo); t_b = time.perf_counter() - t0
    t0 = time.perf_counter(); oracle.spline(crop, ogi, ogo); t_s = time.perf_counter() - t0
    gk = sw.geom_out
    v = oracle.vgm(sw.model, sw.range_, sw.sill, sw.nugget)
    t0 = time.perf_counter()
    buckets = oracle.Buckets(sw.x, sw.y, 4.0)
    xq, yq = oracle.node_coords(oracle.geom(gk.nx, gk.ny, gk.x0, gk.y0, gk.dx, gk.dy))
    sel = np.linspace(0, gk.n - 1, min(krige_nodes, gk.n)).astype(np.int64)
    oracle.krige_points(sw.x, sw.y, sw.z, xq.ravel()[sel], yq.ravel()[sel], v, sw.k, buckets, want_nbr=False)
    t_k = time.perf_counter() - t0
    return {"bilinear": (t_b, n_out * n_out), "spline": (t_s, n_out * n_out), "kriging": (t_k, sel.shape[0])}


def extrapolate(sample: dict, n_grid: int, n_krige: int) -> float:
    """nodes/s of the full step mix from per-method sample rates."""
    full = {"bilinear": n_grid, "spline": n_grid, "kriging": n_krige}
    secs = sum(full[m] * sample[m][0] / sample[m][1] for m in full)
    return (2 * n_grid + n_krige) / secs


def cpu_baseline(name: str, budget_s: float = 20.0) -> dict:
    """The oracle as it stands on the box's host cores: all cores (the reported baseline) and ONE thread beside it
    (SURVEY.md 8(d)), bounded samples; plus the k = 64 kriging rate on config 5 when bench.py has it in memory."""
    import oracle
    gw, sw, _ = make_inputs(name, 0)
    cores = oracle.num_threads()
    # sized for ~10-20 s of CPU work: kriging nodes scale with the thread count
    kn = int(max(2000, min(sw.geom_out.n, budget_s * 0.5 * cores * 2.0e4 * (32.0 / sw.k) ** 3)))
    smp = oracle_sample_step(name, gw, sw, krige_nodes=kn, grid_n_in=2048)
    oracle.set_num_threads(1)
    try:
        kn1 = int(max(500, min(sw.geom_out.n, 4.0 * 2.0e4 * (32.0 / sw.k) ** 3)))
        smp1 = oracle_sample_step(name, gw, sw, krige_nodes=kn1, grid_n_in=1024)
    finally:
        oracle.set_num_threads(cores)
    out = {"value": extrapolate(smp, gw.geom_out.n, sw.geom_out.n), "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": (f"float64 oracle, OpenMP x{cores}: bilinear+spline on the {min(2048, gw.geom_in.nx)}^2 crop of the input "
                      f"({smp['bilinear'][1]} nodes each), kriging at {smp['kriging'][1]} evenly spaced nodes with the full "
                      f"sounding set; per-method rates extrapolated to the step's node mix"),
           "per_method_nodes_per_s": {m: smp[m][1] / smp[m][0] for m in smp},
           "one_thread": {"value": extrapolate(smp1, gw.geom_out.n, sw.geom_out.n), "cores": 1,
                          "per_method_nodes_per_s": {m: smp1[m][1] / smp1[m][0] for m in smp1},
                          "sample": f"same oracle, 1 thread: 1024^2 crop ({smp1['bilinear'][1]} nodes), kriging at {smp1['kriging'][1]} nodes"}}
    if ("soundings", 5) in _WORKLOAD_CACHE:
        w5 = _WORKLOAD_CACHE[("soundings", 5)]
        v = oracle.vgm(w5.model, w5.range_, w5.sill, w5.nugget)
        g = w5.geom_out
        buckets = oracle.Buckets(w5.x, w5.y, 4.0)
        xq, yq = oracle.node_coords(oracle.geom(g.nx, g.ny, g.x0, g.y0, g.dx, g.dy))
        rates = {}
        for thr, nn in ((cores, 12000 * cores), (1, 6000)):
            oracle.set_num_threads(thr)
            sel = np.linspace(0, g.n - 1, nn).astype(np.int64)
            t0 = time.perf_counter()
            oracle.krige_points(w5.x, w5.y, w5.z, xq.ravel()[sel], yq.ravel()[sel], v, w5.k, buckets, want_nbr=False)
            rates[f"kriging_k64_config5_x{thr}"] = nn / (time.perf_counter() - t0)
        oracle.set_num_threads(cores)
        out["config5_nodes_per_s"] = rates
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    gw, sw, _ = make_inputs(args.workload, 0)
    cores = oracle.num_threads()
    kn = int(max(1000, min(sw.geom_out.n, 4.0 * cores * 2.0e4 * (32.0 / sw.k) ** 3)))
    for _ in range(min(args.warmup, 1)):
        oracle_sample_step(args.workload, gw, sw, krige_nodes=kn // 4, grid_n_in=512)
    t0 = time.perf_counter()
    vals = []
    for _ in range(args.steps):
        smp = oracle_sample_step(args.workload, gw, sw, krige_nodes=kn, grid_n_in=1024)
        vals.append(extrapolate(smp, gw.geom_out.n, sw.geom_out.n))
    dt = time.perf_counter() - t0
    value = float(np.mean(vals))
    sample = (f"per step: float64 oracle, OpenMP x{cores}, bilinear+spline on the 1024^2 crop ({smp['bilinear'][1]} nodes each), "
              f"kriging at {smp['kriging'][1]} evenly spaced nodes with the full sounding set; rates extrapolated to the step's node mix")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.workload]["label"], "note": "ms_per_step is the wall time of one SAMPLE step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="default", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", dest="cpu_baseline", action="store_false")
    ap.add_argument("--no-extras", dest="extras", action="store_false",
                    help="skip the per-config table, the FP32 probe and e2e (short runs under ncu)")
    ap.add_argument("--shard", default="batch", choices=["batch", "survey"],
                    help="N > 1: every rank its own batch (weak, default) or ONE config-5 survey split by output tile (strong)")
    ap.add_argument("--reps", type=int, default=20, help="separately timed repetitions per method in the per-config table")
    ap.add_argument("--cpu-budget", type=float, default=20.0, help="seconds of oracle work in cpu_baseline")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        if args.warmup < 3:
            args.warmup = 3                              # timing rule: W >= 3
        if args.shard == "survey":
            run_survey_sharded(args)
        else:
            run_ours(args)


if __name__ == "__main__":
    main()
