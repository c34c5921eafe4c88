"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NO interpolation arithmetic.  It only draws the synthetic
bathymetry (plane + Gaussian seamounts/pits + noise), the NaN masks and the
simulated multibeam soundings, and hands identical fp32 buffers to the oracle
(tests) and to the CUDA path.  Recipe: SURVEY.md §8(d) / DESIGN.md "Input recipe".
They stand in for the paper's workloads (§V-B: Grid A
densification -> configs 2-3, Grid B random cell removal -> config 1; onboard
multibeam gridding, PAPER.md:L39, L73-L75 -> configs 4-5).  GEBCO is not used.
"""
from __future__ import annotations

import dataclasses
import numpy as np

SEEDS = {1: 1001, 2: 1002, 3: 1003, 4: 1004, 5: 1005}


@dataclasses.dataclass(frozen=True)
class Geom:
    """Regular grid geometry: node (i, j) sits at x = x0 + j*dx, y = y0 + i*dy."""
    nx: int
    ny: int
    x0: float
    y0: float
    dx: float
    dy: float

    @property
    def shape(self):
        return (self.ny, self.nx)

    @property
    def n(self):
        return self.nx * self.ny


@dataclasses.dataclass(frozen=True)
class Features:
    cx: np.ndarray
    cy: np.ndarray
    amp: np.ndarray
    sigma: np.ndarray


def draw_features(rng: np.random.Generator, n_features: int, extent: float) -> Features:
    """A~U(-80,80) m, sigma~U(2,8) cells, centres uniform over [0, extent]^2."""
    cx = rng.uniform(0.0, extent, n_features)
    cy = rng.uniform(0.0, extent, n_features)
    amp = rng.uniform(-80.0, 80.0, n_features)
    sigma = rng.uniform(2.0, 8.0, n_features)
    return Features(cx, cy, amp, sigma)


def plane(x, y):
    """-5000 m plane tilted 0.5 m/cell along (0.4, 0.3)."""
    return -5000.0 + 0.4 * x + 0.3 * y


def field_on_grid(feat: Features, nx: int, ny: int) -> np.ndarray:
    """Depth field at integer nodes x=j, y=i (float64). Features truncated at 6 sigma."""
    jj = np.arange(nx, dtype=np.float64)
    ii = np.arange(ny, dtype=np.float64)
    z = plane(jj[None, :], ii[:, None]) + np.zeros((ny, nx))
    for cx, cy, a, s in zip(feat.cx, feat.cy, feat.amp, feat.sigma):
        r = 6.0 * s
        j0, j1 = max(int(np.floor(cx - r)), 0), min(int(np.ceil(cx + r)), nx - 1)
        i0, i1 = max(int(np.floor(cy - r)), 0), min(int(np.ceil(cy + r)), ny - 1)
        if j1 < j0 or i1 < i0:
            continue
        dx2 = (jj[j0:j1 + 1] - cx) ** 2
        dy2 = (ii[i0:i1 + 1] - cy) ** 2
        r2 = dy2[:, None] + dx2[None, :]
        z[i0:i1 + 1, j0:j1 + 1] += np.where(r2 <= r * r, a * np.exp(-r2 / (2.0 * s * s)), 0.0)
    return z


def field_at_points(feat: Features, x: np.ndarray, y: np.ndarray, extent: float) -> np.ndarray:
    """Same field evaluated analytically at scattered points (float64)."""
    z = plane(x, y).astype(np.float64)
    bs = 64.0                                   # coarse bucket size, metres
    nb = int(np.ceil(extent / bs)) + 2
    bx = np.clip(np.floor(x / bs).astype(np.int64) + 1, 0, nb - 1)
    by = np.clip(np.floor(y / bs).astype(np.int64) + 1, 0, nb - 1)
    cell = by * nb + bx
    order = np.argsort(cell, kind="stable")
    xs, ys = x[order], y[order]
    start = np.searchsorted(cell[order], np.arange(nb * nb + 1))
    acc = np.zeros_like(xs)
    for cx, cy, a, s in zip(feat.cx, feat.cy, feat.amp, feat.sigma):
        r = 6.0 * s
        bx0 = min(max(int(np.floor((cx - r) / bs)) + 1, 0), nb - 1)
        bx1 = min(max(int(np.floor((cx + r) / bs)) + 1, 0), nb - 1)
        by0 = min(max(int(np.floor((cy - r) / bs)) + 1, 0), nb - 1)
        by1 = min(max(int(np.floor((cy + r) / bs)) + 1, 0), nb - 1)
        for b in range(by0, by1 + 1):
            lo, hi = start[b * nb + bx0], start[b * nb + bx1 + 1]
            if hi <= lo:
                continue
            r2 = (xs[lo:hi] - cx) ** 2 + (ys[lo:hi] - cy) ** 2
            acc[lo:hi] += np.where(r2 <= r * r, a * np.exp(-r2 / (2.0 * s * s)), 0.0)
    z[order] += acc
    return z


# --------------------------------------------------------------------------- gridded configs

@dataclasses.dataclass
class GridWorkload:
    config: int
    z: np.ndarray            # fp32 [ny, nx] input depth grid (config 1: contains NaN)
    geom_in: Geom
    geom_out: Geom
    nan_mask: np.ndarray | None = None


def upsample_geom(n_in: int, factor: int) -> Geom:
    n_out = (n_in - 1) * factor + 1
    return Geom(n_out, n_out, 0.0, 0.0, 1.0 / factor, 1.0 / factor)


def grid_config(config: int, n_in: int | None = None, factor: int | None = None,
                n_features: int | None = None, seed: int | None = None) -> GridWorkload:
    """Configs 1-3. Optional overrides give reduced-size variants with the same recipe."""
    defaults = {1: (64, 4, 20), 2: (1024, 4, 500), 3: (4096, 2, 8000)}
    d = defaults[config]
    n_in = d[0] if n_in is None else n_in
    factor = d[1] if factor is None else factor
    n_features = d[2] if n_features is None else n_features
    rng = np.random.default_rng(SEEDS[config] if seed is None else seed)
    feat = draw_features(rng, n_features, float(n_in))
    z = field_on_grid(feat, n_in, n_in)
    z += rng.normal(0.0, 0.5, size=z.shape)
    z32 = z.astype(np.float32)
    mask = None
    if config == 1:
        n_nan = int(round(0.10 * n_in * n_in))
        perm = rng.permutation(n_in * n_in)[:n_nan]
        mask = np.zeros(n_in * n_in, dtype=bool)
        mask[perm] = True
        mask = mask.reshape(n_in, n_in)
        z32 = z32.copy()
        z32[mask] = np.nan
    gi = Geom(n_in, n_in, 0.0, 0.0, 1.0, 1.0)
    return GridWorkload(config, z32, gi, upsample_geom(n_in, factor), mask)


def grid_to_scattered(z32: np.ndarray):
    """Valid cells of a NaN-holed grid as scattered (x=j, y=i, z) fp32 triples, row-major order."""
    ii, jj = np.nonzero(~np.isnan(z32))
    return jj.astype(np.float32), ii.astype(np.float32), z32[ii, jj].astype(np.float32)


def sample_variance(z: np.ndarray) -> float:
    """Unbiased (n-1) sample variance in float64 -- 'sill = sample variance'."""
    return float(np.var(z.astype(np.float64), ddof=1))


# --------------------------------------------------------------------------- sounding configs

@dataclasses.dataclass
class SoundingWorkload:
    config: int
    x: np.ndarray            # fp32 [N]
    y: np.ndarray
    z: np.ndarray
    geom_out: Geom
    k: int
    model: int               # 0 exponential, 1 spherical
    range_: float
    sill: float
    nugget: float
    tiles: list | None = None    # config 5: list of (i0, j0, ny, nx) in arrival order


def _flag_close(x32: np.ndarray, y32: np.ndarray, delta: float) -> np.ndarray:
    """Superset of points that have another point within `delta` (4 shifted hash grids)."""
    flagged = np.zeros(x32.shape[0], dtype=bool)
    cell = 2.0 * delta
    xd, yd = x32.astype(np.float64), y32.astype(np.float64)
    for sx in (0.0, delta):
        for sy in (0.0, delta):
            kx = np.floor((xd + sx) / cell).astype(np.int64)
            ky = np.floor((yd + sy) / cell).astype(np.int64)
            key = kx * np.int64(1 << 31) + ky
            order = np.argsort(key, kind="stable")
            ks = key[order]
            same = ks[1:] == ks[:-1]
            flagged[order[1:][same]] = True
            flagged[order[:-1][same]] = True
    return flagged


def swath_soundings(rng: np.random.Generator, width: float, n_target: int, beams: int = 256,
                    line_spacing: float = 200.0, altitude: float = 100.0,
                    ping_spacing: float | None = None):
    """Lawnmower multibeam survey: lines parallel to y at x=100+200*l,
    `beams` beams over a +/-60 deg fan + N(0,0.5 deg) roll per ping, flat bottom at `altitude`.
    Memory order = survey order (line, ping, beam). Returns float64 x, y."""
    n_lines = max(int(round(width / line_spacing)), 1)
    if ping_spacing is None:
        pings = int(np.ceil(n_target / (beams * n_lines)))
    else:
        pings = int(round(width / ping_spacing))
    b = np.arange(beams, dtype=np.float64)
    xs, ys = [], []
    for l in range(n_lines):
        xl = 0.5 * line_spacing + line_spacing * l
        roll = rng.normal(0.0, 0.5, pings)
        along = (np.arange(pings) + 0.5) * (width / pings) + rng.normal(0.0, 0.1, pings)
        if l % 2 == 1:                            # alternate heading
            along = width - along
        theta = np.deg2rad(-60.0 + 120.0 * b[None, :] / (beams - 1) + roll[:, None])
        sgn = 1.0 if l % 2 == 0 else -1.0
        xs.append((xl + sgn * altitude * np.tan(theta)).ravel())
        ys.append(np.repeat(along, beams))
    return np.concatenate(xs), np.concatenate(ys)


def sounding_config(config: int, width: float | None = None, n_target: int | None = None,
                    n_out: int | None = None, seed: int | None = None,
                    n_features: int = 8000) -> SoundingWorkload:
    """Configs 4-5. Optional overrides give reduced-size variants with the same recipe
    (same density 0.25 /m^2 when n_target = width^2/4)."""
    defaults = {4: (2000.0, 1_000_000, 2048, 32, 0, 50.0), 5: (4000.0, 4_000_000, 4096, 64, 1, 80.0)}
    d = defaults[config]
    width = d[0] if width is None else width
    n_target = d[1] if n_target is None else n_target
    n_out = d[2] if n_out is None else n_out
    k, model, range_ = d[3], d[4], d[5]
    rng = np.random.default_rng(SEEDS[config] if seed is None else seed)
    # the config-3 feature set over [0, 4096]^2 (own stream so it is the same for configs 3-5)
    feat = draw_features(np.random.default_rng(SEEDS[3]), n_features, 4096.0)
    x, y = swath_soundings(rng, width, n_target)
    x32, y32 = x.astype(np.float32), y.astype(np.float32)
    for _ in range(20):                           # re-jitter near-duplicates (min separation 1e-3 m)
        bad = _flag_close(x32, y32, 1e-3)
        if not bad.any():
            break
        nb = int(bad.sum())
        x[bad] += rng.normal(0.0, 0.05, nb)
        y[bad] += rng.normal(0.0, 0.05, nb)
        x32, y32 = x.astype(np.float32), y.astype(np.float32)
    else:
        raise RuntimeError("could not separate near-duplicate soundings")
    z = field_at_points(feat, x32.astype(np.float64), y32.astype(np.float64), 4096.0)
    z += rng.normal(0.0, 0.3, z.shape)
    z32 = z.astype(np.float32)
    sill = sample_variance(z32)
    d_out = width / n_out
    geom = Geom(n_out, n_out, 0.5 * d_out, 0.5 * d_out, d_out, d_out)
    tiles = None
    if config == 5:
        tiles = boustrophedon_tiles(n_out, max(n_out // 8, 1))
    return SoundingWorkload(config, x32, y32, z32, geom, k, model, range_, sill, 0.01 * sill, tiles)


def boustrophedon_tiles(n_out: int, tile: int):
    """Tiles of `tile`^2 nodes in arrival order: tile columns left to right (following the survey
    lines, which are parallel to y), alternating up/down within a column."""
    nt = (n_out + tile - 1) // tile
    order = []
    for tj in range(nt):
        rows = range(nt) if tj % 2 == 0 else range(nt - 1, -1, -1)
        for ti in rows:
            i0, j0 = ti * tile, tj * tile
            order.append((i0, j0, min(tile, n_out - i0), min(tile, n_out - j0)))
    return order


def tile_geom(g: Geom, i0: int, j0: int, ny: int, nx: int) -> Geom:
    """Sub-geometry of a tile: x0/y0 shifted to the tile's first node.
    With the config-5 geometry (dx = 125/128, x0 = dx/2) every node coordinate is exact in
    fp32, so tile nodes are bit-identical to the monolithic grid's nodes."""
    return Geom(nx, ny, g.x0 + j0 * g.dx, g.y0 + i0 * g.dy, g.dx, g.dy)
