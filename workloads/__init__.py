"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the oracle and the CUDA path and therefore holds none of the method's
arithmetic: it only evaluates analytic bathymetry b(x, y) and initial surface eta0(x, y) at cell
centres and builds h = max(0, eta0 - b), hu = hv = 0.  The paper's real workloads (P:273-292 Japan
2011, P:333-345 Seattle Fault) need PMEL deformation files, topography and gauge records that are
not in this container; these inputs stand in for their structure (deep-ocean propagation on lon/lat
AMR; long irregular wet/dry shoreline).  All randomness: numpy default_rng(1901067980 + config).
"""
from dataclasses import dataclass, field
from typing import Callable, Tuple

import numpy as np

SEED0 = 1901067980
EARTH_RADIUS = 6367500.0
DEG2M = EARTH_RADIUS * np.pi / 180.0  # metres per degree of latitude (generator-side geometry only)


@dataclass
class Workload:
    name: str
    params: dict                      # kwargs for Context(...): coord, g, dry_tol, sea_level, earth_radius, limiter, bc
    xlo: float
    ylo: float
    dx: float
    dy: float
    nx: int
    ny: int
    bathy: Callable                   # b(x, y) vectorised
    eta0: Callable                    # eta0(x, y) vectorised
    cfl: float = 0.9
    nsteps: int = 0                   # coarse steps (single-level configs)
    t_end: float = 0.0                # simulated seconds (AMR configs)
    ratios: Tuple[int, ...] = ()      # refinement ratios level l -> l+1
    flag: dict = field(default_factory=dict)   # flag parameters per the AMR driver
    regrid_interval: int = 4
    patch_min: int = 32
    patch_max: int = 64
    forced_boxes: Tuple = ()          # (level, x0, x1, y0, y1, t0, t1): refine level -> level+1 inside
    wave_levels: int = 99             # the wave criteria (tol_eta, ...) flag levels 1..wave_levels only; finer levels come from boxes
    deform: dict = None               # seafloor deformation: dict(x0, y0, ddx, ddy, dz (my, mx), t0, t1) or None
    _tiles: dict = field(default_factory=dict, repr=False, compare=False)   # bathy_box cache

    def centers(self, level_dx=None, level_dy=None, i0=0, j0=0, nx=None, ny=None):
        dx = self.dx if level_dx is None else level_dx
        dy = self.dy if level_dy is None else level_dy
        nx = self.nx if nx is None else nx
        ny = self.ny if ny is None else ny
        x = self.xlo + (np.arange(i0, i0 + nx, dtype=np.float64) + 0.5) * dx
        y = self.ylo + (np.arange(j0, j0 + ny, dtype=np.float64) + 0.5) * dy
        return np.meshgrid(x, y)

    TILE = 256                        # bathy_box: cells per tile side
    TILE_CACHE_BYTES = 6 << 30        # the cache is dropped when it grows past this

    def bathy_box(self, level_dx=None, level_dy=None, i0=0, j0=0, nx=None, ny=None):
        """b at the cell centres of the box [i0,i0+nx) x [j0,j0+ny) of a level with the given cell size.
        The bathymetry is static, so it is evaluated once per cell and level -- in tiles of TILE x TILE cells aligned to
        the level's global cell indices, kept for the life of the workload -- the way a topography file is read once;
        a regrid that re-refines a region already seen costs a copy.  A cell's value does not depend on which box asks."""
        dx = self.dx if level_dx is None else level_dx
        dy = self.dy if level_dy is None else level_dy
        nx = self.nx if nx is None else nx
        ny = self.ny if ny is None else ny
        T = self.TILE
        out = np.empty((ny, nx), dtype=np.float64)
        for tj in range(j0 // T, (j0 + ny - 1) // T + 1):
            for ti in range(i0 // T, (i0 + nx - 1) // T + 1):
                key = (id(self.bathy), dx, dy, ti, tj)
                tile = self._tiles.get(key)
                if tile is None:
                    if sum(t.nbytes for t in self._tiles.values()) > self.TILE_CACHE_BYTES:
                        self._tiles.clear()
                    X, Y = self.centers(dx, dy, ti * T, tj * T, T, T)
                    tile = np.ascontiguousarray(self.bathy(X, Y), dtype=np.float64)
                    self._tiles[key] = tile
                a0, a1 = max(i0, ti * T), min(i0 + nx, (ti + 1) * T)
                c0, c1 = max(j0, tj * T), min(j0 + ny, (tj + 1) * T)
                out[c0 - j0:c1 - j0, a0 - i0:a1 - i0] = tile[c0 - tj * T:c1 - tj * T, a0 - ti * T:a1 - ti * T]
        return out

    def bathy_tile(self, dx, dy, ti, tj):
        """the cached T x T tile (ti, tj) of the level with cell size (dx, dy), evaluated on first use"""
        key = (id(self.bathy), dx, dy, ti, tj)
        tile = self._tiles.get(key)
        if tile is None:
            if sum(t.nbytes for t in self._tiles.values()) > self.TILE_CACHE_BYTES:
                self._tiles.clear()
            X, Y = self.centers(dx, dy, ti * self.TILE, tj * self.TILE, self.TILE, self.TILE)
            tile = np.ascontiguousarray(self.bathy(X, Y), dtype=np.float64)
            self._tiles[key] = tile
        return tile

    def fields(self, level_dx=None, level_dy=None, i0=0, j0=0, nx=None, ny=None):
        """b, h, hu, hv at cell centres of the box [i0,i0+nx) x [j0,j0+ny) of a level with the given cell size."""
        X, Y = self.centers(level_dx, level_dy, i0, j0, nx, ny)
        b = self.bathy_box(level_dx, level_dy, i0, j0, nx, ny)
        eta = np.asarray(self.eta0(X, Y), dtype=np.float64)
        h = np.maximum(0.0, eta - b)
        z = np.zeros_like(h)
        return b, h, z, z.copy()


def cfg1(n=64):
    """Config 1: 64x64 Cartesian, dx = 1 km, b = -4000 m, 1 m Gaussian hump (sigma 5 km) centred on a cell corner, walls."""
    L = n * 1000.0
    def bathy(x, y): return np.full(np.broadcast(x, y).shape, -4000.0)
    def eta0(x, y): return np.exp(-((x - 0.5 * L) ** 2 + (y - 0.5 * L) ** 2) / (2.0 * 5000.0 ** 2))
    return Workload("cfg1", dict(coord=0, dry_tol=1e-3, bc=(1, 1, 1, 1)), 0.0, 0.0, 1000.0, 1000.0, n, n,
                    bathy, eta0, cfl=0.9, nsteps=100)


def cfg2(n=512):
    """Config 2: Cartesian n x n, dx = 100 m, slope -200 m .. +20 m plus 8 seeded Fourier modes (total amplitude 2 m);
    2 m Gaussian ridge along y at x = 10 km (scaled with n); extrapolation BCs; wet and dry cells."""
    rng = np.random.default_rng(SEED0 + 2)
    L = n * 100.0
    modes = []
    while len(modes) < 8:
        m, k = int(rng.integers(0, 5)), int(rng.integers(0, 5))
        if m == 0 and k == 0:
            continue
        modes.append((m, k, float(rng.uniform(0.0, 2.0 * np.pi))))
    x0 = 10000.0 * n / 512.0
    sig = 1500.0 * n / 512.0
    def bathy(x, y):
        b = -200.0 + 220.0 * x / L
        for m, k, ph in modes:
            b = b + 0.25 * np.cos(2.0 * np.pi * (m * x + k * y) / L + ph)
        return b
    def eta0(x, y): return 2.0 * np.exp(-((x - x0) ** 2) / (2.0 * sig ** 2)) + 0.0 * y
    return Workload("cfg2", dict(coord=0, dry_tol=1e-3, bc=(0, 0, 0, 0)), 0.0, 0.0, 100.0, 100.0, n, n,
                    bathy, eta0, cfl=0.9, nsteps=2000)


def _dist_m(lon, lat, lon0, lat0):
    """Local flat-earth distance components in metres (generator geometry only)."""
    ex = (lon - lon0) * DEG2M * np.cos(np.deg2rad(lat0))
    ey = (lat - lat0) * DEG2M
    return ex, ey


def cfg3(n=256):
    """Config 3: spherical 2-level AMR, coarse n x n at 2 arcmin over ~8.5 deg; seamount; 0.5 m elliptical Gaussian."""
    rng = np.random.default_rng(SEED0 + 3)
    d = 2.0 / 60.0
    xlo, ylo = 140.0, 30.0
    W = n * d
    sm = (xlo + W * rng.uniform(0.25, 0.75), ylo + W * rng.uniform(0.25, 0.75))
    src = (xlo + W * rng.uniform(0.35, 0.65), ylo + W * rng.uniform(0.35, 0.65))
    ang = float(rng.uniform(0.0, np.pi))
    def bathy(x, y):
        ex, ey = _dist_m(x, y, *sm)
        return -3000.0 + 2800.0 * np.exp(-(ex ** 2 + ey ** 2) / (2.0 * 40000.0 ** 2))
    def eta0(x, y):
        ex, ey = _dist_m(x, y, *src)
        a = ex * np.cos(ang) + ey * np.sin(ang)
        c = -ex * np.sin(ang) + ey * np.cos(ang)
        return 0.5 * np.exp(-(a ** 2 / (2.0 * 60000.0 ** 2) + c ** 2 / (2.0 * 25000.0 ** 2)))
    return Workload("cfg3", dict(coord=1, dry_tol=1e-3, bc=(0, 0, 0, 0)), xlo, ylo, d, d, n, n, bathy, eta0,
                    cfl=0.9, t_end=3600.0, ratios=(4,), flag=dict(tol_eta=0.01, buffer=4),
                    regrid_interval=4, patch_min=32, patch_max=64)


def cfg4(nx=1800, ny=900):
    """Config 4: transoceanic synthetic, 120 x 60 deg at 4 arcmin, ratios 5, 6, 4; ridges, shelf, east coastline strip."""
    rng = np.random.default_rng(SEED0 + 4)
    d = 120.0 / nx
    xlo, ylo = 130.0, 0.0
    W, H = nx * d, ny * d
    ridges = [(xlo + W * rng.uniform(0.15, 0.8), ylo + H * rng.uniform(0.1, 0.9), rng.uniform(500.0, 2500.0),
               rng.uniform(1.0, 4.0), rng.uniform(0.3, 1.5)) for _ in range(12)]
    wav = [(rng.uniform(0.2, 0.8), int(rng.integers(1, 6)), rng.uniform(0, 2 * np.pi)) for _ in range(4)]
    coast0 = xlo + 0.94 * W
    src = (xlo + 0.08 * W, ylo + 0.62 * H)
    def coastline(y):
        c = np.full_like(np.asarray(y, dtype=np.float64), coast0)
        for a, k, ph in wav:
            c = c + a * np.sin(2 * np.pi * k * (y - ylo) / H + ph)
        return c
    def bathy(x, y):
        b = np.full(np.broadcast(x, y).shape, -4500.0)
        for cx, cy, amp, sx, sy in ridges:
            b = b + amp * np.exp(-((x - cx) ** 2 / (2 * sx ** 2) + (y - cy) ** 2 / (2 * sy ** 2)))
        s = x - coastline(y)  # degrees east of the coastline
        shelf = -200.0 + (b + 200.0) * 0.5 * (1.0 - np.tanh((s + 3.0) / 0.5))   # abyssal -> shelf 3 deg offshore
        strip = np.clip(s / 0.5, -1.0, 1.0)                                     # shelf -> +30 m across the coast
        return np.where(s > -0.5, -200.0 + 230.0 * 0.5 * (strip + 1.0) * (s > -0.5), shelf) + 0.0
    def eta0(x, y):
        ex, ey = _dist_m(x, y, *src)
        up = 5.0 * np.exp(-(ex ** 2 / (2 * 80000.0 ** 2) + ey ** 2 / (2 * 200000.0 ** 2)))
        ex2, ey2 = _dist_m(x, y, src[0] - 1.8, src[1])
        dn = -2.0 * np.exp(-(ex2 ** 2 / (2 * 80000.0 ** 2) + ey2 ** 2 / (2 * 200000.0 ** 2)))
        return up + dn
    cy = ylo + 0.5 * H
    boxes = ((2, coast0 - 2.0, coast0 + 0.6, cy - 1.5, cy + 1.5, 6.0 * 3600, 1e30),
             (3, coast0 - 0.8, coast0 + 0.4, cy - 0.4, cy + 0.4, 6.5 * 3600, 1e30))
    return Workload("cfg4", dict(coord=1, dry_tol=1e-3, bc=(0, 0, 0, 0)), xlo, ylo, d, d, nx, ny, bathy, eta0,
                    cfl=0.9, t_end=36000.0, ratios=(5, 6, 4), flag=dict(tol_eta=0.02, offshore_only=1, buffer=3),
                    regrid_interval=3, patch_min=50, patch_max=200, forced_boxes=boxes, wave_levels=1)


def cfg4_deformation(nx=1800, ny=900, t_rise=120.0, spacing=0.1):
    """Config 4 started the way the paper starts its tsunamis: the ocean is at rest and the +5 m / -2 m dipole is a
    seafloor deformation on a uniform node grid of `spacing` degrees around the source, applied over [0, t_rise] seconds
     -- instead of an initial surface displacement over a static bed."""
    wl = cfg4(nx, ny)
    src_x, src_y = wl.xlo + 0.08 * nx * wl.dx, wl.ylo + 0.62 * ny * wl.dy
    x0, y0 = max(wl.xlo, src_x - 8.0), src_y - 10.0
    mx, my = int(round((src_x + 6.0 - x0) / spacing)) + 1, int(round(20.0 / spacing)) + 1
    X, Y = np.meshgrid(x0 + spacing * np.arange(mx), y0 + spacing * np.arange(my))
    dz = np.ascontiguousarray(wl.eta0(X, Y), dtype=np.float64)
    dz[np.abs(dz) < 1e-4] = 0.0                                    # a deformation file has a finite footprint
    wl.deform = dict(x0=float(x0), y0=float(y0), ddx=float(spacing), ddy=float(spacing), dz=dz, t0=0.0, t1=float(t_rise))
    wl.eta0 = lambda x, y: np.zeros(np.broadcast(x, y).shape)
    wl.name = "cfg4-deformation"
    return wl


def cfg5(n=8192):
    """Config 5: spherical single level n x n at 0.5 arcmin, seeded smooth bathymetry in [-6000, -50] m (fully wet),
    12 seeded +-Gaussians of |a| <= 1 m; extrapolation BCs.  Tiled by the caller into equal square patches."""
    rng = np.random.default_rng(SEED0 + 5)
    d = 0.5 / 60.0
    W = n * d
    xlo, ylo = 0.0, -0.5 * W
    modes = [(int(rng.integers(0, 4)), int(rng.integers(0, 4)), float(rng.uniform(0, 2 * np.pi)), float(rng.uniform(0.3, 1.0)))
             for _ in range(16)]
    modes = [(m if (m or k) else 1, k, ph, a) for m, k, ph, a in modes]
    asum = sum(a for _, _, _, a in modes)
    bumps = [(xlo + W * rng.uniform(0.1, 0.9), ylo + W * rng.uniform(0.1, 0.9), float(rng.uniform(-1.0, 1.0)),
              float(rng.uniform(50e3, 150e3)) * (n / 8192.0)) for _ in range(12)]
    def bathy(x, y):
        s = np.zeros(np.broadcast(x, y).shape)
        for m, k, ph, a in modes:
            s = s + a * np.cos(2 * np.pi * (m * (x - xlo) + k * (y - ylo)) / W + ph)
        return -3025.0 + 2975.0 * (s / asum)  # affine map of [-1, 1] onto [-6000, -50]
    def eta0(x, y):
        e = np.zeros(np.broadcast(x, y).shape)
        for cx, cy, a, sg in bumps:
            ex, ey = _dist_m(x, y, cx, cy)
            e = e + a * np.exp(-(ex ** 2 + ey ** 2) / (2 * sg ** 2))
        return e
    return Workload("cfg5", dict(coord=1, dry_tol=1e-3, bc=(0, 0, 0, 0)), xlo, ylo, d, d, n, n, bathy, eta0,
                    cfl=0.9, nsteps=200)


def tile(nx, ny, side):
    """Equal square patches of the given side covering an nx x ny level, sorted by (j0, i0)."""
    assert nx % side == 0 and ny % side == 0
    i0, j0 = np.meshgrid(np.arange(0, nx, side), np.arange(0, ny, side))
    p = np.stack([i0.ravel(), j0.ravel(), np.full(i0.size, side), np.full(i0.size, side)], axis=1)
    return np.ascontiguousarray(p, dtype=np.int32)
