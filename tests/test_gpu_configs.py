"""GPU parity at the sizes of BASELINE.json's configs (prefixes of the full runs where the oracle would need minutes):
config 2 at 512 x 512, config 3 at 256 x 256 coarse with ratio 4, config 4's four-level hierarchy at a reduced coarse
grid, and config 5 at the full 8192 x 8192 in bench.py's launch configuration, compared on sampled windows the oracle
recomputes one by one.  State and masks bit-exact."""
import numpy as np
import pytest

import workloads
from harness import driver
from test_gpu_amr import lockstep_hierarchies, same_storage

pytestmark = pytest.mark.gpu


def test_config2_full_size_prefix(gc, gco):
    wl = workloads.cfg2(512)
    Lg = driver.setup_level(gc.Context(**wl.params), wl, patches=workloads.tile(512, 512, 128))
    Lo = driver.setup_level(gco.Context(**wl.params), wl)
    hg = driver.run_single_level(Lg, 120, wl.cfl)
    ho = driver.run_single_level(Lo, 120, wl.cfl)
    assert [d for d, _ in hg] == [d for d, _ in ho]
    assert [s["n_clipped"] for _, s in hg] == [s["n_clipped"] for _, s in ho]
    for f in ("h", "hu", "hv"):
        assert np.array_equal(Lg.get_global(f), Lo.get_global(f)), f
    mg = driver.unpack_cells(Lg, Lg.wet_mask()); mo = driver.unpack_cells(Lo, Lo.wet_mask())
    assert np.array_equal(mg, mo) and 0 < mo.sum() < mo.size       # wet and dry cells both present


def test_config3_full_size_prefix(gc, gco):
    wl = workloads.cfg3(256)
    Hg, Ho = lockstep_hierarchies(gc, gco, wl, 5)
    assert len(Hg.levels) == 2 and Hg.regrids >= 1 and Hg.levels[1].ncells > 20000


def test_config4_four_levels_reduced(gc, gco):
    wl = workloads.cfg4(120, 60)
    wl.patch_max = 60
    wl.forced_boxes = tuple((lv, x0, x1, y0, y1, 0.0, t1) for lv, x0, x1, y0, y1, t0, t1 in wl.forced_boxes)   # coastal boxes on from t = 0
    Hg, Ho = lockstep_hierarchies(gc, gco, wl, 2)
    assert len(Hg.levels) == 4
    assert any(int(L.wet_mask().sum()) < L.ncells for L in Hg.levels[2:])      # the fine levels straddle the shoreline


def test_config5_full_size_sampled_windows(gc, gco):
    """8192 x 8192 in 32 x 32 patches of side 256 (the bench configuration): one level step, then windows of the result
    against the oracle stepping a one-patch level that holds the same initial data (ghost cells included)."""
    n, side, w = 8192, 256, 24
    wl = workloads.cfg5(n)
    ctx = gc.Context(**wl.params)
    L = ctx.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, workloads.tile(n, n, side))
    rows = (1 << 24) // n
    for j0 in range(0, n, rows):
        b, h, hu, hv = wl.fields(i0=0, j0=j0, nx=n, ny=rows)
        L.set_global("b", b, 0, j0); L.set_global("h", h, 0, j0); L.set_global("hu", hu, 0, j0); L.set_global("hv", hv, 0, j0)
    L.fill_ghost_b()
    dt = driver.probe_dt(L, wl.cfl)
    L.fill_ghost(None, 1.0)
    st = L.step(dt)
    assert st["nan_seen"] == 0 and 0.85 < st["cfl_max"] <= 0.9 * (1 + 1e-12)
    # windows: patch interiors, patch corners (four patches meet), the domain corner and edges
    wins = [(100, 100), (256 - 12, 512 - 12), (4096 - 12, 4096 - 12), (0, 0), (n - w, 3000), (5000, n - w), (8192 - 256 - 12, 17)]
    co = gco.Context(**wl.params)
    sdx = 0.0
    for (i0, j0) in wins:
        Lo = co.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, np.array([[i0, j0, w, w]], dtype=np.int32))
        # storage-shaped input (ghost cells included) straight from the analytic recipe; ghost cells outside the domain
        # take the nearest interior cell (zero-order extrapolation) -- no ghost fill is run on this side
        gi = np.clip(np.arange(i0 - 2, i0 + w + 2), 0, n - 1); gj = np.clip(np.arange(j0 - 2, j0 + w + 2), 0, n - 1)
        a0, c0 = int(gi.min()), int(gj.min())
        fb = wl.fields(i0=a0, j0=c0, nx=int(gi.max()) - a0 + 1, ny=int(gj.max()) - c0 + 1)
        for p_, (f, v) in enumerate(zip(("b", "h", "hu", "hv"), fb)):
            Lo.set_field(0, f, v[np.ix_(gj - c0, gi - a0)])
        so = Lo.step(dt)
        sdx = max(sdx, so["s_over_dx_max"])
        for f in ("h", "hu", "hv"):
            g = L.get_global(f, gi0=i0, gj0=j0, gnx=w, gny=w)
            o = Lo.get_global(f, gi0=i0, gj0=j0, gnx=w, gny=w)
            assert np.array_equal(g, o), (f, i0, j0, np.abs(g - o).max())
        Lo.destroy()
    assert sdx <= st["s_over_dx_max"]
    L.destroy()
