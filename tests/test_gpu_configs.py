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


def _extrapolate_outside(a, n_lo_x, n_hi_x, n_lo_y, n_hi_y):
    """zero-order extrapolation of a storage-shaped array: the n_* outermost columns / rows lie outside the
    domain and take the nearest cell inside it, x faces first, then y faces over all columns"""
    if n_lo_x: a[:, :n_lo_x] = a[:, n_lo_x:n_lo_x + 1]
    if n_hi_x: a[:, -n_hi_x:] = a[:, -n_hi_x - 1:-n_hi_x]
    if n_lo_y: a[:n_lo_y, :] = a[n_lo_y:n_lo_y + 1, :]
    if n_hi_y: a[-n_hi_y:, :] = a[-n_hi_y - 1:-n_hi_y, :]
    return a


def test_config5_full_size_sampled_windows(gc, gco):
    """8192 x 8192 in 32 x 32 patches of side 256 (the bench configuration and its launch path: gc_fill_ghost +
    gc_level_step_auto, dt chained on the device), K = 10 steps.  Windows of the result against the oracle, which advances
    one-patch levels grown by 2 K cells around each window (the domain of dependence of K steps: 2 cells per sweep direction and
    step) from the same initial data with the dt sequence the device chain produced.  The oracle's patches get no ghost fill from
    neighbours they do not have, so what is wrong creeps in from their rim by 2 cells per step and stops short of the window;
    where a window touches the domain boundary the test applies the extrapolation rule itself."""
    import torch
    n, side, w, K = 8192, 256, 24, 10
    m = 2 * K
    wl = workloads.cfg5(n)
    ctx = gc.Context(**wl.params)
    L = ctx.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, workloads.tile(n, n, side))
    rows = (1 << 24) // n
    for j0 in range(0, n, rows):
        b, h, hu, hv = wl.fields(i0=0, j0=j0, nx=n, ny=rows)
        L.set_global("b", b, 0, j0); L.set_global("h", h, 0, j0); L.set_global("hu", hu, 0, j0); L.set_global("hv", hv, 0, j0)
    L.fill_ghost_b()
    dt0 = driver.probe_dt(L, wl.cfl)
    dt_dev = torch.tensor([dt0], dtype=torch.float64, device=ctx.device)
    dts, sdxs = [], []
    for k in range(K):
        dts.append(float(dt_dev.item()))
        L.fill_ghost(None, 1.0)
        L.step_auto(dt_dev, wl.cfl)
        st = L.stats()
        assert st["nan_seen"] == 0
        sdxs.append(st["s_over_dx_max"])
        assert float(dt_dev.item()) == wl.cfl / st["s_over_dx_max"]                    # the device chain: dt_{k+1} = cfl / max s/(kappa dx)
    assert all(0.85 < d * s_ <= 0.9 * (1 + 1e-12) for d, s_ in zip(dts, sdxs))        # (the deepest point sets the speed: dt barely moves)
    # windows: patch interiors, patch corners (four patches meet), the domain corner and edges
    wins = [(100, 100), (256 - 12, 512 - 12), (4096 - 12, 4096 - 12), (0, 0), (n - w, 3000), (5000, n - w), (8192 - 256 - 12, 17)]
    co = gco.Context(**wl.params)
    sdx0 = 0.0
    for (i0, j0) in wins:
        a0, a1 = max(i0 - m, 0), min(i0 + w + m, n)
        c0, c1 = max(j0 - m, 0), min(j0 + w + m, n)
        Lo = co.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, np.array([[a0, c0, a1 - a0, c1 - c0]], dtype=np.int32))
        # storage-shaped input (ghost cells included) straight from the analytic recipe; ghost cells outside the domain
        # take the nearest interior cell (zero-order extrapolation)
        gi = np.clip(np.arange(a0 - 2, a1 + 2), 0, n - 1); gj = np.clip(np.arange(c0 - 2, c1 + 2), 0, n - 1)
        fb = wl.fields(i0=int(gi.min()), j0=int(gj.min()), nx=int(gi.max() - gi.min()) + 1, ny=int(gj.max() - gj.min()) + 1)
        for f, v in zip(("b", "h", "hu", "hv"), fb):
            Lo.set_field(0, f, v[np.ix_(gj - gj.min(), gi - gi.min())])
        out = (2 if a0 == 0 else 0, 2 if a1 == n else 0, 2 if c0 == 0 else 0, 2 if c1 == n else 0)
        for k in range(K):
            if any(out) and k > 0:
                for f in ("h", "hu", "hv"):
                    Lo.set_field(0, f, _extrapolate_outside(Lo.get_field(0, f), *out))
            so = Lo.step(dts[k])
            if k == 0:                                       # later steps: the rim of the oracle's patch may hold anything
                sdx0 = max(sdx0, so["s_over_dx_max"])
        for f in ("h", "hu", "hv"):
            g = L.get_global(f, gi0=i0, gj0=j0, gnx=w, gny=w)
            o = Lo.get_global(f, gi0=i0, gj0=j0, gnx=w, gny=w)
            assert np.array_equal(g, o), (f, i0, j0, np.abs(g - o).max())
            if f != "h":
                assert np.abs(o).max() > 0.0                                            # momentum has developed: not a step from rest
        Lo.destroy()
    assert sdx0 <= sdxs[0]
    L.destroy()
