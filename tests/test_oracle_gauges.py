"""Pins for the oracle's gauge sampling (oracle/gco_amr.c gco_gauges_sample, reading S-19):
a field linear in x and y is reproduced, also across patch boundaries (the stencil reads the sibling's cells through the ghost
ring); at a cell centre the sample is the cell's value bit for bit; scipy's RegularGridInterpolator (an independent routine)
gives the same numbers on a smooth field; a stencil that touches a dry cell falls back to the containing cell; a point outside
its patch is refused; a gauge in an ocean at rest over rough bathymetry records the sea level throughout a run."""
import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

import workloads
from harness import driver
from test_oracle_2d import make_level


def patch_of(patches, dx, dy, x, y, xlo=0.0, ylo=0.0):
    ic, jc = int(np.floor((x - xlo) / dx)), int(np.floor((y - ylo) / dy))
    for p, (i0, j0, nx, ny) in enumerate(patches):
        if i0 <= ic < i0 + nx and j0 <= jc < j0 + ny:
            return p
    raise ValueError("no patch")


def centres(n, d):
    return (np.arange(n) + 0.5) * d


def test_linear_field_is_reproduced_across_patch_boundaries(gco):
    n, d = 24, 50.0
    X, Y = np.meshgrid(centres(n, d), centres(n, d))
    b = np.full((n, n), -30.0)
    h = 20.0 + 0.004 * X - 0.003 * Y
    hu = 1.0 + 0.002 * X + 0.001 * Y
    hv = -2.0 + 0.0005 * X - 0.002 * Y
    pats = np.array([[0, 0, 10, 24], [10, 0, 14, 9], [10, 9, 14, 15]], dtype=np.int32)
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(0, 0, 0, 0)), n, n, d, d, b, h, hu=hu, hv=hv, patches=pats)
    L.fill_ghost(None, 1.0)
    rng = np.random.default_rng(4)
    pts = rng.uniform(1.5 * d, (n - 1.5) * d, (400, 2))                    # a cell away from the domain edge (its ghosts are constant)
    pts = np.vstack([pts, [[10 * d + 1e-9, 300.0], [10 * d - 1e-9, 300.0], [600.0, 9 * d + 1.0], [600.0, 9 * d - 1.0]]])
    pid = [patch_of(pats, d, d, x, y) for x, y in pts]
    assert len(set(pid)) == 3
    out = L.gauges_sample(pid, pts)
    x, y = pts[:, 0], pts[:, 1]
    exact = np.stack([20.0 + 0.004 * x - 0.003 * y, 1.0 + 0.002 * x + 0.001 * y, -2.0 + 0.0005 * x - 0.002 * y,
                      -10.0 + 0.004 * x - 0.003 * y], axis=1)
    assert np.abs(out - exact).max() <= 2e-13 * 30.0


def test_cell_centres_return_the_cell_bit_for_bit(gco):
    wl = workloads.cfg2(32)
    pats = workloads.tile(32, 32, 8)
    L = driver.setup_level(gco.Context(**wl.params), wl, patches=pats)
    driver.run_single_level(L, 12, wl.cfl)
    L.fill_ghost(None, 1.0)
    H, U, V, B = (L.get_global(f) for f in ("h", "hu", "hv", "b"))
    xs = wl.xlo + centres(32, wl.dx); ys = wl.ylo + centres(32, wl.dy)
    pts = np.array([[x, y] for y in ys for x in xs])
    pid = [patch_of(pats, wl.dx, wl.dy, x, y, wl.xlo, wl.ylo) for x, y in pts]
    out = L.gauges_sample(pid, pts).reshape(32, 32, 4)
    assert (H <= 1e-3).any() and (H > 1e-3).any()                             # wet and dry cells, both rules exercised
    assert np.array_equal(out[..., 0], H) and np.array_equal(out[..., 1], U) and np.array_equal(out[..., 2], V)
    assert np.array_equal(out[..., 3], H + B)


def test_against_scipy_linear_interpolator(gco):
    n, d = 40, 125.0
    rng = np.random.default_rng(8)
    X, Y = np.meshgrid(centres(n, d), centres(n, d))
    b = -50.0 + 5.0 * np.sin(X / 700.0) * np.cos(Y / 900.0)
    h = 50.0 + 3.0 * np.cos(X / 500.0 + 0.3) + 2.0 * np.sin(Y / 350.0)        # all wet
    hu = 10.0 * np.sin((X + Y) / 800.0); hv = rng.normal(0.0, 1.0, (n, n))
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(0, 0, 0, 0)), n, n, d, d, b, h, hu=hu, hv=hv)
    L.fill_ghost(None, 1.0)
    pts = rng.uniform(0.5 * d, (n - 0.5) * d * (1 - 1e-12), (1000, 2))        # inside the hull of the cell centres
    out = L.gauges_sample(np.zeros(len(pts), dtype=np.int32), pts)
    c = centres(n, d)
    for f, field in enumerate((h, hu, hv, h + b)):
        ref = RegularGridInterpolator((c, c), field.T, method="linear")(pts)  # axes (x, y)
        assert np.abs(out[:, f] - ref).max() <= 1e-12 * np.abs(field).max()


def test_a_dry_cell_in_the_stencil_falls_back_to_the_containing_cell(gco):
    n, d = 12, 10.0
    b = np.full((n, n), -2.0); b[:, 6:] = 1.0                                 # land from column 6 on
    h = np.maximum(0.0, 0.25 - b)
    hu = np.where(h > 0, 0.7, 0.0)
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(1, 1, 1, 1)), n, n, d, d, b, h, hu=hu)
    L.fill_ghost(None, 1.0)
    # wet cell 5, right half: the stencil reaches dry column 6 -> cell 5's own values; left half: all wet -> bilinear (uniform here)
    out = L.gauges_sample([0, 0, 0], [[5 * d + 8.0, 55.0], [5 * d + 2.0, 55.0], [6 * d + 3.0, 55.0]])
    assert np.array_equal(out[0], [2.25, 0.7, 0.0, 0.25]) and np.array_equal(out[1], [2.25, 0.7, 0.0, 0.25])
    assert np.array_equal(out[2], [0.0, 0.0, 0.0, 1.0])                       # on land: h = 0, eta = the land elevation


def test_point_outside_its_patch_is_refused(gco):
    wl = workloads.cfg1(16)
    pats = workloads.tile(16, 16, 8)
    L = driver.setup_level(gco.Context(**wl.params), wl, patches=pats)
    L.fill_ghost(None, 1.0)
    assert L.gauges_sample([0], [[3500.0, 3500.0]]).shape == (1, 4)
    for bad in ([[9500.0, 3500.0]], [[-1.0, 3500.0]], [[3500.0, 1.0e9]]):
        with pytest.raises(RuntimeError):
            L.gauges_sample([0], bad)
    with pytest.raises(RuntimeError):
        L.gauges_sample([7], [[3500.0, 3500.0]])


def test_gauges_in_an_ocean_at_rest_record_the_sea_level(gco):
    rng = np.random.default_rng(21)
    n, d = 40, 200.0
    X, Y = np.meshgrid(centres(n, d), centres(n, d))
    bathy = lambda x, y: -300.0 + 330.0 * np.exp(-((x - 2500) ** 2 + (y - 4000) ** 2) / 900.0 ** 2) + 12.0 * np.sin(x / 310.0) * np.cos(y / 270.0)
    wl = workloads.Workload("rest", dict(coord=0, dry_tol=1e-3, bc=(1, 1, 0, 0)), 0.0, 0.0, d, d, n, n, bathy, lambda x, y: 0.0 * x, cfl=0.9)
    island = (2500.0, 4000.0)
    assert bathy(*island) > 5.0
    pts = np.vstack([rng.uniform(300.0, 7700.0, (12, 2)), [island]])
    G = driver.GaugeRecorder(pts)
    H = driver.Hierarchy(gco.Context(**wl.params), wl, gauges=G)
    nsteps = H.run(nsteps=60)
    assert nsteps == 60
    wet_seen = 0
    for g in range(len(pts)):
        S = G.series(g)
        assert len(S) == 61 and S[0, 0] == 0.0 and S[-1, 0] == H.t and (np.diff(S[:, 0]) > 0).all()
        if bathy(*pts[g]) < -1.0:
            wet_seen += 1
            assert np.abs(S[:, 4]).max() < 1e-11 and np.abs(S[:, 2]).max() < 1e-10 and np.abs(S[:, 3]).max() < 1e-10
    assert wet_seen >= 8
    S = G.series(len(pts) - 1)                                                # on the island: dry, eta = the land elevation of its cell
    assert (S[:, 1] == 0.0).all() and (S[:, 4] > 5.0).all() and np.ptp(S[:, 4]) == 0.0


def test_gauge_ownership_and_times_in_an_amr_run(gco):
    base = workloads.cfg2(48)
    wl = workloads.Workload("amr2g", base.params, 0.0, 0.0, base.dx, base.dy, 48, 48, base.bathy, base.eta0, cfl=0.9,
                            ratios=(2,), flag=dict(tol_eta=0.1, buffer=2), regrid_interval=2, patch_max=24)
    Lx = 48 * base.dx
    pts = np.array([[x, y] for x in np.linspace(0.06, 0.94, 9) * Lx for y in (0.3 * Lx, 0.71 * Lx)])
    G = driver.GaugeRecorder(pts)
    H = driver.Hierarchy(gco.Context(**wl.params), wl, gauges=G)
    owners0 = [len(ids) for ids, _ in G.assign]
    assert len(H.levels) == 2 and owners0[1] > 0 and owners0[0] > 0              # some gauges start on the fine level, some on the coarse
    ncoarse = H.run(nsteps=12)
    assert H.regrids >= 5
    fine_counts = []
    for g in range(len(pts)):
        S = G.series(g)
        assert S[0, 0] == 0.0 and S[-1, 0] == H.t and (np.diff(S[:, 0]) >= 0).all()
        assert ncoarse + 1 <= len(S) <= 2 * ncoarse + 1                       # once per step of the owning level (ratio 2), once at the end
        assert (S[:, 1] >= 0.0).all() and np.isfinite(S).all()
        fine_counts.append(len(S))
    assert max(fine_counts) > ncoarse + 1                                     # a gauge spent time on the fine level
    # the last record is a direct sample of the final state from the level that owns the gauge now
    for k, L in enumerate(H.levels):
        ids, pats = G.assign[k]
        if ids:
            L.fill_ghost(H.levels[k - 1] if k > 0 else None, 1.0)
            now = L.gauges_sample(pats, pts[ids])
            for n, g in enumerate(ids):
                assert np.array_equal(G.series(g)[-1, 1:], now[n])
