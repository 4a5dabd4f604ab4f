"""GPU parity of the time-dependent bathymetry (gc_bathy_update): the CUDA path against the
oracle through the C ABI, bit for bit -- the update itself on a tiled wet/dry level (every storage cell, ghost cells included),
a single-level run through a ramp, and config 4's four-level hierarchy started by a seafloor deformation instead of its static
dipole, with regrids while the bed is still moving."""
import numpy as np
import pytest

import workloads
from harness import driver
from test_gpu_amr import lockstep_hierarchies, same_storage

pytestmark = pytest.mark.gpu


def _dome(seed=4):
    rng = np.random.default_rng(seed)
    mx, my, x0, y0, ddx, ddy = 13, 9, 2100.0, 3300.0, 1100.0, 1450.0
    xs, ys = x0 + ddx * np.arange(mx), y0 + ddy * np.arange(my)
    dz = 2.0 * np.exp(-(((xs[None, :] - 9000.0) / 4000.0) ** 2 + ((ys[:, None] - 9000.0) / 3000.0) ** 2)) + 0.05 * rng.standard_normal((my, mx))
    return dict(x0=x0, y0=y0, ddx=ddx, ddy=ddy, dz=dz, t0=20.0, t1=140.0)


def test_bathy_update_and_ramped_run_bit_exact(gc, gco):
    n, dx = 40, 500.0
    bathy = lambda X, Y: -80.0 + 120.0 * X / (n * dx) + 3.0 * np.sin(Y / 3000.0)
    d = _dome()
    levels = []
    for be, tiles in ((gc, workloads.tile(n, n, 8)), (gco, None)):
        wl = workloads.Workload("bathy", dict(coord=0, dry_tol=1e-3, bc=(0, 1, 0, 1)), 0.0, 0.0, dx, dx, n, n, bathy,
                                lambda X, Y: 0.0 * X, cfl=0.9)
        wl.deform = d
        levels.append((wl, driver.setup_level(be.Context(**wl.params), wl, patches=tiles)))
    (wg, Lg), (wo, Lo) = levels
    for w in (0.3, -1.25, 1.0):
        Lg.bathy_update(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], w); Lo.bathy_update(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], w)
        Lg.fill_ghost_b(); Lo.fill_ghost_b()
        assert np.array_equal(Lg.get_global("b"), Lo.get_global("b"))
    for p in range(len(Lg.patches)):                                 # ghost cells of every patch against the one-patch oracle level
        i0, j0, nx, ny = Lg.patches[p]
        assert np.array_equal(Lg.get_field(p, "b")[2:-2, 2:-2], Lo.get_global("b")[j0:j0 + ny, i0:i0 + nx])
    Lg.bathy_update(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], -0.05); Lo.bathy_update(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], -0.05)
    Lg.fill_ghost_b(); Lo.fill_ghost_b()
    hg = driver.run_single_level(Lg, 40, 0.9, wl=wg); ho = driver.run_single_level(Lo, 40, 0.9, wl=wo)
    assert [x for x, _ in hg] == [x for x, _ in ho] and sum(x for x, _ in ho) > 140.0
    for f in ("h", "hu", "hv", "b"):
        assert np.array_equal(Lg.get_global(f), Lo.get_global(f)), f
    assert np.abs(Lo.get_global("hu")).max() > 0.1 and 0 < Lo.wet_mask().sum() < n * n


def test_config4_hierarchy_started_by_a_seafloor_deformation(gc, gco):
    wl = workloads.cfg4_deformation(120, 60, t_rise=400.0)
    wl.patch_max = 60
    wl.forced_boxes = tuple((lv, x0, x1, y0, y1, 0.0, t1) for lv, x0, x1, y0, y1, t0, t1 in wl.forced_boxes)   # coastal boxes on from t = 0
    Hg, Ho = lockstep_hierarchies(gc, gco, wl, 3)
    assert len(Ho.levels) == 4 and Ho.t > 400.0 and Ho.regrids >= 3
    for Lg, Lo in zip(Hg.levels, Ho.levels):
        same_storage(Lg, Lo, fields=("b",))
        assert Lg.rho_applied == Lo.rho_applied
    eta = Ho.levels[0].get_global("h") + Ho.levels[0].get_global("b")
    wet = Ho.levels[0].get_global("h") > 1e-3
    assert np.abs(eta[wet]).max() > 1.0                                # the deformation has raised a tsunami
