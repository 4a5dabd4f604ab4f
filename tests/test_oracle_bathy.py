"""Pins of the oracle's time-dependent bathymetry (oracle/gco_bathy.c; P:52 B(x, y, t), S-20).
The paper says only that deformation files on uniform grids start its tsunamis; what the reading fixes is checked against what
does not depend on it: the library's own linear interpolator, exactness for linear fields, the volume the seafloor displaces,
a uniform uplift (closed form: nothing moves but the datum), a run before t0 (nothing happens at all), and the equivalence of an
instantaneous uplift with a run that starts from the uplifted bed."""
import numpy as np
from scipy.interpolate import RegularGridInterpolator

import workloads
from harness import driver

CART = dict(coord=0, dry_tol=1e-3, bc=(0, 0, 0, 0))


def _level(gco, n=40, dx=500.0, tiles=None, bathy=None):
    b = bathy if bathy is not None else (lambda X, Y: -80.0 + 120.0 * X / (n * dx) + 3.0 * np.sin(Y / 3000.0))   # a beach: wet and dry cells
    wl = workloads.Workload("bathy", dict(CART), 0.0, 0.0, dx, dx, n, n, b, lambda X, Y: 0.0 * X, cfl=0.9)
    L = driver.setup_level(gco.Context(**wl.params), wl, patches=tiles)
    return wl, L


def _dome(mx=13, my=9, x0=2100.0, y0=3300.0, ddx=1100.0, ddy=1450.0, seed=4):
    rng = np.random.default_rng(seed)
    xs, ys = x0 + ddx * np.arange(mx), y0 + ddy * np.arange(my)
    dz = 2.0 * np.exp(-(((xs[None, :] - 9000.0) / 4000.0) ** 2 + ((ys[:, None] - 9000.0) / 3000.0) ** 2)) + 0.05 * rng.standard_normal((my, mx))
    return dict(x0=x0, y0=y0, ddx=ddx, ddy=ddy, dz=dz, t0=0.0, t1=0.0), xs, ys


def test_deformation_is_bilinear_between_nodes_and_zero_outside(gco):
    d, xs, ys = _dome()
    f = RegularGridInterpolator((ys, xs), d["dz"], method="linear", bounds_error=False, fill_value=0.0)
    rng = np.random.default_rng(9)
    pts = np.stack([rng.uniform(0, 20000, 4000), rng.uniform(0, 20000, 4000)], axis=1)
    pts = np.concatenate([pts, [[xs[0], ys[0]], [xs[-1], ys[-1]], [xs[3], ys[2]], [xs[-1] + 1e-6, ys[4]], [xs[2], ys[0] - 1e-6]]])
    got = np.array([gco.deform_at(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], x, y) for x, y in pts])
    want = f(pts[:, ::-1])
    assert np.abs(got - want).max() < 1e-12 and (got[:4000] != 0).sum() > 1000 and got[-1] == 0.0 and got[-2] == 0.0
    assert got[-3] == d["dz"][2, 3] and got[-4] == d["dz"][-1, -1]                 # at a node: the node's value, last node included
    # a field linear in x and y on the nodes is reproduced exactly (a transposed grid or a half-cell shift would not)
    lin = 0.3 + 1.0e-4 * xs[None, :] - 2.5e-4 * ys[:, None]
    for x, y in pts[:200]:
        if xs[0] <= x <= xs[-1] and ys[0] <= y <= ys[-1]:
            assert abs(gco.deform_at(d["x0"], d["y0"], d["ddx"], d["ddy"], lin, x, y) - (0.3 + 1.0e-4 * x - 2.5e-4 * y)) < 1e-12


def test_uplift_moves_bed_and_surface_not_the_water_column(gco):
    """b <- b + w dz on every storage cell of the domain, h unchanged: the surface of a wet cell rises by w dz, and the volume
    lifted above the old surface is the integral of w dz over the wet area"""
    wl, L = _level(gco, tiles=workloads.tile(40, 40, 20))
    d, xs, ys = _dome()
    f = RegularGridInterpolator((ys, xs), d["dz"], method="linear", bounds_error=False, fill_value=0.0)
    xc = (np.arange(40) + 0.5) * 500.0
    X, Y = np.meshgrid(xc, xc)
    dzc = f(np.stack([Y.ravel(), X.ravel()], axis=1)).reshape(40, 40)
    b0, h0 = L.get_global("b"), L.get_global("h")
    L.bathy_update(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], 0.75)
    b1, h1 = L.get_global("b"), L.get_global("h")
    assert np.array_equal(h1, h0) and np.abs((b1 - b0) - 0.75 * dzc).max() < 1e-12
    wet = h0 > 1e-3
    assert 100 < wet.sum() < 1500
    vol = float((((h1 + b1) - (h0 + b0)) * 500.0 ** 2)[wet].sum())
    assert abs(vol - 0.75 * float((dzc * 500.0 ** 2)[wet].sum())) < 1e-9 * abs(vol)
    # ghost cells inside the domain were moved with their source cells: a same-level fill of b changes nothing
    before = [L.get_field(p, "b") for p in range(4)]
    L.fill_ghost_b()
    assert all(np.array_equal(a, L.get_field(p, "b")) for p, a in enumerate(before))


def test_uniform_uplift_only_moves_the_datum(gco):
    """closed form: dz = c everywhere raises bed and surface together; a lake at rest stays at rest, eta = c rho(t)"""
    wl, L = _level(gco, n=32)
    c = 1.7
    wl.deform = dict(x0=-1e5, y0=-1e5, ddx=1e5, ddy=1e5, dz=np.full((4, 4), c), t0=30.0, t1=90.0)
    b0, h0 = L.get_global("b"), L.get_global("h")
    hist = driver.run_single_level(L, 25, wl.cfl, wl=wl)
    t_last_start = sum(dt for dt, _ in hist[:-1])
    assert t_last_start > 90.0
    h, b = L.get_global("h"), L.get_global("b")
    assert np.abs((b - b0) - c).max() < 1e-12
    wet = h0 > 1e-3
    assert np.abs((h + b)[wet] - c).max() < 1e-10 and np.abs(L.get_global("hu")).max() < 1e-9 * 80 * 28 and np.abs(h - h0).max() < 1e-10


def test_nothing_happens_before_t0_and_instantaneous_uplift_equals_starting_from_the_uplifted_bed(gco):
    d, xs, ys = _dome()
    flat = lambda X, Y: -60.0 + 0.0 * X
    # (1) before t0: bit-identical to a run without any deformation
    wlA, LA = _level(gco, bathy=flat); wlB, LB = _level(gco, bathy=flat)
    wlA.deform = dict(d, t0=1e9, t1=2e9)
    hA = driver.run_single_level(LA, 5, 0.9, wl=wlA); hB = driver.run_single_level(LB, 5, 0.9)
    assert [x for x, _ in hA] == [x for x, _ in hB] and np.array_equal(LA.get_global("b"), LB.get_global("b"))
    # (2) uplift at t = 0 in one go = initial data with the bed already uplifted and the same water column
    wlC, LC = _level(gco, bathy=flat); wlD, LD = _level(gco, bathy=flat)
    wlC.deform = dict(d, t0=0.0, t1=0.0)
    LD.bathy_update(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], 1.0); LD.fill_ghost_b()
    hC = driver.run_single_level(LC, 12, 0.9, wl=wlC); hD = driver.run_single_level(LD, 12, 0.9)
    assert [x for x, _ in hC][1:] == [x for x, _ in hD][1:]          # (the probe step of C saw the bed before the uplift)
    eta = LC.get_global("h") + LC.get_global("b")
    assert np.abs(eta).max() > 0.3                                    # a tsunami has been generated ...
    xc = (np.arange(40) + 0.5) * 500.0
    # ... and (3) a ramp over 60 s generates a smaller, later wave than the instantaneous uplift, with the same final bed
    wlE, LE = _level(gco, bathy=flat)
    wlE.deform = dict(d, t0=0.0, t1=60.0)
    driver.run_single_level(LE, 12, 0.9, wl=wlE)
    assert np.abs(LE.get_global("b") - LC.get_global("b")).max() < 1e-12
