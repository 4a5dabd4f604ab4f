"""Pins of the AMR harness itself (harness/driver.py), which both backends share and which parity therefore cannot check
(VERDICT r1 weak #2).  Neither test goes through Hierarchy to produce its expected value.

 1. A straight-line two-level stepping script -- the order of P:140-146 / Fig. 1 written out call by call, with the ghost-ring
    refresh of DESIGN.md 3.6 -- must reproduce Hierarchy.step bit for bit on the oracle (dt sequence and every cell), on a coarse
    level cut into four patches so that the fine level's coarse-to-fine fill reads ghost cells on patch seams.  Dropping the refresh
    (the two-step-stale ring of round 1) changes the result: the test shows that too, so the bug cannot come back unseen.
 2. Refinement convergence: as the flagging tolerance goes to zero a two-level run approaches the uniformly fine run.
"""
import numpy as np

import workloads
from harness import driver

CART = dict(coord=0, dry_tol=1e-3, bc=(1, 1, 1, 1))


def _workload(n=24, r=2):
    eta0 = lambda X, Y: 1.2 * np.exp(-((X - 1150.0) ** 2 + (Y - 1300.0) ** 2) / (2 * 260.0 ** 2))
    bath = lambda X, Y: -14.0 + 2.0 * np.sin(X / 500.0) * np.cos(Y / 700.0)
    return workloads.Workload("pin", dict(CART), 0.0, 0.0, 100.0, 100.0, n, n, bath, eta0, cfl=0.9, ratios=(r,),
                              flag=dict(tol_eta=-1.0, buffer=0), regrid_interval=10 ** 6, patch_max=32,
                              forced_boxes=((1, 700.0, 1900.0, 800.0, 1700.0, 0.0, 1e30),))


def _straight_line(gco, wl, coarse_patches, fine_patches, nsteps, reflux, refresh_ring=True):
    """P:140-146 for two levels, no regridding, call by call"""
    r = wl.ratios[0]
    ctx = gco.Context(**wl.params)
    C = driver.setup_level(ctx, wl, patches=coarse_patches)
    F = ctx.level_create(2, wl.xlo, wl.ylo, wl.dx / r, wl.dy / r, wl.nx * r, wl.ny * r, r, fine_patches)
    driver.set_initial(F, wl, state=True)
    if reflux:
        C.flux_attach(F)
    # dt_0: probe steps with dt = 0 on both levels, the fine level's speed counted per coarse cell
    C.fill_ghost(None, 1.0); sC = C.step(0.0)["s_over_dx_max"]
    F.fill_ghost(C, 1.0); sF = F.step(0.0)["s_over_dx_max"]
    dt = wl.cfl / max(sC, sF / r)
    dts = []
    for _ in range(nsteps):
        dts.append(dt)
        C.fill_ghost(None, 1.0)                                 # step 1: advance the coarse level
        sC = C.step(dt)["s_over_dx_max"]
        if refresh_ring:
            C.fill_ghost(None, 1.0)                             # ring of the new buffer at the new time
        sF = 0.0
        for s in range(r):                                      # steps 2-3: r substeps of the fine level
            F.fill_ghost(C, s / r)                              #   ghosts from the coarse level at the substep's start time
            sF = max(sF, F.step(dt / r)["s_over_dx_max"])
            if refresh_ring:
                F.fill_ghost(C, (s + 1) / r)
        if reflux:
            C.flux_fixup(F)                                     # step 5 (before averaging: the two touch disjoint cells)
        C.average_down_from(F)                                  # step 4
        dt = wl.cfl / max(sC, sF / r)
    return C, F, dts


def _fine_patches(gco, wl):
    H = driver.Hierarchy(gco.Context(**wl.params), wl)
    p = np.array(H.levels[1].patches)
    H.destroy()
    return p


def test_hierarchy_step_equals_the_straight_line_script(gco):
    wl = _workload()
    n = wl.nx
    quad = np.array([[0, 0, 10, 13], [10, 0, n - 10, 13], [0, 13, 10, n - 13], [10, 13, n - 10, n - 13]], dtype=np.int32)   # seams under the fine patch
    fine = _fine_patches(gco, wl)
    for reflux in (False, True):
        H = driver.Hierarchy(gco.Context(**wl.params), wl, reflux=reflux, patches1=quad)
        assert np.array_equal(H.levels[1].patches, fine)
        dts = []; dt = H.probe()
        for _ in range(6):
            dts.append(dt); dt = H.step(dt)
        C, F, dts2 = _straight_line(gco, wl, quad, fine, 6, reflux)
        assert dts == dts2
        for f in ("h", "hu", "hv"):
            assert np.array_equal(H.levels[0].get_global(f), C.get_global(f)), f
            assert np.array_equal(H.levels[1].get_global(f, fill=0.0), F.get_global(f, fill=0.0)), f
    # the stale ring of round 1 (no refresh after a step) is a different scheme: this pin would see it come back
    C0, F0, _ = _straight_line(gco, wl, quad, fine, 6, True, refresh_ring=False)
    assert not np.array_equal(F0.get_global("h", fill=0.0), F.get_global("h", fill=0.0))
    # ... and the tiling of the coarse level does not matter once the ring is current (one patch = four patches)
    C1, F1, dts1 = _straight_line(gco, wl, np.array([[0, 0, n, n]], dtype=np.int32), fine, 6, True)
    assert dts1 == dts2 and np.array_equal(F1.get_global("h", fill=0.0), F.get_global("h", fill=0.0))


def _run_to(H_or_L, wl, t_end, single=False):
    if not single:
        H_or_L.run(t_end=t_end)
        return
    L, t = H_or_L, 0.0
    dt = driver.probe_dt(L, wl.cfl)
    while t < t_end:
        dt = min(dt, t_end - t)
        L.fill_ghost(None, 1.0)
        st = L.step(dt)
        t += dt
        dt = wl.cfl / st["s_over_dx_max"]


def test_two_level_run_converges_to_the_uniformly_fine_run(gco):
    n, r, T = 24, 2, 40.0
    base = _workload(n, r)
    S = driver.setup_level(gco.Context(**base.params), base, dx=base.dx / r, dy=base.dy / r, nxl=n * r, nyl=n * r)
    _run_to(S, base, T, single=True)
    ref = S.get_global("h") + S.get_global("b")
    refC = ref.reshape(n, r, n, r).mean(axis=(1, 3))
    errs = []
    for tol in (0.3, 0.08, 0.02, 0.002):
        wl = workloads.Workload("conv", base.params, 0.0, 0.0, base.dx, base.dy, n, n, base.bathy, base.eta0, cfl=0.9, ratios=(r,),
                                flag=dict(tol_eta=tol, buffer=2), regrid_interval=2, patch_max=32)
        H = driver.Hierarchy(gco.Context(**wl.params), wl)
        _run_to(H, wl, T)
        C = H.levels[0]
        errs.append(float(np.abs((C.get_global("h") + C.get_global("b")) - refC).max()))
        H.destroy()
    assert errs[0] > 3 * errs[-1] and errs[-1] < 2e-3, errs           # 1.2 m hump: the finest tolerance is within 2 mm of the fine run
    assert all(a >= b * 0.999 for a, b in zip(errs, errs[1:])), errs   # and the error does not grow as the tolerance shrinks


def test_native_bookkeeping_equals_the_python_definition(gco):
    """harness/amr_host.c (clustering, nesting mask, flag unpacking in C) against the Python functions that define them"""
    rng = np.random.default_rng(42)
    for t in range(150):
        ny, nx = (int(v) for v in rng.integers(1, 90, 2))
        fl = np.zeros((ny, nx), dtype=bool)
        for _ in range(int(rng.integers(1, 6))):
            a, b = sorted(int(v) for v in rng.integers(0, ny, 2)); c, d = sorted(int(v) for v in rng.integers(0, nx, 2))
            fl[a:b + 1, c:d + 1] = True
        fl |= rng.random(fl.shape) < rng.choice([0.0, 0.01, 0.1])
        valid = np.ones_like(fl)
        if t % 2:
            valid[:int(rng.integers(0, 4))] = False; valid[:, -int(rng.integers(1, 4)):] = False
        fl &= valid
        kw = dict(valid=valid if t % 3 else None, efficiency=0.7, max_side=int(rng.choice([1, 4, 16, 64])))
        assert driver.cluster(fl, **kw) == driver.cluster_native(fl, **kw), t
    ctx = gco.Context(**CART)
    pats = np.array([[4, 2, 10, 6], [14, 2, 6, 12], [4, 8, 10, 6], [0, 20, 30, 4]], dtype=np.int32)
    L = ctx.level_create(1, 0.0, 0.0, 1.0, 1.0, 30, 24, 1, pats)
    packed = (rng.random(L.ncells) < 0.3).astype(np.uint8)
    for bbox in (None, driver.level_bbox(L), (3, 1, 22, 15)):
        full = (0, 0, L.nxl, L.nyl) if bbox is None else bbox
        assert np.array_equal(driver.nesting_mask(L, bbox=bbox), driver.nesting_mask_native(L, full))
    for bbox in (None, driver.level_bbox(L)):
        full = (0, 0, L.nxl, L.nyl) if bbox is None else bbox
        assert np.array_equal(driver.unpack_cells(L, packed, bbox=bbox), driver.unpack_cells_native(L, packed, full))
    # bathymetry blocks packed natively from the tile cache = bathy_box patch by patch
    wl = workloads.cfg4(120, 60)
    Lb = ctx.level_create(2, wl.xlo, wl.ylo, wl.dx / 5, wl.dy / 5, 600, 300, 5, np.array([[0, 0, 300, 40], [250, 40, 350, 260], [5, 295, 40, 5]], dtype=np.int32))
    got = driver.pack_bathy_native(Lb, wl)
    o = 0
    for i0, j0, nx, ny in Lb.patches:
        a0, a1, c0, c1 = max(i0 - 2, 0), min(i0 + nx + 2, 600), max(j0 - 2, 0), min(j0 + ny + 2, 300)
        want = np.zeros((ny + 4, nx + 4))
        want[c0 - (j0 - 2):c1 - (j0 - 2), a0 - (i0 - 2):a1 - (i0 - 2)] = wl.bathy_box(Lb.dx, Lb.dy, a0, c0, a1 - a0, c1 - c0)
        assert np.array_equal(got[o:o + want.size].reshape(want.shape), want)
        o += want.size
    assert o == got.size
