"""Pins for the oracle's level-transfer operations (oracle/gco_amr.c, gco_flux.c) and for the host AMR driver:
coarse-to-fine interpolation is exact for fields linear in space and time; the ocean at rest stays at rest
through ghost fill, regrid transfer and averaging; a fine level covering the whole domain reproduces the
single-level fine run bitwise and its average-down is the block mean; the flux registers make the composite
mass of a closed basin constant across a coarse-fine interface; flags against scipy's binary dilation
(P:136); clustering covers every flagged cell with disjoint boxes."""
import numpy as np
import pytest
from scipy import ndimage

import workloads
from harness import driver

G = 9.81
CART = dict(coord=0, dry_tol=1e-3, bc=(1, 1, 1, 1))


def two_levels(ctxs, n, r, fine_patches, bfun, etafun, dx=100.0, params=CART, state_fine=True):
    """coarse n x n level + fine level with the given patches (fine cell units); analytic b, eta at cell centres"""
    out = []
    for ctx in ctxs:
        C = ctx.level_create(1, 0.0, 0.0, dx, dx, n, n, 1, np.array([[0, 0, n, n]], dtype=np.int32))
        F = ctx.level_create(2, 0.0, 0.0, dx / r, dx / r, n * r, n * r, r, np.asarray(fine_patches, dtype=np.int32))
        for L in (C, F):
            x = (np.arange(L.nxl) + 0.5) * L.dx
            X, Y = np.meshgrid(x, x)
            b = bfun(X, Y)
            L.set_global("b", b)
            if L is C or state_fine:
                h = np.maximum(0.0, etafun(X, Y) - b)
                L.set_global("h", h); L.set_global("hu", 0 * h); L.set_global("hv", 0 * h)
            L.fill_ghost_b()
        out.append((C, F))
    return out


def test_interpolation_exact_for_linear_fields_in_space_and_time(gco):
    n, r = 12, 4
    bfun = lambda X, Y: -50.0 + 0.0 * X
    eta_lin = lambda X, Y: 0.002 * X - 0.001 * Y + 1.0
    fp = [[8, 12, 16, 20]]                      # fine patch strictly inside: every ghost comes from the coarse level
    (C, F), = two_levels([gco.Context(**CART)], n, r, fp, bfun, eta_lin, state_fine=False)
    # eta linear in x and y, uniform velocity (0.3, -0.2): minmod of two equal one-sided differences is the exact slope
    xc = (np.arange(n) + 0.5) * 100.0
    X, Y = np.meshgrid(xc, xc)
    h_old = eta_lin(X, Y) + 50.0
    C.set_global("h", h_old); C.set_global("hu", 0.3 * h_old); C.set_global("hv", -0.2 * h_old)
    C.fill_ghost(None, 1.0)
    F.fill_ghost(C, 1.0)
    xf = (np.arange(-2, 16 + 2) + 8 + 0.5) * 25.0
    yf = (np.arange(-2, 20 + 2) + 12 + 0.5) * 25.0
    XF, YF = np.meshgrid(xf, yf)
    h = F.get_field(0, "h"); hu = F.get_field(0, "hu"); hv = F.get_field(0, "hv")
    ghost = np.ones_like(h, dtype=bool); ghost[2:-2, 2:-2] = False
    want = eta_lin(XF, YF) + 50.0
    assert np.abs(h - want)[ghost].max() < 1e-12 * 60.0
    assert np.abs(hu - 0.3 * want)[ghost].max() < 1e-12 * 60.0
    assert np.abs(hv + 0.2 * want)[ghost].max() < 1e-12 * 60.0
    # a transposed / sign-flipped offset would give errors of order slope * dx_f = 0.05


def test_time_interpolation_is_linear(gco):
    n, r = 8, 2
    bfun = lambda X, Y: -20.0 + 0.0 * X
    (C, F), = two_levels([gco.Context(**CART)], n, r, [[4, 4, 8, 8]], bfun, lambda X, Y: 0.0 * X, state_fine=False)
    C.fill_ghost(None, 1.0)
    dt = 0.9 / C.step(0.0)["s_over_dx_max"]
    # old: flat; one real step keeps it flat; then overwrite the NEW buffer with a raised flat state
    C.step(dt)
    C.set_global("h", np.full((n, n), 24.0)); C.fill_ghost(None, 1.0)
    for alpha in (0.0, 0.25, 0.5, 1.0):
        F.fill_ghost(C, alpha)
        h = F.get_field(0, "h")
        assert np.allclose(h[0, 2:-2], 20.0 + 4.0 * alpha, rtol=0, atol=1e-13)


def rough_bathy(seed=5, amp=30.0):
    rng = np.random.default_rng(seed)
    ph = rng.uniform(0, 2 * np.pi, 6)
    def b(X, Y):
        s = -300.0 + 0.0 * X
        for k in range(6):
            s = s + amp / 6 * np.cos((k + 1) * X / 700.0 + ph[k]) * np.sin((6 - k) * Y / 900.0 + ph[5 - k])
        return s
    return b


def test_ocean_at_rest_through_fill_regrid_and_average(gco):
    n, r = 16, 4
    bfun = rough_bathy()
    rest = lambda X, Y: 0.0 * X
    (C, F), = two_levels([gco.Context(**CART)], n, r, [[8, 8, 24, 16], [32, 8, 16, 32]], bfun, rest, state_fine=False)
    C.fill_ghost(None, 1.0)
    F.init_from(None, C)
    F.fill_ghost(C, 1.0)
    for p in range(2):
        eta = F.get_field(p, "h") + F.get_field(p, "b")
        assert np.abs(eta).max() < 1e-12 * 330.0
        assert np.abs(F.get_field(p, "hu")).max() == 0.0
    C.average_down_from(F)
    assert np.abs(C.get_global("h") + C.get_global("b")).max() < 1e-12 * 330.0


def test_lake_at_rest_two_level_run_with_regrids(gco):
    wl = workloads.Workload("rest", dict(CART), 0.0, 0.0, 100.0, 100.0, 24, 24, rough_bathy(7), lambda X, Y: 0.0 * X,
                            cfl=0.9, ratios=(2,), flag=dict(tol_eta=-1.0, buffer=1), regrid_interval=2, patch_max=16,
                            forced_boxes=((1, 600.0, 1500.0, 500.0, 1800.0, 0.0, 1e30),))
    H = driver.Hierarchy(gco.Context(**wl.params), wl)
    assert len(H.levels) == 2
    H.run(nsteps=8)
    assert H.regrids >= 3
    for L in H.levels:
        hu, hv, h = L.get_global("hu", fill=0.0), L.get_global("hv", fill=0.0), L.get_global("h", fill=0.0)
        c = np.sqrt(G * 330.0)
        assert max(np.abs(hu).max(), np.abs(hv).max()) < 1e-11 * 330.0 * c
        eta = L.get_global("h") + L.get_global("b")
        assert np.nanmax(np.abs(eta)) < 1e-11 * 330.0


def test_full_cover_fine_level_equals_single_level_run(gco):
    """subcycling driver pin: the fine level covers the domain, so it never sees the coarse level; it must equal a
    single-level run with the same dt sequence bit for bit, and the coarse level is its block mean after each step"""
    n, r = 12, 2
    wl = workloads.cfg1(n)
    wl2 = workloads.Workload("cover", wl.params, 0.0, 0.0, wl.dx, wl.dy, n, n, wl.bathy, wl.eta0, cfl=0.9, ratios=(r,),
                             flag=dict(tol_eta=-1.0, buffer=0), regrid_interval=1000, patch_max=64,
                             forced_boxes=((1, -1e30, 1e30, -1e30, 1e30, 0.0, 1e30),))
    H = driver.Hierarchy(gco.Context(**wl2.params), wl2, reflux=True)
    assert len(H.levels) == 2 and H.levels[1].ncells == (n * r) ** 2
    S = driver.setup_level(gco.Context(**wl.params), wl, dx=wl.dx / r, dy=wl.dy / r, nxl=n * r, nyl=n * r)
    dt = H.probe()
    for _ in range(5):
        dtn = H.step(dt)
        for _ in range(r):
            S.fill_ghost(None, 1.0); S.step(dt / r)
        for f in ("h", "hu", "hv"):
            assert np.array_equal(H.levels[1].get_global(f), S.get_global(f))
        hf = S.get_global("h")
        blockmean = hf.reshape(n, r, n, r).mean(axis=(1, 3))
        assert np.abs(H.levels[0].get_global("h") - blockmean).max() < 1e-12 * 4000.0
        dt = dtn


@pytest.mark.parametrize("reflux", [True, False])
def test_flux_registers_conserve_composite_mass(gco, reflux):
    """closed Cartesian basin, flat bottom, a hump that crosses the coarse-fine interface of a static fine patch"""
    n, r = 20, 2
    eta0 = lambda X, Y: 1.5 * np.exp(-((X - 900.0) ** 2 + (Y - 1000.0) ** 2) / (2 * 250.0 ** 2))
    wl = workloads.Workload("mass", dict(CART), 0.0, 0.0, 100.0, 100.0, n, n, lambda X, Y: -12.0 + 0.0 * X, eta0,
                            cfl=0.9, ratios=(r,), flag=dict(tol_eta=-1.0, buffer=0), regrid_interval=1000, patch_max=16,
                            forced_boxes=((1, 500.0, 1300.0, 600.0, 1400.0, 0.0, 1e30),))
    H = driver.Hierarchy(gco.Context(**wl.params), wl, reflux=reflux)
    assert len(H.levels) == 2 and len(H.levels[1].patches) >= 1
    m0 = H.composite_mass()
    drift = []
    H.run(nsteps=30, record=lambda n_, dt, h: drift.append(abs(h.composite_mass() - m0) / m0))
    if reflux:
        assert max(drift) < 5e-14, max(drift)
    else:
        assert max(drift) > 1e-9, max(drift)      # the pin is sensitive: without step 5 mass is not conserved


def test_flags_against_binary_dilation(gco):
    n = 20
    rng = np.random.default_rng(11)
    xc = (np.arange(n) + 0.5) * 100.0
    X, Y = np.meshgrid(xc, xc)
    b = -5.0 + 8.0 * X / 2000.0
    eta = 0.3 * np.exp(-((X - 500.0) ** 2 + (Y - 900.0) ** 2) / (2 * 200.0 ** 2)) + 0.02 * rng.standard_normal((n, n))
    h = np.maximum(0.0, eta - b)
    ctx = gco.Context(**CART)
    pats = np.array([[0, 0, 12, 20], [12, 0, 8, 8], [12, 8, 8, 12]], dtype=np.int32)
    L = ctx.level_create(1, 0.0, 0.0, 100.0, 100.0, n, n, 1, pats)
    L.set_global("b", b); L.set_global("h", h); L.set_global("hu", 0 * h); L.set_global("hv", 0 * h)
    L.fill_ghost_b(); L.fill_ghost(None, 1.0)
    box = (1500.0, 1800.0, 100.0, 400.0, 5.0, 10.0)
    for bw in (0, 1, 3):
        for t in (0.0, 7.0):
            packed, nf = L.flag(tol_eta=0.05, offshore_only=1, buffer=bw, boxes=[box], t=t)
            got = driver.unpack_cells(L, packed).astype(bool)
            raw = (h > 1e-3) & (b < 0.0) & (np.abs(h + b) > 0.05)
            if t == 7.0:
                raw |= (X >= box[0]) & (X <= box[1]) & (Y >= box[2]) & (Y <= box[3])
            want = ndimage.binary_dilation(raw, structure=np.ones((2 * bw + 1, 2 * bw + 1), dtype=bool)) if bw else raw
            assert np.array_equal(got, want) and nf == want.sum()
    # slope criterion on a plane: central difference per cell = 0.5 * |eta(i+1) - eta(i-1)|
    L.set_global("h", (0.01 * X / 100.0 + 20.0)); L.set_global("b", np.full((n, n), -20.0)); L.fill_ghost_b(); L.fill_ghost(None, 1.0)
    assert L.flag(tol_slope=0.0099)[1] == n * n - 2 * n       # wall ghosts mirror: the slope vanishes... only in the two edge columns
    assert L.flag(tol_slope=0.0101)[1] == 0


def test_cluster_covers_flags_with_disjoint_valid_boxes():
    rng = np.random.default_rng(2)
    fl = np.zeros((40, 50), dtype=bool)
    fl[5:12, 4:30] = True; fl[20:35, 10:14] = True; fl[30:33, 40:48] = True
    fl |= rng.random(fl.shape) < 0.01
    valid = np.ones_like(fl); valid[0:3, :] = False
    fl &= valid
    boxes = driver.cluster(fl, valid=valid, efficiency=0.7, max_side=16)
    cover = np.zeros_like(fl, dtype=int)
    for i0, j0, nx, ny in boxes:
        assert nx <= 16 and ny <= 16 and valid[j0:j0 + ny, i0:i0 + nx].all()
        cover[j0:j0 + ny, i0:i0 + nx] += 1
    assert cover.max() == 1 and (cover[fl] == 1).all()
    assert fl.sum() / (cover > 0).sum() > 0.5
    assert boxes == sorted(boxes, key=lambda b: (b[1], b[0]))


def _run_hierarchy(gco, wl, n, **kw):
    H = driver.Hierarchy(gco.Context(**wl.params), wl, **kw)
    dts = []; dt = H.probe()
    for _ in range(n):
        dts.append(dt); dt = H.step(dt)
    return H, dts


@pytest.mark.parametrize("case", ["four_levels_fixed_boxes", "two_levels_wave_following", "three_levels", "four_levels_no_reflux"])
def test_keeping_a_level_whose_regrid_reproduces_it_changes_no_bit(gco, monkeypatch, case):
    """every ghost cell is rewritten before it is read (a level's ghost ring is refilled right after its own step, at
    the new state's time), and the regrid transfer copies every interior cell of an unchanged level -- so a level whose regrid
    reproduces its patch list may simply stay.  With the switch on and off: same dt sequence, same patch lists, same flagging passes,
    every interior cell of every level identical."""
    kw = {}
    if case.startswith("four_levels"):
        wl = workloads.cfg4(120, 60); wl.patch_max = 60
        wl.forced_boxes = tuple((lv, x0, x1, y0, y1, 0.0, t1) for lv, x0, x1, y0, y1, t0, t1 in wl.forced_boxes)
        n = 3
        kw = dict(reflux=not case.endswith("no_reflux"))
    elif case == "two_levels_wave_following":
        base = workloads.cfg2(48)
        wl = workloads.Workload("amr2", base.params, 0.0, 0.0, base.dx, base.dy, 48, 48, base.bathy, base.eta0, cfl=0.9,
                                ratios=(2,), flag=dict(tol_eta=0.1, buffer=2), regrid_interval=2, patch_max=24)
        n = 12
    else:
        base = workloads.cfg1(24)
        wl = workloads.Workload("amr3", base.params, 0.0, 0.0, base.dx, base.dy, 24, 24, base.bathy, base.eta0, cfl=0.9,
                                ratios=(2, 3), flag=dict(tol_eta=0.25, buffer=1), regrid_interval=2, patch_max=18)
        n = 8
    Ha, da = _run_hierarchy(gco, wl, n, keep_unchanged=True, **kw)
    Hb, db = _run_hierarchy(gco, wl, n, keep_unchanged=False, **kw)
    assert Hb.kept == 0 and da == db and Ha.regrids == Hb.regrids and len(Ha.levels) == len(Hb.levels)
    if case.startswith("four_levels"):
        assert Ha.kept >= 30 and len(Ha.levels) == 4                         # the fixed-box levels came back unchanged every time
    for La, Lb in zip(Ha.levels, Hb.levels):
        assert np.array_equal(La.patches, Lb.patches)
        for f in ("h", "hu", "hv", "b"):
            assert np.array_equal(La.get_global(f, fill=0.0), Lb.get_global(f, fill=0.0)), (case, La.level, f)
    # the keeping run does not flag again a level whose flags can only come from unchanged forced boxes: its log is a sub-sequence
    # of the other's, and every pass it did run saw the same flags
    ref = {}
    for kb, tb, fb in Hb.flag_log:
        ref.setdefault((kb, tb), []).append(fb)                # (a level can be flagged twice at one time: its own regrid, then a coarser level's)
    assert 0 < len(Ha.flag_log) <= len(Hb.flag_log)
    for ka, ta, fa in Ha.flag_log:
        assert any(np.array_equal(fa, fb) for fb in ref[(ka, ta)])
