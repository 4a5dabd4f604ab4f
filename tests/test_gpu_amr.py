"""GPU parity for the level-transfer rows (A3, A8-A11) and for whole AMR runs: the CUDA path through the C ABI
against the oracle on the same seeded inputs.  Flags, wet masks, patch lists: bit-exact.  State: bit-exact
(the design is bit-reproducible), which implies the BASELINE tolerances (1e-12 per step)."""
import numpy as np
import pytest

import workloads
from harness import driver

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True, params=["by size", "march"])
def sweep_family(request, monkeypatch):
    """The levels of these tests are small, so by size they run on the edge-parallel kernels; forced onto the marching kernels
    they also go through the chains (fine patches that continue each other are walked as one line) next to
    coarse-fine boundaries, with and without flux registers attached.  Same bits either way."""
    from paper_1901_06798_b200 import binding
    if request.param == "march":
        monkeypatch.setitem(binding.DEFAULT_OPTIONS, binding.OPT_SWEEP_FAMILY, binding.SWEEP_MARCH)
    return request.param


def shore_bathy(X, Y):
    return -8.0 + 11.0 * X / 3200.0 + 1.2 * np.sin(Y / 350.0) + 0.6 * np.cos(X / 170.0 + Y / 260.0)


def hump(X, Y):
    return 0.9 * np.exp(-((X - 900.0) ** 2 + (Y - 1500.0) ** 2) / (2 * 320.0 ** 2))


def make_pair(ctx, n, r, fine_patches, coarse_patches=None, params=None):
    dx = 100.0
    cp = np.array([[0, 0, n, n]], dtype=np.int32) if coarse_patches is None else np.asarray(coarse_patches, dtype=np.int32)
    C = ctx.level_create(1, 0.0, 0.0, dx, dx, n, n, 1, cp)
    F = ctx.level_create(2, 0.0, 0.0, dx / r, dx / r, n * r, n * r, r, np.asarray(fine_patches, dtype=np.int32))
    for L in (C, F):
        x = (np.arange(L.nxl) + 0.5) * L.dx
        X, Y = np.meshgrid(x, x)
        b = shore_bathy(X, Y)
        h = np.maximum(0.0, hump(X, Y) - b)
        L.set_global("b", b); L.set_global("h", h); L.set_global("hu", 0.1 * h); L.set_global("hv", -0.05 * h)
        L.fill_ghost_b()
    return C, F


def same_storage(Lg, Lo, fields=("h", "hu", "hv"), which=0):
    for p in range(len(Lo.patches)):
        for f in fields:
            a, c = Lg.get_field(p, f, which), Lo.get_field(p, f, which)
            assert np.array_equal(a, c), (p, f, np.abs(a - c).max())


PARAMS = dict(coord=0, dry_tol=1e-3, bc=(0, 1, 0, 1))
FINE4 = [[16, 24, 40, 32], [56, 24, 24, 56], [16, 56, 40, 24], [96, 100, 16, 12]]       # r = 4, cells of the fine level
COARSE_TILES = [[0, 0, 16, 32], [16, 0, 16, 12], [16, 12, 16, 20]]


@pytest.mark.parametrize("coarse_patches", [None, COARSE_TILES])
def test_coarse_ghost_fill_average_down_and_regrid_transfer(gc, gco, coarse_patches):
    n, r = 32, 4
    pairs = [make_pair(b.Context(**PARAMS), n, r, FINE4, coarse_patches) for b in (gc, gco)]
    (Cg, Fg), (Co, Fo) = pairs
    # two coarse steps so that the OLD and NEW coarse buffers differ
    for C in (Cg, Co):
        dt = driver.probe_dt(C, 0.8)
        for _ in range(2):
            C.fill_ghost(None, 1.0); st = C.step(dt); dt = 0.8 / st["s_over_dx_max"]
        C.fill_ghost(None, 1.0)
    same_storage(Cg, Co)
    for alpha in (0.0, 0.25, 0.75, 1.0):
        Fg.fill_ghost(Cg, alpha); Fo.fill_ghost(Co, alpha)
        same_storage(Fg, Fo)
    # A11: new fine level partly over the old one, partly over coarse cells only
    new_p = [[24, 16, 48, 40], [72, 32, 16, 64], [8, 72, 32, 24]]
    news = []
    for (C, F), b in zip(pairs, (gc, gco)):
        N = C.ctx.level_create(2, 0.0, 0.0, 25.0, 25.0, n * r, n * r, r, np.asarray(new_p, dtype=np.int32))
        x = (np.arange(N.nxl) + 0.5) * N.dx
        X, Y = np.meshgrid(x, x)
        N.set_global("b", shore_bathy(X, Y)); N.fill_ghost_b()
        N.init_from(F, C)
        news.append(N)
    same_storage(news[0], news[1])
    assert np.array_equal(news[0].wet_mask(), news[1].wet_mask())
    for (C, F), N in zip(pairs, news):
        N2 = C.ctx.level_create(2, 0.0, 0.0, 25.0, 25.0, n * r, n * r, r, np.asarray(new_p, dtype=np.int32))
        N2.set_global("b", N.get_global("b", fill=0.0)); N2.fill_ghost_b()
        N2.init_from(None, C)
        N.extra = N2
    same_storage(news[0].extra, news[1].extra)
    # A9: fine steps then average down (wet and dry fine cells under one coarse cell occur along the shoreline)
    for C, F in pairs:
        F.fill_ghost(C, 1.0)
        F.step(0.2)
        C.average_down_from(F)
    same_storage(Fg, Fo)
    same_storage(Cg, Co)
    assert np.array_equal(Cg.wet_mask(), Co.wet_mask())


def test_average_down_spherical_weights(gc, gco):
    wl = workloads.cfg3(32)
    res = []
    for b in (gc, gco):
        ctx = b.Context(**wl.params)
        C = driver.setup_level(ctx, wl)
        F = driver.setup_level(ctx, wl, level=2, dx=wl.dx / 4, dy=wl.dy / 4, nxl=128, nyl=128, ratio=4,
                               patches=np.array([[32, 32, 64, 48], [32, 80, 32, 16]], dtype=np.int32))
        C.fill_ghost(None, 1.0); F.fill_ghost(C, 1.0)
        F.step(1.0); F.fill_ghost(C, 1.0); F.step(1.0)
        C.average_down_from(F)
        res.append((C, F))
    same_storage(res[0][0], res[1][0])
    same_storage(res[0][1], res[1][1])


def test_flags_bit_exact(gc, gco):
    n = 48
    rng = np.random.default_rng(4)
    x = (np.arange(n) + 0.5) * 100.0
    X, Y = np.meshgrid(x, x)
    b = -6.0 + 9.0 * X / 4800.0 + 0.8 * np.sin(Y / 500.0)
    eta = 0.4 * np.exp(-((X - 1500.0) ** 2 + (Y - 2000.0) ** 2) / (2 * 500.0 ** 2)) + 0.004 * rng.standard_normal((n, n))
    h = np.maximum(0.0, eta - b)
    pats = np.array([[0, 0, 16, 48], [16, 0, 32, 10], [16, 10, 12, 38], [28, 10, 20, 24], [28, 34, 20, 14]], dtype=np.int32)
    Ls = []
    for bk in (gc, gco):
        L = bk.Context(**PARAMS).level_create(1, 0.0, 0.0, 100.0, 100.0, n, n, 1, pats)
        L.set_global("b", b); L.set_global("h", h); L.set_global("hu", 0 * h); L.set_global("hv", 0 * h)
        L.fill_ghost_b(); L.fill_ghost(None, 1.0)
        Ls.append(L)
    boxes = [(3000.0, 3600.0, 400.0, 900.0, 10.0, 20.0), (100.0, 250.0, 4000.0, 4700.0, 0.0, 5.0)]
    nonzero = 0
    for kw in (dict(tol_eta=0.05), dict(tol_eta=0.05, offshore_only=1, buffer=2), dict(tol_slope=0.004, buffer=1),
               dict(tol_eta=0.2, tol_slope=0.01, buffer=5, boxes=boxes, t=12.0), dict(boxes=boxes, t=2.0, buffer=3),
               dict(tol_eta=10.0)):
        (fg, ng), (fo, no) = Ls[0].flag(**kw), Ls[1].flag(**kw)
        assert ng == no and np.array_equal(fg, fo), kw
        nonzero += no > 0
    assert nonzero >= 5


def lockstep_hierarchies(gc, gco, wl, nsteps, **kw):
    Hg = driver.Hierarchy(gc.Context(**wl.params), wl, **kw)
    Ho = driver.Hierarchy(gco.Context(**wl.params), wl, **kw)
    dtg, dto = Hg.probe(), Ho.probe()
    for n in range(nsteps):
        assert dtg == dto, (n, dtg, dto)
        dtg, dto = Hg.step(dtg), Ho.step(dto)
        assert len(Hg.levels) == len(Ho.levels)
        for Lg, Lo in zip(Hg.levels, Ho.levels):
            assert np.array_equal(Lg.patches, Lo.patches), n
            assert np.array_equal(Lg.wet_mask(), Lo.wet_mask()), n
            same_storage(Lg, Lo)
    assert len(Hg.flag_log) == len(Ho.flag_log)
    for (kg, tg, fg), (ko, to, fo) in zip(Hg.flag_log, Ho.flag_log):
        assert kg == ko and tg == to and np.array_equal(fg, fo)
    return Hg, Ho


@pytest.mark.parametrize("reflux", [True, False])
def test_two_level_wet_dry_run_with_regrids(gc, gco, reflux):
    base = workloads.cfg2(48)
    wl = workloads.Workload("amr2", base.params, 0.0, 0.0, base.dx, base.dy, 48, 48, base.bathy, base.eta0, cfl=0.9,
                            ratios=(2,), flag=dict(tol_eta=0.1, buffer=2), regrid_interval=2, patch_max=24)
    Hg, Ho = lockstep_hierarchies(gc, gco, wl, 12, reflux=reflux)
    assert len(Hg.levels) == 2 and Hg.regrids >= 5
    assert abs(Hg.composite_mass() - Ho.composite_mass()) <= 1e-13 * abs(Ho.composite_mass())


def test_set_patches_and_patchwise_initialisation(gc, gco):
    """gc_level_set_patches: every patch's storage-shaped block in one call.  Random data on a fine level whose patches touch the
    domain edge and each other: every in-level cell of every patch, ghost cells included, takes its block's value, cells outside
    the level are the boundary fill's.  Then driver.set_initial's patch-by-patch path (used at every regrid) on both backends."""
    n, r = 32, 4
    fine = np.array([[0, 0, 40, 32], [40, 0, 24, 56], [0, 32, 40, 24], [112, 116, 16, 12]], dtype=np.int32)   # two touch x = 0, y = 0; one the far corner
    rng = np.random.default_rng(17)
    levels = []
    for b in (gc, gco):
        ctx = b.Context(**PARAMS)
        levels.append(ctx.level_create(2, 0.0, 0.0, 25.0, 25.0, n * r, n * r, r, fine))
    Lg, Lo = levels
    sizes = [(nx + 4) * (ny + 4) for _, _, nx, ny in fine]
    for f in ("h", "hu", "hv", "b"):
        packed = rng.uniform(0.5, 2.0, sum(sizes))
        Lg.set_patches(f, packed); Lo.set_patches(f, packed)
        o = 0
        for p, (i0, j0, nx, ny) in enumerate(fine):
            blk = packed[o:o + sizes[p]].reshape(ny + 4, nx + 4); o += sizes[p]
            gi = i0 - 2 + np.arange(nx + 4); gj = j0 - 2 + np.arange(ny + 4)
            inside = np.outer((gj >= 0) & (gj < n * r), (gi >= 0) & (gi < n * r))
            got = Lg.get_field(p, f)
            assert np.array_equal(got[inside], blk[inside]), (f, p)
            assert np.array_equal(Lo.get_field(p, f)[inside], blk[inside]), (f, p)
    # the initialisation path of every regrid: analytic bathymetry and state patch by patch, then the ghost fill of b
    base = workloads.cfg2(n * r)
    wl = workloads.Workload("fine", base.params, 0.0, 0.0, 25.0, 25.0, n * r, n * r, base.bathy, base.eta0)
    assert Lg.nxl * Lg.nyl > 2 * Lg.ncells                                # the patch-by-patch branch
    for L in (Lg, Lo):
        driver.set_initial(L, wl, state=True)
    same_storage(Lg, Lo, fields=("b", "h", "hu", "hv"))
    x = (np.arange(n * r) + 0.5) * 25.0
    X, Y = np.meshgrid(x, x)
    want = np.asarray(base.bathy(X, Y))
    got = Lg.get_global("b", fill=np.nan)
    cov = ~np.isnan(got)
    assert cov.sum() == Lg.ncells and np.array_equal(got[cov], want[cov])


def test_two_level_run_with_manning_friction(gc, gco):
    """friction inside the AMR recursion: every level applies it after its own y-sweep with its own dt"""
    base = workloads.cfg2(48)
    wl = workloads.Workload("amr2f", dict(base.params, manning_n=0.025), 0.0, 0.0, base.dx, base.dy, 48, 48, base.bathy, base.eta0,
                            cfl=0.9, ratios=(2,), flag=dict(tol_eta=0.1, buffer=2), regrid_interval=2, patch_max=24)
    Hg, Ho = lockstep_hierarchies(gc, gco, wl, 12, reflux=True)
    assert len(Hg.levels) == 2 and Hg.regrids >= 5


def test_three_levels_middle_level_is_coarse_and_fine_side(gc, gco):
    base = workloads.cfg1(24)
    wl = workloads.Workload("amr3", base.params, 0.0, 0.0, base.dx, base.dy, 24, 24, base.bathy, base.eta0, cfl=0.9,
                            ratios=(2, 3), flag=dict(tol_eta=0.25, buffer=1), regrid_interval=2, patch_max=18)
    Hg, Ho = lockstep_hierarchies(gc, gco, wl, 6)
    assert len(Hg.levels) == 3
    m0 = Ho.composite_mass()
    assert abs(Hg.composite_mass() - m0) <= 1e-13 * m0


def test_config3_reduced_spherical_amr(gc, gco):
    """config 3 recipe at 64 x 64 coarse cells, ratio 4, regrid every 4 coarse steps, 10 coarse steps"""
    wl = workloads.cfg3(64)
    wl.patch_max = 32
    Hg, Ho = lockstep_hierarchies(gc, gco, wl, 10)
    assert len(Hg.levels) == 2 and Hg.regrids >= 2 and Hg.levels[1].ncells > 1000


def test_flux_fixup_requires_attach_and_nesting_errors(gc):
    ctx = gc.Context(**PARAMS)
    C, F = make_pair(ctx, 16, 2, [[12, 8, 8, 8]], coarse_patches=[[0, 0, 8, 16]])   # fine patch beyond the coarse level
    with pytest.raises(RuntimeError):
        C.flux_fixup(F)
    with pytest.raises(RuntimeError):
        F.fill_ghost(C, 1.0)
    with pytest.raises(RuntimeError):
        C.average_down_from(F)


def test_step_accum_leaves_the_maximum_and_the_sums_of_a_run_of_steps(gc):
    """gc_level_step_accum / gc_level_stats_reset (the subcycled levels of the recursion are not waited for step by step): same state
    as gc_level_step, and the statistics read afterwards are the maximum (s_over_dx_max), the sums (n_clipped, clipped_mass) and the
    OR (nan_seen) of the steps since the reset"""
    wl = workloads.cfg2(96)
    La = driver.setup_level(gc.Context(**wl.params), wl, patches=workloads.tile(96, 96, 32))
    Lb = driver.setup_level(gc.Context(**wl.params), wl, patches=workloads.tile(96, 96, 32))
    La.fill_ghost(None, 1.0)
    dt = 0.8 / La.step(0.0)["s_over_dx_max"]
    Lb.fill_ghost(None, 1.0); Lb.step(0.0)
    Lb.stats_reset()
    assert Lb.stats()["s_over_dx_max"] == 0.0
    sd, nc, cm = [], 0, 0.0
    for k in range(30):
        La.fill_ghost(None, 1.0); Lb.fill_ghost(None, 1.0)
        st = La.step(dt)
        Lb.step_accum(dt)
        sd.append(st["s_over_dx_max"]); nc += st["n_clipped"]; cm += st["clipped_mass"]
    sb = Lb.stats()
    assert sb["s_over_dx_max"] == max(sd) and max(sd) > min(sd) and sb["n_clipped"] == nc and sb["nan_seen"] == 0
    assert abs(sb["clipped_mass"] - cm) <= 1e-12 * abs(cm) + 1e-300
    for f in ("h", "hu", "hv"):
        assert np.array_equal(La.get_global(f), Lb.get_global(f))
    Lb.stats_reset()
    assert Lb.stats()["s_over_dx_max"] == 0.0 and Lb.stats()["n_clipped"] == 0
