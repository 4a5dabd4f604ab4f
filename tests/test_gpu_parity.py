"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element on the same
seeded inputs.  Bars (BASELINE.json north_star): wet masks bit-exact; dt within 1e-14 relative per step;
h, hu, hv within 1e-12 relative per step and 1e-9 max|eta| at the end.  The design is bit-reproducible
(fused multiply-adds only where DESIGN.md 3 writes them, on both sides), so the expected difference is exactly 0 and
the tests assert that where noted."""
import numpy as np
import pytest

import workloads
from harness import driver

pytestmark = pytest.mark.gpu
G = 9.81


@pytest.fixture(autouse=True, params=["edge", "march"])
def sweep_mode(request, monkeypatch):
    """Both sweep kernel families (edge-parallel tiles k_sweep / line marching k_marchp) must give the oracle's
    bits; the library picks one by level size unless gc_ctx_set_option says otherwise (read when a level is created)."""
    from paper_1901_06798_b200 import binding
    fam = binding.SWEEP_EDGE if request.param == "edge" else binding.SWEEP_MARCH
    monkeypatch.setitem(binding.DEFAULT_OPTIONS, binding.OPT_SWEEP_FAMILY, fam)
    return request.param


def unpack(L, packed):
    """interior-packed per-patch array -> level-global 2-D array"""
    out = np.full((L.nyl, L.nxl), 255, dtype=packed.dtype)
    o = 0
    for i0, j0, nx, ny in L.patches:
        out[j0:j0 + ny, i0:i0 + nx] = packed[o:o + nx * ny].reshape(ny, nx)
        o += nx * ny
    return out


def lockstep(Lg, Lo, nsteps, cfl, eta_scale, exact=True, hmax=None):
    """Advance both backends with their own dt control; compare every step."""
    dtg = driver.probe_dt(Lg, cfl)
    dto = driver.probe_dt(Lo, cfl)
    worst = dict(dt=0.0, h=0.0, hu=0.0, hv=0.0)
    for n in range(nsteps):
        assert abs(dtg - dto) <= 1e-14 * dto, (n, dtg, dto)
        Lg.fill_ghost(None, 1.0); Lo.fill_ghost(None, 1.0)
        sg = Lg.step(dtg); so = Lo.step(dto)
        worst["dt"] = max(worst["dt"], abs(dtg - dto) / dto)
        assert sg["n_clipped"] == so["n_clipped"], n
        assert abs(sg["clipped_mass"] - so["clipped_mass"]) <= 1e-12 * abs(so["clipped_mass"]) + 1e-300
        assert sg["nan_seen"] == 0 and so["nan_seen"] == 0
        assert abs(sg["s_over_dx_max"] - so["s_over_dx_max"]) <= 1e-14 * so["s_over_dx_max"]
        assert np.array_equal(unpack(Lg, Lg.wet_mask()), unpack(Lo, Lo.wet_mask())), "wet mask differs at step %d" % n
        ho = Lo.get_global("h")
        hscale = np.nanmax(np.abs(ho))
        mscale = max(np.nanmax(np.abs(Lo.get_global("hu"))), np.nanmax(np.abs(Lo.get_global("hv"))), eta_scale * np.sqrt(G * hscale))
        for f, sc in (("h", hscale), ("hu", mscale), ("hv", mscale)):
            a, c = Lg.get_global(f), Lo.get_global(f)
            assert np.array_equal(np.isnan(a), np.isnan(c))
            d = np.nanmax(np.abs(a - c))
            worst[f] = max(worst[f], d / sc)
            assert d <= 1e-12 * sc, (f, n, d, sc)
        dtg = cfl / sg["s_over_dx_max"]; dto = cfl / so["s_over_dx_max"]
    if exact:
        assert worst["h"] == 0.0 and worst["hu"] == 0.0 and worst["hv"] == 0.0 and worst["dt"] == 0.0, worst
    return worst


def both(gc, gco, wl, patches_g=None, patches_o=None, **kw):
    cg = gc.Context(**wl.params); co = gco.Context(**wl.params)
    Lg = driver.setup_level(cg, wl, patches=patches_g, **kw)
    Lo = driver.setup_level(co, wl, patches=patches_o, **kw)
    return Lg, Lo


def test_config1_100_steps(gc, gco):
    wl = workloads.cfg1()
    Lg, Lo = both(gc, gco, wl)
    lockstep(Lg, Lo, 100, wl.cfl, 1.0)
    assert abs(Lg.mass() - Lo.mass()) <= 1e-13 * Lo.mass()
    for f in ("h", "hu", "hv", "b"):  # ghost cells too (physical boundary A4)
        Lg.fill_ghost(None, 1.0); Lo.fill_ghost(None, 1.0)
        assert np.array_equal(Lg.get_field(0, f), Lo.get_field(0, f))


def test_config2_wet_dry_reduced(gc, gco):
    """config 2 at 128 x 128 (same recipe), 300 steps of run-up; masks bit-exact every step."""
    wl = workloads.cfg2(128)
    Lg, Lo = both(gc, gco, wl)
    w = Lo.wet_mask()
    assert 0 < w.sum() < w.size
    lockstep(Lg, Lo, 300, wl.cfl, 2.0)


@pytest.mark.parametrize("bc", [(1, 1, 1, 1), (0, 0, 0, 0), (1, 0, 0, 1)])
def test_tilings_match_single_patch_oracle(gc, gco, bc):
    """A2 + A4: any partition of the level into patches (ragged sizes, several tiles, corners) gives the bits of
    the oracle's single-patch run."""
    n = 48
    wl = workloads.cfg2(n)
    wl.params = dict(wl.params, bc=bc)
    tilings = [
        workloads.tile(n, n, 16),
        np.array([[0, 0, 20, 48], [20, 0, 28, 10], [20, 10, 28, 38]], dtype=np.int32),
        workloads.tile(n, n, 2),
        workloads.tile(n, n, 6),
        # columns 2, 3, 5 and 38 cells wide (rows 5, 43 high; 2 is the narrowest patch gc_level_create accepts): the
        # x-sweep's 4-cell output groups with only a head (2), a one-cell tail (3), a three-cell tail (5), and 38 cut into
        # segments of 12, 16, 10 cells (two-cell tails, and no tail)
        np.array([[0, 0, 2, 5], [2, 0, 3, 5], [5, 0, 5, 5], [10, 0, 38, 5],
                  [0, 5, 2, 43], [2, 5, 3, 43], [5, 5, 5, 43], [10, 5, 38, 43]], dtype=np.int32),
    ]
    for pats in tilings:
        Lg, Lo = both(gc, gco, wl, patches_g=pats)
        lockstep(Lg, Lo, 30, wl.cfl, 2.0)


def test_long_rows_and_columns_chunking(gc, gco):
    """patch wider than one x-tile (nx + 3 > 256) and taller than one y-segment; odd sizes."""
    wl = workloads.cfg2(64)
    wl.nx, wl.ny = 301, 37
    Lg, Lo = both(gc, gco, wl)
    lockstep(Lg, Lo, 20, wl.cfl, 2.0)
    wl.nx, wl.ny = 11, 277
    Lg, Lo = both(gc, gco, wl)
    lockstep(Lg, Lo, 20, wl.cfl, 2.0)


def test_config5_reduced_spherical_tilings(gc, gco):
    """config 5 recipe at 256 x 256 (0.5 arcmin, spherical, extrapolation): tilings 16, 32, 64, 128, 256 against the
    oracle's single patch (tiling invariance makes them comparable)."""
    n = 256
    wl = workloads.cfg5(n)
    for side in (16, 32, 64, 128, 256):
        Lg, Lo = both(gc, gco, wl, patches_g=workloads.tile(n, n, side))
        lockstep(Lg, Lo, 8, wl.cfl, 1.0)


def test_spherical_walls(gc, gco):
    n = 40
    wl = workloads.cfg3(n)
    wl.params = dict(wl.params, bc=(1, 1, 1, 1))
    Lg, Lo = both(gc, gco, wl, patches_g=workloads.tile(n, n, 10))
    lockstep(Lg, Lo, 20, wl.cfl, 0.5)


@pytest.mark.parametrize("fric", [dict(manning_n=0.025), dict(manning_n=0.025, friction_depth=5.0), dict(manning_n=0.1)])
def test_manning_friction_wet_dry(gc, gco, fric):
    """DESIGN.md 3.9 (S-16): the friction fractional step after the y-sweep and the clean-up, on the wet/dry shoreline of the
    config-2 recipe -- everywhere, in cells no deeper than 5 m only, and with a large n; patches of 16 and one ragged tiling."""
    n = 48
    wl = workloads.cfg2(n)
    wl.params = dict(wl.params, **fric)
    ragged = np.array([[0, 0, 20, 48], [20, 0, 28, 10], [20, 10, 28, 38]], dtype=np.int32)
    for pats in (workloads.tile(n, n, 16), ragged):
        Lg, Lo = both(gc, gco, wl, patches_g=pats)
        lockstep(Lg, Lo, 40, wl.cfl, 2.0)
        assert np.abs(Lo.get_global("hu")).max() > 1e-3          # the run has flow for friction to act on


def test_manning_friction_spherical(gc, gco):
    n = 128
    wl = workloads.cfg5(n)
    wl.params = dict(wl.params, manning_n=0.025)
    Lg, Lo = both(gc, gco, wl, patches_g=workloads.tile(n, n, 32))
    lockstep(Lg, Lo, 10, wl.cfl, 1.0)
    # and it is not a no-op there: the same run without friction ends with different momenta
    wl0 = workloads.cfg5(n)
    L0 = driver.setup_level(gco.Context(**wl0.params), wl0)
    driver.run_single_level(L0, 10, wl0.cfl)
    assert not np.array_equal(L0.get_global("hu"), Lo.get_global("hu"))


def test_first_order_mode(gc, gco):
    wl = workloads.cfg2(64)
    wl.params = dict(wl.params, limiter=0)
    Lg, Lo = both(gc, gco, wl)
    lockstep(Lg, Lo, 40, wl.cfl, 2.0)


def test_step_auto_device_dt_chain(gc, gco):
    """gc_level_step_auto keeps dt on the device: same states and dt sequence as the host-controlled loop."""
    import torch
    wl = workloads.cfg1()
    Lg, Lo = both(gc, gco, wl)
    dto = driver.probe_dt(Lo, wl.cfl)
    dtg = driver.probe_dt(Lg, wl.cfl)
    dt_dev = torch.tensor([dtg], dtype=torch.float64, device="cuda")
    for n in range(25):
        Lg.fill_ghost(None, 1.0); Lo.fill_ghost(None, 1.0)
        Lg.step_auto(dt_dev, wl.cfl)
        so = Lo.step(dto)
        dto = wl.cfl / so["s_over_dx_max"]
    assert dt_dev.item() == dto
    for f in ("h", "hu", "hv"):
        assert np.array_equal(Lg.get_global(f), Lo.get_global(f))


def test_empty_level_and_bad_arguments(gc):
    ctx = gc.Context(coord=0)
    L = ctx.level_create(1, 0.0, 0.0, 1.0, 1.0, 16, 16, 1, np.zeros((0, 4), dtype=np.int32))
    L.fill_ghost(None, 1.0)
    st = L.step(1.0)
    assert st["s_over_dx_max"] == 0.0 and L.ncells == 0
    with pytest.raises(RuntimeError):
        ctx.level_create(1, 0.0, 0.0, 1.0, 1.0, 16, 16, 1, np.array([[0, 0, 8, 8], [4, 4, 8, 8]], dtype=np.int32))  # overlap
    with pytest.raises(RuntimeError):
        ctx.level_create(1, 0.0, 0.0, 1.0, 1.0, 16, 16, 1, np.array([[10, 0, 8, 8]], dtype=np.int32))  # outside
    with pytest.raises(RuntimeError):
        ctx.level_create(2, 0.0, 0.0, 1.0, 1.0, 16, 16, 4, np.array([[2, 0, 8, 8]], dtype=np.int32))  # not aligned


def test_device_tensor_io(gc):
    import torch
    wl = workloads.cfg1(32)
    ctx = gc.Context(**wl.params)
    L = ctx.level_create(1, 0.0, 0.0, wl.dx, wl.dy, 32, 32, 1, workloads.tile(32, 32, 16))
    b, h, hu, hv = wl.fields()
    L.set_global("h", torch.from_numpy(h).cuda())
    out = torch.full((32, 32), float("nan"), dtype=torch.float64, device="cuda")
    L.get_global("h", out=out)
    assert np.array_equal(out.cpu().numpy(), h)
