"""GPU parity of the unsplit step with transverse Riemann solves (gc_level_step_unsplit): the CUDA
path against the oracle through the C ABI, bit for bit -- Cartesian wet/dry with ragged tilings, the sphere (config 5's recipe and
config 3's seamount), friction on, the dt = 0 probe, and the refusal on a level that carries flux registers."""
import numpy as np
import pytest

import workloads
from harness import driver

pytestmark = pytest.mark.gpu


def _lockstep(Lg, Lo, nsteps, cfl):
    Lg.fill_ghost(None, 1.0); Lo.fill_ghost(None, 1.0)
    sg, so = Lg.step_unsplit(0.0), Lo.step_unsplit(0.0)                   # probe: nothing changes, speeds returned
    assert sg["s_over_dx_max"] == so["s_over_dx_max"] > 0.0
    dt = cfl / so["s_over_dx_max"]
    for n in range(nsteps):
        Lg.fill_ghost(None, 1.0); Lo.fill_ghost(None, 1.0)
        sg, so = Lg.step_unsplit(dt), Lo.step_unsplit(dt)
        assert sg["s_over_dx_max"] == so["s_over_dx_max"] and sg["n_clipped"] == so["n_clipped"], n
        assert abs(sg["clipped_mass"] - so["clipped_mass"]) <= 1e-12 * abs(so["clipped_mass"]) + 1e-300
        for f in ("h", "hu", "hv"):
            a, c = Lg.get_global(f), Lo.get_global(f)
            assert np.array_equal(a, c), (n, f, np.abs(a - c).max())
        assert np.array_equal(driver.unpack_cells(Lg, Lg.wet_mask()), driver.unpack_cells(Lo, Lo.wet_mask()))
        dt = cfl / so["s_over_dx_max"]


@pytest.mark.parametrize("tiles", [None, "regular", "ragged"])
def test_unsplit_cartesian_wet_dry(gc, gco, tiles):
    wl = workloads.cfg2(64)
    pats = {None: None, "regular": workloads.tile(64, 64, 16),
            "ragged": np.array([[0, 0, 38, 20], [38, 0, 26, 20], [0, 20, 5, 44], [5, 20, 59, 3], [5, 23, 59, 41]], dtype=np.int32)}[tiles]
    Lg = driver.setup_level(gc.Context(**wl.params), wl, patches=pats)
    Lo = driver.setup_level(gco.Context(**wl.params), wl)
    _lockstep(Lg, Lo, 25, 0.45)
    assert 0 < Lo.wet_mask().sum() < 64 * 64 and np.abs(Lo.get_global("hv")).max() > 1e-6


def test_unsplit_on_the_sphere_and_with_friction(gc, gco):
    wl = workloads.cfg5(96)
    Lg = driver.setup_level(gc.Context(**wl.params), wl, patches=workloads.tile(96, 96, 32))
    Lo = driver.setup_level(gco.Context(**wl.params), wl)
    _lockstep(Lg, Lo, 12, 0.45)
    wl = workloads.cfg3(64)
    wl.params = dict(wl.params, manning_n=0.025)
    Lg = driver.setup_level(gc.Context(**wl.params), wl, patches=workloads.tile(64, 64, 16))
    Lo = driver.setup_level(gco.Context(**wl.params), wl)
    _lockstep(Lg, Lo, 10, 0.45)


def test_unsplit_refuses_a_level_with_flux_registers(gc):
    wl = workloads.cfg1(16)
    ctx = gc.Context(**wl.params)
    C = driver.setup_level(ctx, wl)
    F = ctx.level_create(2, wl.xlo, wl.ylo, wl.dx / 2, wl.dy / 2, 32, 32, 2, np.array([[8, 8, 16, 16]], dtype=np.int32))
    C.flux_attach(F)
    C.fill_ghost(None, 1.0)
    with pytest.raises(RuntimeError):
        C.step_unsplit(1.0)
