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


def _extrapolate_outside(a, n_lo_x, n_hi_x, n_lo_y, n_hi_y):
    """zero-order extrapolation of a storage-shaped array: x faces first, then y faces over all columns"""
    if n_lo_x: a[:, :n_lo_x] = a[:, n_lo_x:n_lo_x + 1]
    if n_hi_x: a[:, -n_hi_x:] = a[:, -n_hi_x - 1:-n_hi_x]
    if n_lo_y: a[:n_lo_y, :] = a[n_lo_y:n_lo_y + 1, :]
    if n_hi_y: a[-n_hi_y:, :] = a[-n_hi_y - 1:-n_hi_y, :]
    return a


def test_unsplit_full_size_sampled_windows(gc, gco):
    """8192 x 8192 in 32 x 32 patches of side 256 (what `bench.py --scheme unsplit` times), K = 4 unsplit steps at the probe's dt.
    Windows of the result against the oracle, which advances one-patch levels grown by 3 K cells around each window (one unsplit
    step reaches 2 cells along and 1 across each direction) from the same initial data; where a window touches the domain boundary
    the test applies the extrapolation rule itself.  Patch interiors, a corner where four patches meet (the shuffle and ring seams of
    k_uns_update lie inside every patch: columns 30, 60, ... and rows 32, 64, ...), the domain corner and two edges."""
    n, side, w, K = 8192, 256, 40, 4
    m = 3 * K
    wl = workloads.cfg5(n)
    ctx = gc.Context(**wl.params)
    L = ctx.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, workloads.tile(n, n, side))
    rows = (1 << 24) // n
    for j0 in range(0, n, rows):
        b, h, hu, hv = wl.fields(i0=0, j0=j0, nx=n, ny=rows)
        L.set_global("b", b, 0, j0); L.set_global("h", h, 0, j0); L.set_global("hu", hu, 0, j0); L.set_global("hv", hv, 0, j0)
    L.fill_ghost_b()
    L.fill_ghost(None, 1.0)
    sdx = L.step_unsplit(0.0)["s_over_dx_max"]
    dt = wl.cfl / sdx
    for k in range(K):
        L.fill_ghost(None, 1.0)
        st = L.step_unsplit(dt)
        assert st["nan_seen"] == 0 and st["n_clipped"] == 0
    wins = [(100, 100), (256 - 20, 512 - 20), (4096 - 20, 4096 - 20), (0, 0), (n - w, 3000), (5000, n - w), (1024 + 20, 2048 + 12)]
    co = gco.Context(**wl.params)
    sdx0 = 0.0
    for (i0, j0) in wins:
        a0, a1 = max(i0 - m, 0), min(i0 + w + m, n)
        c0, c1 = max(j0 - m, 0), min(j0 + w + m, n)
        Lo = co.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, np.array([[a0, c0, a1 - a0, c1 - c0]], dtype=np.int32))
        gi = np.clip(np.arange(a0 - 2, a1 + 2), 0, n - 1); gj = np.clip(np.arange(c0 - 2, c1 + 2), 0, n - 1)
        fb = wl.fields(i0=int(gi.min()), j0=int(gj.min()), nx=int(gi.max() - gi.min()) + 1, ny=int(gj.max() - gj.min()) + 1)
        for f, v in zip(("b", "h", "hu", "hv"), fb):
            Lo.set_field(0, f, v[np.ix_(gj - gj.min(), gi - gi.min())])
        out = (2 if a0 == 0 else 0, 2 if a1 == n else 0, 2 if c0 == 0 else 0, 2 if c1 == n else 0)
        sdx0 = max(sdx0, Lo.step_unsplit(0.0)["s_over_dx_max"])
        for k in range(K):
            if any(out) and k > 0:
                for f in ("h", "hu", "hv"):
                    Lo.set_field(0, f, _extrapolate_outside(Lo.get_field(0, f), *out))
            Lo.step_unsplit(dt)
        for f in ("h", "hu", "hv"):
            g = L.get_global(f, gi0=i0, gj0=j0, gnx=w, gny=w)
            o = Lo.get_global(f, gi0=i0, gj0=j0, gnx=w, gny=w)
            assert np.array_equal(g, o), (f, i0, j0, np.abs(g - o).max())
            if f != "h":
                assert np.abs(o).max() > 0.0
        Lo.destroy()
    assert sdx0 <= sdx
    L.destroy()
