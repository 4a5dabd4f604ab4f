"""2-D pins for the oracle's level step and ghost fill (oracle/gco_level.c): y-independent data
reproduces the 1-D sweep bitwise; tiling invariance (any partition into patches gives identical bits);
mirror symmetry of config 1; closed-basin mass balance with the clean-up accounted for; lake at rest
with islands; sphere: band area closed form, constant-metric sphere == Cartesian, lake at rest."""
import numpy as np
import pytest

import workloads
from harness import driver

G = 9.81


def make_level(gco, params, nx, ny, dx, dy, b, h, hu=None, hv=None, patches=None, xlo=0.0, ylo=0.0):
    ctx = gco.Context(**params)
    if patches is None:
        patches = np.array([[0, 0, nx, ny]], dtype=np.int32)
    L = ctx.level_create(1, xlo, ylo, dx, dy, nx, ny, 1, patches)
    L.set_global("b", b); L.set_global("h", h)
    L.set_global("hu", np.zeros_like(h) if hu is None else hu)
    L.set_global("hv", np.zeros_like(h) if hv is None else hv)
    L.fill_ghost_b()
    return L


def shoreline_case(n=24, seed=3):
    rng = np.random.default_rng(seed)
    x = (np.arange(n) + 0.5) * 100.0
    X, Y = np.meshgrid(x, x)
    b = -6.0 + 9.0 * X / x[-1] + 1.5 * np.sin(Y / 400.0) + rng.uniform(-0.2, 0.2, (n, n))
    eta = 0.8 * np.exp(-((X - 600) ** 2 + (Y - 1100) ** 2) / (2 * 300.0 ** 2))
    h = np.maximum(0.0, eta - b)
    return b, h


def test_y_independent_equals_1d(gco):
    import test_oracle_1d as T1
    n = 48
    rng = np.random.default_rng(2)
    x = (np.arange(n) + 0.5) * 50.0
    b1 = -5.0 + 7.0 * x / x[-1] + rng.uniform(-0.1, 0.1, n)
    h1 = np.maximum(0.0, 0.5 * np.exp(-((x - 800) / 200) ** 2) - b1)
    b = np.tile(b1, (8, 1)); h = np.tile(h1, (8, 1))
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(0, 0, 0, 0)), n, 8, 50.0, 50.0, b, h)
    hist = driver.run_single_level(L, 40, 0.9)
    # 1-D reference with the same dt sequence
    P = gco.make_params(coord=0, dry_tol=1e-3)
    hh = np.zeros(n + 4); hu = np.zeros(n + 4); hv = np.zeros(n + 4); bb = np.zeros(n + 4)
    hh[2:-2], bb[2:-2] = h1, b1
    T1.fill_bc(bb, False)
    rdx = np.full(n + 4, 1 / 50.0); ef = np.ones(n + 5)
    for dt, st in hist:
        T1.fill_bc(hh, False); T1.fill_bc(hu, False)
        hn, hun, _, sdx = gco.sweep_line(P, hh, hu, hv, bb, rdx, ef, dt)
        dry = hn < 1e-3
        hn[dry] = np.maximum(hn[dry], 0.0); hun[dry] = 0.0
        hh, hu = hn, hun
        assert st["s_over_dx_max"] >= sdx  # the 2-D maximum also covers the y-sweep on Q*
    H2 = L.get_global("h"); U2 = L.get_global("hu"); V2 = L.get_global("hv")
    for j in range(8):
        assert np.array_equal(H2[j], hh[2:-2]) and np.array_equal(U2[j], hu[2:-2])
    assert not V2.any()


@pytest.mark.parametrize("bc", [(1, 1, 1, 1), (0, 0, 0, 0), (1, 0, 0, 1)])
def test_tiling_invariance(gco, bc):
    n = 24
    b, h = shoreline_case(n)
    tilings = [
        np.array([[0, 0, n, n]]),
        workloads.tile(n, n, 12),
        np.array([[0, 0, 10, 24], [10, 0, 14, 8], [10, 8, 14, 16]]),
        workloads.tile(n, n, 4),
    ]
    ref = None
    for pats in tilings:
        L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=bc), n, n, 100.0, 100.0, b, h, patches=pats.astype(np.int32))
        hist = driver.run_single_level(L, 25, 0.9)
        out = (L.get_global("h"), L.get_global("hu"), L.get_global("hv"), [d for d, _ in hist],
               [s["cfl_max"] for _, s in hist], L.wet_mask().sum())
        assert not np.isnan(out[0]).any()
        if ref is None:
            ref = out
            assert (out[0] > 1e-3).sum() not in (0, n * n)  # wet and dry cells present
        else:
            for a, c in zip(ref[:3], out[:3]):
                assert np.array_equal(a, c)
            assert ref[3] == out[3] and ref[4] == out[4] and ref[5] == out[5]


def test_config1_mirror_symmetry_and_mass(gco):
    wl = workloads.cfg1()
    ctx = gco.Context(**wl.params)
    L = driver.setup_level(ctx, wl)
    m0 = L.mass()
    hist = driver.run_single_level(L, 100, wl.cfl)
    h, hu, hv = L.get_global("h"), L.get_global("hu"), L.get_global("hv")
    sc = np.abs(h - 4000).max()
    assert np.abs(h - h[:, ::-1]).max() <= 1e-13 * 4000 and np.abs(h - h[::-1]).max() <= 1e-13 * 4000
    assert np.abs(hu + hu[:, ::-1]).max() <= 1e-12 * np.abs(hu).max() + 1e-12
    assert np.abs(hv + hv[::-1]).max() <= 1e-12 * np.abs(hv).max() + 1e-12
    # x <-> y transpose only to splitting error (x-then-y is not transpose invariant)
    assert np.abs(h - h.T).max() < 0.02 * sc
    assert abs(L.mass() - m0) <= 1e-14 * m0
    assert all(s["n_clipped"] == 0 for _, s in hist)
    assert max(s["cfl_max"] for _, s in hist) <= 0.9001 and abs(hist[0][0] - 0.9 * 1000 / np.sqrt(G * 4001)) < 0.02
    # the hump has split into an outgoing ring: radial symmetry to truncation error
    assert 0.1 < (h - 4000).max() < 0.6


def test_mass_balance_with_shoreline(gco):
    """walls: M^{n+1} - M^n = clipped mass of that step, to roundoff (S-9)."""
    n = 32
    b, h = shoreline_case(n, seed=9)
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(1, 1, 1, 1)), n, n, 100.0, 100.0, b, h)
    m = [L.mass()]
    clipped = []
    driver.run_single_level(L, 60, 0.9, record=lambda k, dt, st, lev: (m.append(lev.mass()), clipped.append(st["clipped_mass"])))
    m = np.array(m); clipped = np.array(clipped)
    assert np.abs((m[1:] - m[:-1]) - clipped).max() <= 2e-14 * m[0] and clipped.max() > 0
    assert np.isfinite(m).all()


def test_lake_at_rest_2d_islands(gco):
    rng = np.random.default_rng(21)
    n = 40
    x = (np.arange(n) + 0.5) * 200.0
    X, Y = np.meshgrid(x, x)
    b = -300.0 + 330.0 * np.exp(-((X - 2500) ** 2 + (Y - 4000) ** 2) / 900.0 ** 2) \
        + 310.0 * np.exp(-((X - 6000) ** 2 + (Y - 2500) ** 2) / 700.0 ** 2) + rng.uniform(-3, 3, (n, n))
    h = np.maximum(0.0, -b)
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(1, 1, 0, 0)), n, n, 200.0, 200.0, b, h)
    hist = driver.run_single_level(L, 200, 0.9)
    H, U, V = L.get_global("h"), L.get_global("hu"), L.get_global("hv")
    wet = H > 1e-3
    assert 0 < (~wet).sum() < n * n
    assert np.abs(U).max() < 1e-10 and np.abs(V).max() < 1e-10
    assert np.abs((H + b)[wet]).max() < 1e-11


# ---------------------------------------------------------------- sphere

def test_sphere_band_area_closed_form(gco):
    R = 6367500.0
    ctx = gco.Context(coord=1, bc=(0, 0, 0, 0))
    n, d = 120, 0.5
    L = ctx.level_create(1, 10.0, -20.0, d, d, 80, n, 1, np.array([[0, 0, 80, n]], dtype=np.int32))
    kappa, rdx, rdy, ey = L.metric()
    area = (kappa[2:-2] * d * d).sum() * 80
    exact = R * R * np.deg2rad(80 * d) * (np.sin(np.deg2rad(-20.0 + n * d)) - np.sin(np.deg2rad(-20.0)))
    assert abs(area - exact) <= 1e-13 * exact
    # edge factor e_y = R cos(lat) pi/180 at the lower edge of each row; kappa ~ e_x e_y at mid latitude
    lat_e = np.deg2rad(-20.0 + (np.arange(n + 5) - 2) * d)
    assert np.allclose(ey, R * np.cos(lat_e) * np.pi / 180, rtol=1e-15)
    ex = R * np.pi / 180
    lat_c = np.deg2rad(-20.0 + (np.arange(n + 4) - 1.5) * d)
    assert np.allclose(kappa, ex * R * np.cos(lat_c) * np.pi / 180, rtol=1e-5)
    assert np.array_equal(rdx, 1.0 / (kappa * d))


def test_sphere_wall_metric_is_mirrored(gco):
    ctx = gco.Context(coord=1, bc=(1, 1, 1, 1))
    L = ctx.level_create(1, 0.0, 30.0, 0.5, 0.5, 8, 8, 1, np.array([[0, 0, 8, 8]], dtype=np.int32))
    k, rdx, rdy, ey = L.metric()
    assert k[1] == k[2] and k[0] == k[3] and k[-2] == k[-3] and k[-1] == k[-4]
    assert ey[1] == ey[3] and ey[0] == ey[4] and ey[-2] == ey[-4] and ey[-1] == ey[-5]


def test_sphere_equator_strip_close_to_cartesian(gco):
    """Near the equator on a tiny patch the metric is constant to ~1e-7: spherical run == Cartesian run with
    dx = R pi/180 * dlon up to that perturbation."""
    R = 6367500.0
    n, d = 32, 1e-3
    dxm = R * np.pi / 180 * d
    x = (np.arange(n) + 0.5)
    X, Y = np.meshgrid(x, x)
    b = -100.0 + 5.0 * np.sin(X / 5.0) * np.cos(Y / 7.0)
    h = np.maximum(0.0, 0.3 * np.exp(-((X - 16) ** 2 + (Y - 14) ** 2) / 18.0) - b)
    Ls = make_level(gco, dict(coord=1, bc=(0, 0, 0, 0)), n, n, d, d, b, h, ylo=-n * d / 2)
    Lc = make_level(gco, dict(coord=0, bc=(0, 0, 0, 0)), n, n, dxm, dxm, b, h)
    hs = driver.run_single_level(Ls, 30, 0.9)
    hc = driver.run_single_level(Lc, 30, 0.9)
    assert abs(hs[0][0] - hc[0][0]) < 1e-6 * hc[0][0]
    for f in ("h", "hu", "hv"):
        a, c = Ls.get_global(f), Lc.get_global(f)
        assert np.abs(a - c).max() < 1e-5 * (np.abs(c).max() + 1e-3)


def test_sphere_lake_at_rest(gco):
    rng = np.random.default_rng(4)
    n = 24
    b = -4000.0 + 800.0 * rng.uniform(-1, 1, (n, n))
    h = -b
    L = make_level(gco, dict(coord=1, bc=(1, 1, 1, 1)), n, n, 0.5, 0.5, b, h, xlo=140.0, ylo=30.0)
    driver.run_single_level(L, 100, 0.9)
    H, U, V = L.get_global("h"), L.get_global("hu"), L.get_global("hv")
    c = np.sqrt(G * 4800.0)
    assert np.abs(U).max() < 1e-13 * 4800 * c and np.abs(V).max() < 1e-13 * 4800 * c
    assert np.abs(H + b).max() < 1e-12 * 4800
