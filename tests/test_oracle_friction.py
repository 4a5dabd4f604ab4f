"""Pins for the oracle's Manning friction step (oracle/gco_level.c gco_cbrt, gco_friction; eq. 1b-1c, 2;
DESIGN.md 3.9, reading S-16), none of which re-types its formula:

* the fixed cube-root sequence against libm's cbrt (an independent routine) over 24 decades;
* a uniform flow over a flat bed, through the whole level step: the hyperbolic part does nothing, and friction alone obeys
  d|u|/dt = -k |u|^2, k = g n^2 / h^(4/3) (the Manning law), whose exact solution |u|(t) = |u0| / (1 + k |u0| t) the
  semi-implicit step reproduces step by step; direction and depth unchanged.  h != 1 separates "momentum under the root"
  from the paper's printed "velocity under the root"; the oblique flow needs both components in the magnitude;
* friction_depth, dry cells and n = 0 leave every bit alone; lake at rest with islands stays at rest; the closed-basin
  mass balance holds with friction on (it never touches h); friction never raises or turns a momentum."""
import numpy as np
import pytest

import workloads
from harness import driver
from test_oracle_2d import make_level, shoreline_case

G = 9.81


def test_cbrt_sequence_against_libm(gco):
    rng = np.random.default_rng(11)
    xs = np.concatenate([np.exp(np.linspace(0.0, np.log(8.0), 20001)),           # one period of the bit seed
                         10.0 ** rng.uniform(-12.0, 12.0, 40000),
                         np.arange(1.0, 300.0) ** 3, [1e-3, 0.025, 1.0, 4500.0]])
    ys = np.array([gco.cbrt(x) for x in xs])
    ref = np.cbrt(xs)
    assert (np.abs(ys - ref) <= 4.0 * np.spacing(ref)).all()                     # measured: 3 ulp
    assert np.abs((ys * ys) * ys / xs - 1.0).max() < 2e-15
    assert (np.diff(np.array([gco.cbrt(x) for x in np.sort(xs)])) >= 0).all()    # monotone on the sample


@pytest.mark.parametrize("h0,u0,v0,n_man", [(0.5, 1.2, 0.0, 0.025), (0.5, 0.0, -0.9, 0.025), (0.25, 0.8, 0.6, 0.025),
                                             (2.0, -3.0, 1.0, 0.06)])
def test_uniform_flow_decays_by_the_manning_law(gco, h0, u0, v0, n_man):
    n, dx, dt, nsteps = 12, 50.0, 0.75, 60
    b = np.full((n, n), -h0)
    h = np.full((n, n), h0)
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(0, 0, 0, 0), manning_n=n_man), n, n, dx, dx, b, h,
                   hu=np.full((n, n), h0 * u0), hv=np.full((n, n), h0 * v0))
    k = G * n_man ** 2 / h0 ** (4.0 / 3.0)
    sp0 = float(np.hypot(u0, v0))
    for s in range(1, nsteps + 1):
        L.fill_ghost(None, 1.0)
        st = L.step(dt)
        assert st["nan_seen"] == 0
        if s in (1, 7, nsteps):
            H, U, V = L.get_global("h"), L.get_global("hu"), L.get_global("hv")
            assert (H == h0).all()                                               # friction never touches the depth
            assert np.ptp(U) == 0.0 and np.ptp(V) == 0.0                         # the flow stays uniform
            sp = sp0 / (1.0 + k * sp0 * s * dt)                                  # exact solution of the decay law
            assert abs(np.hypot(U[0, 0], V[0, 0]) / h0 - sp) <= 2e-13 * sp0
            assert abs(U[0, 0] * v0 - V[0, 0] * u0) <= 1e-15 * h0 * sp0 * sp0    # direction unchanged
    assert sp < 0.98 * sp0                                                       # and it did decay measurably


def test_friction_depth_dry_cells_and_zero_n_leave_every_bit(gco):
    n = 12
    b = np.full((n, n), -0.5); h = np.full((n, n), 0.5)
    hu = np.full((n, n), 0.6); hv = np.full((n, n), -0.2)
    for params in (dict(manning_n=0.025, friction_depth=0.2), dict(manning_n=0.0), dict()):
        L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(0, 0, 0, 0), **params), n, n, 50.0, 50.0, b, h, hu=hu, hv=hv)
        driver.run_single_level(L, 10, 0.9)
        assert (L.get_global("hu") == 0.6).all() and (L.get_global("hv") == -0.2).all()
    # a full wet/dry run: n = 0 given explicitly is the default path bit for bit
    wl = workloads.cfg2(32)
    res = []
    for extra in (dict(), dict(manning_n=0.0, friction_depth=3.0)):
        L = driver.setup_level(gco.Context(**dict(wl.params, **extra)), wl)
        driver.run_single_level(L, 25, wl.cfl)
        res.append([L.get_global(f) for f in ("h", "hu", "hv")])
    assert all(np.array_equal(a, c) for a, c in zip(*res))
    # one cell at a time: dry cells and cells deeper than friction_depth are returned unchanged
    assert gco.friction(1.0, 1e-3, 3.0, 4.0, manning_n=0.025) == (3.0, 4.0)
    assert gco.friction(1.0, 2.0, 3.0, 4.0, manning_n=0.025, friction_depth=1.0) == (3.0, 4.0)
    assert gco.friction(1.0, 2.0, 0.0, 0.0, manning_n=0.025) == (0.0, 0.0)


def test_friction_never_raises_or_turns_a_momentum(gco):
    rng = np.random.default_rng(5)
    for _ in range(2000):
        h = 10.0 ** rng.uniform(-2.5, 3.5); dt = 10.0 ** rng.uniform(-2, 1.5)
        hu, hv = rng.normal(0, 5.0, 2) * h
        a, c = gco.friction(dt, h, hu, hv, manning_n=0.025)
        assert 0.0 < a / hu <= 1.0 and 0.0 < c / hv <= 1.0
        assert abs(a / hu - c / hv) <= 4e-16                                     # one common factor 1 / d
    # shallower water is braked harder (D grows as h^(-7/3) at fixed momentum)
    f = [gco.friction(1.0, h, 1.0, 0.0, manning_n=0.025)[0] for h in (0.05, 0.2, 1.0, 5.0, 50.0)]
    assert all(x < y for x, y in zip(f, f[1:])) and f[-1] < 1.0


def test_mass_balance_and_lake_at_rest_with_friction(gco):
    """friction is a momentum source only: the closed-basin mass balance of test_oracle_2d holds unchanged, run-up is
    damped, and an ocean at rest over islands stays at rest."""
    n = 32
    b, h = shoreline_case(n, seed=9)
    out = {}
    for n_man in (0.0, 0.025, 0.1):
        L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(1, 1, 1, 1), manning_n=n_man), n, n, 100.0, 100.0, b, h)
        m = [L.mass()]; clipped = []
        driver.run_single_level(L, 60, 0.9, record=lambda k, dt, st, lev: (m.append(lev.mass()), clipped.append(st["clipped_mass"])))
        m = np.array(m); clipped = np.array(clipped)
        assert np.abs((m[1:] - m[:-1]) - clipped).max() <= 2e-14 * m[0]
        H, U, V = L.get_global("h"), L.get_global("hu"), L.get_global("hv")
        out[n_man] = 0.5 * np.where(H > 1e-3, (U * U + V * V) / np.maximum(H, 1e-3), 0.0).sum()
    assert out[0.1] < out[0.025] < out[0.0]                                     # kinetic energy: more friction, less motion
    rng = np.random.default_rng(21)
    n = 40
    x = (np.arange(n) + 0.5) * 200.0
    X, Y = np.meshgrid(x, x)
    b = -300.0 + 330.0 * np.exp(-((X - 2500) ** 2 + (Y - 4000) ** 2) / 900.0 ** 2) \
        + 310.0 * np.exp(-((X - 6000) ** 2 + (Y - 2500) ** 2) / 700.0 ** 2) + rng.uniform(-3, 3, (n, n))
    h = np.maximum(0.0, -b)
    L = make_level(gco, dict(coord=0, dry_tol=1e-3, bc=(1, 1, 0, 0), manning_n=0.025), n, n, 200.0, 200.0, b, h)
    driver.run_single_level(L, 200, 0.9)
    H, U, V = L.get_global("h"), L.get_global("hu"), L.get_global("hv")
    wet = H > 1e-3
    assert 0 < (~wet).sum() < n * n
    assert np.abs(U).max() < 1e-10 and np.abs(V).max() < 1e-10
    assert np.abs((H + b)[wet]).max() < 1e-11
