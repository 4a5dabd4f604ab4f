"""Round-2 pins of the oracle: the parts that seeded single-line mistakes slipped through in round 1.
None of these re-types an oracle routine: each states what the mathematics fixes -- a closed form of the sphere, a conservation
law, exactness for linear data, the textbook limiter values, an invariance the specification implies -- and checks the oracle
against it.  DESIGN.md 7 lists which seeded mistake fails which test.

  sphere, y direction   a y-only flow on a high-latitude level = the 1-D sweep fed with R cos(phi) pi/180 and the
                                        zone-area capacity; its mass change = the converging-meridian term, to roundoff
  refluxing, momentum (3.8)      flat bottom, oblique pulse through a static fine patch: composite sums of hu and hv constant
  coarse-to-fine interpolation (3.6)    eta, u, v linear in x AND y with different slopes: exact
  average-down on the sphere (3.7)      sum over fine cells of (h, hu, hv) x area = coarse value x coarse area at 60 N
  MC limiter (3.4)               Phi(theta) recovered from the correction flux at theta = -1, 0.2, 1/3, 1, 3, 10
  R3 (3.3)                              a dry step above the water surface but below the run-up height acts as a step at the surface
  R7 near-critical list (3.3)           an edge that only the 7th / only the 8th criterion catches takes the steady jump -(bR - bL)
  CFL range (3.4, S-6)                  ghost ROWS are swept in x but their speeds are not counted
"""
import math

import numpy as np
import pytest

import workloads
from harness import driver

G = 9.81
R_EARTH = 6367500.0
CART = dict(coord=0, dry_tol=1e-3, bc=(1, 1, 1, 1))


# ---------------------------------------------------------------------------------------------------------------- sphere, y
def _sphere_column_level(gco, nx=6, ny=48, ylo=55.0, d=0.05):
    """x-independent state on a spherical level at 55-57.4 N: a hump in eta and a northward current in mid-domain, at rest near the
    y boundaries.  hu = 0, so the x-sweep changes nothing and the level step is a set of identical 1-D y-sweeps."""
    P = dict(coord=1, dry_tol=1e-3, bc=(0, 0, 0, 0), earth_radius=R_EARTH)
    L = gco.Context(**P).level_create(1, 10.0, ylo, d, d, nx, ny, 1, np.array([[0, 0, nx, ny]], dtype=np.int32))
    yc = ylo + (np.arange(ny) + 0.5) * d
    b = -3000.0 + 400.0 * np.sin((yc - ylo) * 2.1)
    bump = np.exp(-((yc - (ylo + 0.5 * ny * d)) / (5 * d)) ** 2)
    h = (0.8 * bump) - b
    hv = h * (0.6 * bump)
    col = lambda v: np.repeat(v[:, None], nx, axis=1)
    L.set_global("b", col(b)); L.set_global("h", col(h)); L.set_global("hu", col(0 * h)); L.set_global("hv", col(hv))
    L.fill_ghost_b(); L.fill_ghost(None, 1.0)
    return L, P


def _closed_form_metric(ylo, d, ny):
    """DESIGN.md 3.5 written out with libm: per storage row k (global row k-2) the capacity kappa = zone area per square degree,
    per storage edge k (lower edge of row k) the factor R cos(phi) pi/180"""
    d2r = math.pi / 180.0
    ef = np.array([R_EARTH * math.cos((ylo + (k - 2) * d) * d2r) * d2r for k in range(ny + 5)])
    kap = np.array([d2r * R_EARTH * R_EARTH * (math.sin((ylo + (k - 1) * d) * d2r) - math.sin((ylo + (k - 2) * d) * d2r)) / d
                    for k in range(ny + 4)])
    return kap, ef


def test_sphere_y_sweep_equals_1d_sweep_with_closed_form_metric(gco):
    ny, ylo, d = 48, 55.0, 0.05
    L, P = _sphere_column_level(gco, ny=ny, ylo=ylo, d=d)
    dt = 0.8 / L.step(0.0)["s_over_dx_max"]
    hc, hvc, huc, bc = (L.get_field(0, f)[:, 3].copy() for f in ("h", "hv", "hu", "b"))
    st = L.step(dt)
    kap, ef = _closed_form_metric(ylo, d, ny)
    ho, po, to, sdx = gco.sweep_line(gco.make_params(**P), hc, hvc, huc, bc, 1.0 / (kap * d), ef, dt)
    assert np.abs(ho[2:-2] - hc[2:-2]).max() > 1e-3                               # the step did something
    for got, want in ((L.get_global("h")[:, 1], ho[2:-2]), (L.get_global("hv")[:, 1], po[2:-2])):
        assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()
    # an edge factor or capacity taken one row off is wrong by tan(56 deg) * 0.05 deg = 1.3e-3 relative
    assert st["s_over_dx_max"] >= sdx * (1 - 1e-12)                                # the level's maximum also holds the x-sweep


def test_sphere_mass_change_is_the_converging_meridian_term(gco):
    """SURVEY C.5 / DESIGN.md 3.5: with edge-scaled fluctuations the mass sum over j of h kappa dx dy changes in one step by
    dt dx sum_j hv_j (e_{j+1/2} - e_{j-1/2}) per column (summation by parts of sum_e e_e (hv_e - hv_{e-1}); F-tilde telescopes)
    when nothing reaches the y boundaries -- and by nothing else."""
    nx, ny, ylo, d = 6, 48, 55.0, 0.05
    L, P = _sphere_column_level(gco, nx=nx, ny=ny, ylo=ylo, d=d)
    dt = 0.8 / L.step(0.0)["s_over_dx_max"]
    hv = L.get_global("hv")[:, 0].copy()
    m0 = L.mass()
    L.step(dt)
    m1 = L.mass()
    _, ef = _closed_form_metric(ylo, d, ny)
    e_lo, e_hi = ef[2:ny + 2], ef[3:ny + 3]                  # lower / upper edge of interior row j
    want = dt * d * nx * float(np.sum(hv * (e_hi - e_lo)))
    assert abs(want) > 1e-9 * m0                             # the term is far above roundoff here ...
    assert abs((m1 - m0) - want) <= 2e-6 * abs(want)         # ... and it is the whole change (roundoff of m ~ 1e-16 m0 ~ 1e-7 |want|)


# ------------------------------------------------------------------------------------------------------ refluxing, momentum
def _composite_sum(H, field):
    """sum over the finest available cells of field x cell area (Cartesian)"""
    tot = 0.0
    for k, L in enumerate(H.levels):
        q = L.get_global(field, fill=0.0)
        w = np.zeros_like(q, dtype=bool)
        for i0, j0, nx, ny in L.patches:
            w[j0:j0 + ny, i0:i0 + nx] = True
        if k + 1 < len(H.levels):
            r = H.ratios[k]
            for i0, j0, nx, ny in H.levels[k + 1].patches:
                w[j0 // r:(j0 + ny) // r, i0 // r:(i0 + nx) // r] = False
        tot += float(q[w].sum()) * L.dx * L.dy
    return tot


@pytest.mark.parametrize("reflux", [True, False])
def test_flux_registers_conserve_composite_momentum(gco, reflux):
    """Flat bottom, no wall reached: sum hu and sum hv over the composite grid are constants of the motion (the wall pressures
    at the two ends cancel in still water).  An oblique pulse carrying net momentum crosses all four sides of a static fine
    patch.  P:146 step 5 (momentum components J^n, J^t) restores what the interface loses; without it they drift."""
    n, r, H0 = 44, 2, 12.0
    c0 = math.sqrt(G * H0)
    th = 0.6
    eta = lambda X, Y: 0.4 * np.exp(-((X - 2000.0) ** 2 + (Y - 2100.0) ** 2) / (2 * 150.0 ** 2))
    wl = workloads.Workload("mom", dict(CART), 0.0, 0.0, 100.0, 100.0, n, n, lambda X, Y: -H0 + 0.0 * X, eta,
                            cfl=0.9, ratios=(r,), flag=dict(tol_eta=-1.0, buffer=0), regrid_interval=1000, patch_max=16,
                            forced_boxes=((1, 1700.0, 2600.0, 1800.0, 2700.0, 0.0, 1e30),))
    H = driver.Hierarchy(gco.Context(**wl.params), wl, reflux=reflux)
    assert len(H.levels) == 2
    for L in H.levels:                                       # give the pulse momentum along (cos th, sin th)
        x = (np.arange(L.nxl) + 0.5) * L.dx
        X, Y = np.meshgrid(x, x)
        e = eta(X, Y)
        L.set_global("hu", (c0 * math.cos(th)) * e); L.set_global("hv", (c0 * math.sin(th)) * e)
    mu0, mv0 = _composite_sum(H, "hu"), _composite_sum(H, "hv")
    scale = abs(mu0) + abs(mv0)
    assert scale > 1e5
    drift = []
    H.run(nsteps=9, record=lambda n_, dt, h: drift.append((abs(_composite_sum(h, "hu") - mu0) + abs(_composite_sum(h, "hv") - mv0)) / scale))
    # nothing has reached a wall: the outermost two rings of coarse cells are still at rest
    hC = H.levels[0].get_global("h")
    assert np.abs(np.concatenate([hC[:2].ravel(), hC[-2:].ravel(), hC[:, :2].ravel(), hC[:, -2:].ravel()]) - H0).max() < 1e-11
    if reflux:
        assert max(drift) < 2e-13, max(drift)
    else:
        assert max(drift) > 1e-8, max(drift)


# ------------------------------------------------------------------------------------------------- interpolation, bilinear u, v
def test_interpolation_exact_for_velocities_linear_in_x_and_y(gco):
    from test_oracle_amr import two_levels
    n, r = 12, 4
    eta_lin = lambda X, Y: 0.002 * X - 0.001 * Y + 1.0
    u_lin = lambda X, Y: 0.30 + 2.0e-4 * X - 5.0e-4 * Y
    v_lin = lambda X, Y: -0.20 + 7.0e-4 * X + 3.0e-4 * Y
    (C, F), = two_levels([gco.Context(**CART)], n, r, [[8, 12, 16, 20]], lambda X, Y: -50.0 + 0.0 * X, eta_lin, state_fine=False)
    xc = (np.arange(n) + 0.5) * 100.0
    X, Y = np.meshgrid(xc, xc)
    hC = eta_lin(X, Y) + 50.0
    C.set_global("h", hC); C.set_global("hu", hC * u_lin(X, Y)); C.set_global("hv", hC * v_lin(X, Y))
    C.fill_ghost(None, 1.0)
    F.fill_ghost(C, 1.0)
    XF, YF = np.meshgrid((np.arange(-2, 18) + 8 + 0.5) * 25.0, (np.arange(-2, 22) + 12 + 0.5) * 25.0)
    ghost = np.ones(XF.shape, dtype=bool); ghost[2:-2, 2:-2] = False
    hF = eta_lin(XF, YF) + 50.0
    for f, want in (("h", hF), ("hu", hF * u_lin(XF, YF)), ("hv", hF * v_lin(XF, YF))):
        err = np.abs(F.get_field(0, f) - want)[ghost].max()
        assert err < 1e-11 * 60.0, (f, err)     # slopes along the wrong axis: |7e-4 - 3e-4| * 12.5 m * 50 m = 0.25


# ------------------------------------------------------------------------------------------------ average-down on the sphere
def test_average_down_conserves_area_weighted_sums_at_60N(gco):
    n, r, dC = 6, 4, 1.0                                     # 1-degree coarse cells at 58-64 N: kappa varies by 3 % per coarse cell
    P = dict(coord=1, dry_tol=1e-3, bc=(0, 0, 0, 0), earth_radius=R_EARTH)
    ctx = gco.Context(**P)
    C = ctx.level_create(1, 0.0, 58.0, dC, dC, n, n, 1, np.array([[0, 0, n, n]], dtype=np.int32))
    F = ctx.level_create(2, 0.0, 58.0, dC / r, dC / r, n * r, n * r, r, np.array([[4, 8, 12, 8]], dtype=np.int32))
    rng = np.random.default_rng(3)
    C.set_global("b", np.full((n, n), -100.0)); C.set_global("h", np.full((n, n), 100.0))
    C.set_global("hu", np.zeros((n, n))); C.set_global("hv", np.zeros((n, n)))
    hF = 100.0 + rng.uniform(-20, 20, (n * r, n * r)); uF = rng.uniform(-50, 50, hF.shape); vF = rng.uniform(-50, 50, hF.shape)
    F.set_global("b", np.full(hF.shape, -100.0)); F.set_global("h", hF); F.set_global("hu", uF); F.set_global("hv", vF)
    C.average_down_from(F)
    d2r = math.pi / 180.0
    area = lambda ylo_, dy_, dx_: R_EARTH ** 2 * (dx_ * d2r) * (math.sin((ylo_ + dy_) * d2r) - math.sin(ylo_ * d2r))   # zone area
    for f, fine in (("h", hF), ("hu", uF), ("hv", vF)):
        got = C.get_global(f)
        for J in (2, 3):
            for I in (1, 2, 3):
                s = sum(fine[J * r + jj, I * r + ii] * area(58.0 + (J * r + jj) * dC / r, dC / r, dC / r) for jj in range(r) for ii in range(r))
                assert abs(got[J, I] * area(58.0 + J * dC, dC, dC) - s) <= 1e-13 * abs(s) + 1e-3, (f, I, J)
        # unit weights instead of kappa would be off by ~ (3 % x spread of the values)


# -------------------------------------------------------------------------------------------------------------- MC limiter
@pytest.mark.parametrize("theta", [-1.0, 0.2, 1.0 / 3.0, 1.0, 3.0, 10.0])
def test_mc_limiter_value_recovered_from_the_correction_flux(gco, theta):
    """A right-going simple wave of tiny amplitude on a flat bottom is a scalar problem in family 3: the jump at edge e is a_e, the
    one at the upwind edge e-1 is theta a_e.  eq. 9 gives F~_e = 1/2 (1 - s dt/dx) Phi(theta) Z3_e (+ families 1, 2, smaller by 1e-6),
    and fm_e = F~_e + A-dQ_e.  Textbook MC: Phi = max(0, min((1 + theta)/2, 2, 2 theta))."""
    P = gco.make_params(coord=0, dry_tol=1e-3, limiter=1)
    n, H, a = 12, 10.0, 1.0e-6
    e = 7
    jumps = np.zeros(n + 4)
    jumps[e - 1] = theta * a; jumps[e] = a; jumps[e + 1] = 0.5 * a        # jumps[k] = h[k] - h[k-1]
    h = H + np.cumsum(jumps)
    u = 2.0 * (np.sqrt(G * h) - math.sqrt(G * H))
    p = h * u; t = 0.0 * h; b = np.full(n + 4, -H)
    rdx = np.ones(n + 4); ef = np.ones(n + 5)
    dt = 0.05
    _, _, _, _, fm, _ = gco.sweep_line(P, h, p, t, b, rdx, ef, dt, want_flux=True)
    Zm, _ = gco.riemann(G, 1e-3, h[e - 2], p[e - 2], 0.0, -H, h[e - 1], p[e - 1], 0.0, -H)
    Z, s = gco.riemann(G, 1e-3, h[e - 1], p[e - 1], 0.0, -H, h[e], p[e], 0.0, -H)
    assert abs(Z[0, 0]) < 1e-5 * abs(Z[2, 0]) and s[0] < 0 < s[2]
    th_actual = float(Zm[2] @ Z[2]) / float(Z[2] @ Z[2])
    assert abs(th_actual - theta) < 1e-5 * max(1.0, abs(theta))
    F = fm[e] - sum(Z[w] for w in range(3) if s[w] < 0)          # fm = F~ + A-dQ; A-dQ = the left-going families (tiny here)
    phi = float(F @ Z[2]) / (0.5 * (1.0 - s[2] * dt) * float(Z[2] @ Z[2]))
    want = max(0.0, min(0.5 * (1.0 + th_actual), 2.0, 2.0 * th_actual))
    assert abs(phi - want) < 2e-4, (theta, phi, want)               # minmod: 0.2 -> 0.2 (MC 0.4), 3 -> 1 (MC 2); superbee: 1/3 -> 2/3


# ------------------------------------------------------------------------------------------------------------------- R3
def test_dry_step_between_surface_and_runup_height_acts_at_the_surface(gco):
    """DESIGN.md 3.3 R3: a dry right cell whose bed lies above the water surface but not above the run-up height max(hL, hw) + bL
    is not a wall; the step is lowered to the water surface.  So the solution must not depend on HOW far above the surface the
    bed is, and must equal the one for a bed exactly at the surface; one hair above the run-up height it is the wall solution."""
    hL, uL, bL = 1.0, 1.5, -1.0
    hw, _, _ = gco.middle_state(G, 1e-3, hL, hL, uL, -uL)
    assert hw > hL + 0.3                                          # flow towards the step: the reflected problem piles water up
    ref = gco.riemann(G, 1e-3, hL, hL * uL, 0.2, bL, 0.0, 0.0, 0.0, hL + bL)
    assert np.abs(ref[0]).max() > 0.1
    for frac in (1e-6, 0.3, 0.9, 1.0 - 1e-12):
        bR = (hL + bL) + frac * (hw - hL)
        Z, s = gco.riemann(G, 1e-3, hL, hL * uL, 0.2, bL, 0.0, 0.0, 0.0, bR)
        assert np.array_equal(Z, ref[0]) and np.array_equal(s, ref[1]), frac
    Zw, sw = gco.riemann(G, 1e-3, hL, hL * uL, 0.2, bL, 0.0, 0.0, 0.0, (hw + bL) * (1 + 1e-12) + 1e-12)
    assert sw[1] == 0.0 and sw[2] == 0.0 and not np.array_equal(Zw[0], ref[0][0])      # wall: only the reflected family survives
    # mirror image (dry LEFT cell)
    refm = gco.riemann(G, 1e-3, 0.0, 0.0, 0.0, hL + bL, hL, -hL * uL, 0.2, bL)
    Zm, sm = gco.riemann(G, 1e-3, 0.0, 0.0, 0.0, (hL + bL) + 0.5 * (hw - hL), hL, -hL * uL, 0.2, bL)
    assert np.array_equal(Zm, refm[0]) and np.array_equal(sm, refm[1])


# ----------------------------------------------------------------------------------------------- R7, criteria 7 and 8
def _dh_from_waves(Z, s, hL, hR):
    """R8: delta_1 = (hR - hL) - dh_ss = beta1 + beta3, with Z^1_h = beta1 lambda1, Z^3_h = beta3 lambda3"""
    return (hR - hL) - (Z[0, 0] / s[0] + Z[2, 0] / s[2])


@pytest.mark.parametrize("state,crit", [
    ((1.49, 3.10, -1.49, 1.50, -4.32, -1.300), 7), ((1.07, -0.24, -1.07, 0.72, -3.17, -1.150), 7), ((0.41, -2.58, -0.41, 0.46, 1.64, -0.385), 7),
    ((0.22, 1.86, -0.22, 1.29, -0.88, -0.212), 8), ((0.52, 3.41, -0.52, 2.12, 4.01, -0.459), 8), ((0.51, 3.16, -0.51, 0.81, -2.70, -0.410), 8)])
def test_transcritical_edges_take_the_steady_depth_jump(gco, state, crit):
    """DESIGN.md 3.3 R7: if (uL + cL)(uR + cR) < 0 [7th] or (uL - cL)(uR - cR) < 0 [8th] the edge is near-critical and the depth
    jump removed before the decomposition is -(bR - bL), not g h-bar (bR - bL) / P-bar.  The states were picked so that the other
    seven criteria do not hold and the positivity clamps do not bind; the removed jump is read back from the f-waves."""
    hL, uL, bL, hR, uR, bR = state
    cL, cR = math.sqrt(G * hL), math.sqrt(G * hR)
    prod = (uL + cL) * (uR + cR) if crit == 7 else (uL - cL) * (uR - cR)
    other = (uL - cL) * (uR - cR) if crit == 7 else (uL + cL) * (uR + cR)
    assert prod < 0.0 < other
    Z, s = gco.riemann(G, 1e-3, hL, hL * uL, 0.0, bL, hR, hR * uR, 0.0, bR)
    hbar = 0.5 * (hL + hR)
    pbar = 0.25 * (uL + uR) ** 2 - G * hbar
    dh = _dh_from_waves(Z, s, hL, hR)
    assert abs(dh + (bR - bL)) < 1e-12                           # the steady jump of an ocean at rest ...
    assert abs(dh - G * hbar * (bR - bL) / pbar) > 1e-3 * abs(bR - bL)   # ... which the smooth-flow formula would not give here


# --------------------------------------------------------------------------------------------------------------- CFL range
def test_cfl_does_not_count_x_edges_of_ghost_rows(gco):
    """DESIGN.md 3.4 (S-5, S-6): the x-sweep covers ghost rows, eq. 15 is taken over interior lines.  The outermost ghost rows are
    given a 400 times deeper ocean: a y edge next to them is never counted (edges 1..n+1 lie between rows -1 and n), so the only way
    their speed can enter the level's maximum is through the x-edges of the ghost rows themselves."""
    n, dx, H = 10, 50.0, 10.0
    L = gco.Context(**dict(CART, bc=(0, 0, 0, 0))).level_create(1, 0.0, 0.0, dx, dx, n, n, 1, np.array([[0, 0, n, n]], dtype=np.int32))
    h = np.full((n + 4, n + 4), H); h[0, :] = 4000.0; h[-1, :] = 4000.0
    L.set_field(0, "h", h); L.set_field(0, "b", -h); L.set_field(0, "hu", 0 * h); L.set_field(0, "hv", 0 * h)
    st = L.step(0.0)
    assert abs(st["s_over_dx_max"] - math.sqrt(G * H) / dx) <= 1e-14 * math.sqrt(G * H) / dx
