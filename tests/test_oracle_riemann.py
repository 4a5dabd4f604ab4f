"""Pins for the oracle's Riemann solver (oracle/gco_riemann.c) against what the paper and the
mathematics fix: "preserving steady state of the ocean, handling dry states ... maintaining
non-negative depth"; f-wave consistency sum_p Z^p = f(qR) - f(qL) - source; exact Riemann solutions
(Stoker, Ritter) for the two-wave middle state."""
import numpy as np
import pytest
from scipy.optimize import brentq

G = 9.81
EPS = 1e-3


def test_lake_at_rest_single_edges(gco):
    """eta = const, u = 0 over random bathymetry: every wave vanishes to roundoff."""
    rng = np.random.default_rng(1)
    worst = 0.0
    for _ in range(2000):
        bL, bR = rng.uniform(-5000, -1, 2)
        eta = rng.uniform(-0.5, 0.5)
        hL, hR = eta - bL, eta - bR
        if hL <= EPS or hR <= EPS:
            continue
        Z, s = gco.riemann(G, EPS, hL, 0.0, 0.0, bL, hR, 0.0, 0.0, bR)
        scale = G * max(hL, hR) ** 2
        worst = max(worst, np.abs(Z).max() / scale)
    assert worst < 5e-15


def test_lake_at_rest_against_dry_land(gco):
    """wet cell at rest next to a dry cell whose ground is above the water: wall, no waves."""
    Z, s = gco.riemann(G, EPS, 10.0, 0.0, 0.0, -10.0, 0.0, 0.0, 0.0, 5.0)
    assert np.abs(Z).max() < 1e-12
    Z, s = gco.riemann(G, EPS, 0.0, 0.0, 0.0, 5.0, 10.0, 0.0, 0.0, -10.0)
    assert np.abs(Z).max() < 1e-12


def test_both_dry(gco):
    Z, s = gco.riemann(G, EPS, 5e-4, 1.0, 1.0, 0.0, 0.0, 0.0, 0.0, 1.0)
    assert not Z.any() and not s.any()
    Z, s = gco.riemann(G, EPS, -1.0, 1.0, 1.0, 0.0, -2.0, 0.0, 0.0, 1.0)
    assert not Z.any() and not s.any()


def test_fwave_sums_flat_bottom(gco):
    """Flat bottom, both wet: sum_p Z^p = f(qR) - f(qL) exactly as a flux difference:
    (hu, hu^2 + g h^2/2, huv).  Catches a dropped term / wrong sign / transposed operand in R8."""
    rng = np.random.default_rng(2)
    for _ in range(5000):
        hL, hR = rng.uniform(0.01, 100.0, 2)
        uL, uR, vL, vR = rng.uniform(-5, 5, 4)
        pL, pR, tL, tR = hL * uL, hR * uR, hL * vL, hR * vR
        Z, s = gco.riemann(G, EPS, hL, pL, tL, -3.0, hR, pR, tR, -3.0)
        f = lambda h, p, t: np.array([p, p * p / h + 0.5 * G * h * h, p * t / h])
        df = f(hR, pR, tR) - f(hL, pL, tL)
        sc = np.abs(f(hR, pR, tR)) + np.abs(f(hL, pL, tL)) + 1e-300
        assert np.all(np.abs(Z.sum(axis=0) - df) <= 1e-12 * sc.max())
        assert s[0] <= s[1] <= s[2]
        # outer waves are eigen-directions (1, lambda, v lambda): Z_mom = lambda * Z_h
        assert abs(Z[0, 1] - s[0] * Z[0, 0]) <= 1e-10 * sc.max()
        assert abs(Z[2, 1] - s[2] * Z[2, 0]) <= 1e-10 * sc.max()
        assert Z[1, 0] == 0.0


def test_mass_fwave_with_topography(gco):
    """Mass component: sum_p Z^p_h = (hu)_R - (hu)_L for any bathymetry jump (mass has no source)."""
    rng = np.random.default_rng(3)
    for _ in range(5000):
        hL, hR = rng.uniform(0.01, 100.0, 2)
        bL, bR = rng.uniform(-10, 10, 2)
        uL, uR = rng.uniform(-3, 3, 2)
        Z, s = gco.riemann(G, EPS, hL, hL * uL, 0.3 * hL, bL, hR, hR * uR, -0.2 * hR, bR)
        assert abs(Z[:, 0].sum() - (hR * uR - hL * uL)) <= 1e-12 * (abs(hR * uR) + abs(hL * uL) + 1.0)


def test_mirror_symmetry(gco):
    """Reflecting x -> -x swaps the states, negates normal momentum, reverses the families."""
    rng = np.random.default_rng(4)
    for _ in range(3000):
        hL, hR = rng.uniform(0.0, 50.0, 2)
        bL, bR = rng.uniform(-5, 5, 2)
        pL, pR, tL, tR = rng.uniform(-20, 20, 4)
        Z, s = gco.riemann(G, EPS, hL, pL, tL, bL, hR, pR, tR, bR)
        Zm, sm = gco.riemann(G, EPS, hR, -pR, tR, bR, hL, -pL, tL, bL)
        sc = np.abs(Z).max() + 1e-9
        assert np.allclose(sm[::-1], -s, rtol=0, atol=1e-11 * (np.abs(s).max() + 1))
        # f-waves are flux jumps (right minus left): the fluxes hu and huv are odd under the mirror and the
        # jump direction flips, so their jumps keep sign; the normal-momentum flux is even, so its jump negates
        assert np.allclose(Zm[::-1, 0], Z[:, 0], rtol=0, atol=1e-10 * sc)
        assert np.allclose(Zm[::-1, 1], -Z[:, 1], rtol=0, atol=1e-10 * sc)
        assert np.allclose(Zm[::-1, 2], Z[:, 2], rtol=0, atol=1e-10 * sc)


def stoker_hm(hL, hR):
    """Exact middle depth of the dam break hL > hR > 0 (Stoker): 2(cL - cm) = (hm - hR) sqrt(g/2 (hm+hR)/(hm hR))."""
    cL = np.sqrt(G * hL)
    f = lambda hm: 2 * (cL - np.sqrt(G * hm)) - (hm - hR) * np.sqrt(0.5 * G * (hm + hR) / (hm * hR))
    return brentq(f, hR, hL)


def test_middle_state_branches_against_exact(gco):
    """R5: one secant / Newton step from the exact depth function.  Two rarefactions are a closed
    form (exact); for the others the one-step estimate must bracket correctly and be within a few
    percent for moderate jumps (it only widens speeds, R6)."""
    # two rarefactions: exact hm = (cL + cR - (uR-uL)/2)^2 / (4 g)
    hL, hR, uL, uR = 4.0, 3.0, -1.0, 2.0
    hm, s1, s2 = gco.middle_state(G, EPS, hL, hR, uL, uR)
    cm = 0.5 * (np.sqrt(G * hL) + np.sqrt(G * hR)) - 0.25 * (uR - uL)
    assert abs(hm - cm * cm / G) < 1e-13
    assert abs(s1 - (uL + 2 * np.sqrt(G * hL) - 3 * cm)) < 1e-13 and abs(s2 - (uR - 2 * np.sqrt(G * hR) + 3 * cm)) < 1e-13
    # dam break (mixed): one secant step overestimates F's root from the low side: hR < hm_est, close to exact
    for hL, hR, tol in [(10.0, 2.0, 0.12), (4000.5, 4000.0, 1e-6), (2.0, 1.9, 1e-3)]:
        hm, s1, s2 = gco.middle_state(G, EPS, hL, hR, 0.0, 0.0)
        ex = stoker_hm(hL, hR)
        assert hR < hm < hL
        assert abs(hm - ex) / ex < tol
        hm2, t1, t2 = gco.middle_state(G, EPS, hR, hL, 0.0, 0.0)  # mirrored
        assert abs(hm2 - hm) < 1e-12 * hm and abs(t1 + s2) < 1e-12 * abs(s2) and abs(t2 + s1) < 1e-12 * abs(s1)
    # two shocks: symmetric collision h, +u | h, -u: exact hm solves 2 (hm-h) sqrt(g/2 (1/hm+1/h)) = 2u
    h, u = 5.0, 1.0
    hm, s1, s2 = gco.middle_state(G, EPS, h, h, u, -u)
    ex = brentq(lambda x: (x - h) * np.sqrt(0.5 * G * (1 / x + 1 / h)) - u, h, 3 * h)
    assert abs(hm - ex) / ex < 1e-2 and s1 < 0 < s2 and abs(s1 + s2) < 1e-12
    # dry side: dry-front speed uL + 2 cL (Ritter)
    hm, s1, s2 = gco.middle_state(G, EPS, 3.0, 0.0, 0.5, 0.0)
    assert hm == 0.0 and abs(s1 - (0.5 + 2 * np.sqrt(G * 3.0))) < 1e-13 and s1 == s2


def test_dry_bed_front_speed_in_solver(gco):
    """R6: the outer speed next to a dry cell is widened to the Ritter front speed u + 2c."""
    h = 2.0
    Z, s = gco.riemann(G, EPS, h, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0)
    assert abs(s[2] - 2 * np.sqrt(G * h)) < 1e-12
    assert abs(s[0] + np.sqrt(G * h)) < 1e-12


def test_step_lowered_to_water_surface(gco):
    """R3: still water lower than a dry step that is NOT a wall candidate stays still."""
    # left wet, surface at eta=-1; right dry cell with ground at -0.5 > eta -> wall (ground above water)
    Z, s = gco.riemann(G, EPS, 1.0, 0.0, 0.0, -2.0, 0.0, 0.0, 0.0, -0.5)
    assert np.abs(Z).max() < 1e-13
