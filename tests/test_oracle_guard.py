"""The guard of the CUDA path's open-ocean Riemann code (csrc/gc_riemann.cuh, DESIGN.md 5 "guard"), checked on the ORACLE.

The kernels skip step R5 (the flat-bottom middle state) for edges that satisfy, with c- = min(cL, cR),
    G:  |cL - cR| <= c-/4,   |uL| <= c-/4,   |uR| <= c-/4,   c- >= 0.1,
on the argument that, whatever branch R5 takes, its sigma1 <= -c-/4 and sigma2 >= c-/4, so that R6 returns the Einfeldt speeds
and none of the eight near-critical tests of R7 can fire.  The GPU parity tests compare the two paths on the configs' states; this
file checks the argument itself where those states never go: on the guard's boundary, at the smallest admissible depth, in all
three branches of R5 -- using the oracle's own R5 and its own solver.  Nothing here imports or mirrors the CUDA code."""
import math

import numpy as np

G = 9.81
TAU = 1.0e-6


def _states(rng, n):
    """random edges satisfying G, a third of them pushed onto its boundary"""
    for k in range(n):
        cmn = 10.0 ** rng.uniform(-1.0, 2.5) if k % 5 else 0.1
        d = rng.uniform(0.0, 0.25) if k % 3 else 0.25
        cA, cB = cmn, cmn * (1.0 + d)
        if cB - cA > 0.25 * cmn:                     # rounding pushed it over the boundary
            cB = np.nextafter(cB, 0.0)
        cL, cR = (cA, cB) if rng.random() < 0.5 else (cB, cA)
        hL, hR = cL * cL / G, cR * cR / G
        f = (lambda: rng.uniform(-0.25, 0.25)) if k % 3 else (lambda: rng.choice([-0.25, 0.25, 0.0]))
        uL, uR = f() * cmn, f() * cmn
        # the guard is evaluated on the computed celerities: make sure the state is inside it as the kernels would see it
        cLc, cRc = math.sqrt(G * hL), math.sqrt(G * hR)
        c4 = 0.25 * min(cLc, cRc)
        if not (abs(cLc - cRc) <= c4 and abs(uL) <= c4 and abs(uR) <= c4 and min(cLc, cRc) >= 0.1):
            continue
        yield hL, hR, uL, uR, cLc, cRc


def test_middle_state_speeds_are_bounded_away_from_zero_under_the_guard(gco):
    rng = np.random.default_rng(20261)
    n = 0
    branches = {"2rar": 0, "2shock": 0, "mixed": 0}
    for hL, hR, uL, uR, cL, cR in _states(rng, 60000):
        hm, s1m, s2m = gco.middle_state(G, 1e-3, hL, hR, uL, uR)
        cmn = min(cL, cR)
        assert s1m <= -0.25 * cmn * (1 - 1e-9) and s2m >= 0.25 * cmn * (1 - 1e-9), (hL, hR, uL, uR, s1m, s2m)
        hmin, hmax = min(hL, hR), max(hL, hR)
        branches["2shock" if hm > hmax else "2rar" if hm < hmin else "mixed"] += 1
        n += 1
    assert n > 40000 and min(branches.values()) > 1000, (n, branches)     # all three branches of R5 were exercised


def test_solver_returns_einfeldt_speeds_and_the_smooth_steady_jump_under_the_guard(gco):
    """R6 = R4 and 'not near-critical', read off the oracle's solver: s = (sE1, (sE1 + sE2)/2, sE2) bit for bit, and the depth jump
    removed in R7 is g h-bar (bR - bL) / P-bar (recovered from the f-waves) whenever the positivity clamp cannot bind."""
    rng = np.random.default_rng(20262)
    n = 0
    for hL, hR, uL, uR, cL, cR in _states(rng, 30000):
        bL = -hL + rng.uniform(-1, 1)
        delb = rng.uniform(-0.2, 0.2) * min(hL, hR)
        bR = bL + delb
        Z, s = gco.riemann(G, 1e-3, hL, hL * uL, 0.1 * hL, bL, hR, hR * uR, -0.2 * hR, bR)
        # the oracle forms u = p * (1 / h): use the same velocities
        uLo, uRo = (hL * uL) * (1.0 / hL), (hR * uR) * (1.0 / hR)
        uhat = (cL * uLo + cR * uRo) / (cL + cR)
        chat = math.sqrt(G * (0.5 * (hL + hR)))
        sE1, sE2 = min(uLo - cL, uhat - chat), max(uRo + cR, uhat + chat)
        assert s[0] == sE1 and s[2] == sE2 and s[1] == 0.5 * (sE1 + sE2), (hL, hR, uL, uR)
        hbar = 0.5 * (hL + hR)
        pbar = 0.25 * (uLo + uRo) ** 2 - G * hbar
        dh = (hR - hL) - (Z[0, 0] / s[0] + Z[2, 0] / s[2])
        assert abs(dh - G * hbar * (bR - bL) / pbar) <= 1e-11 * max(hL, hR), (hL, hR, uL, uR, bL, bR)
        # every quantity the near-critical tests compare with tau or sqrt(tau) is at least 50 times larger
        ptil = max(0.0, uLo * uRo) - G * hbar
        assert min(abs(pbar), pbar * ptil, pbar * s[0] * s[2]) > 50 * TAU and min(-s[0], s[2]) > 50 * math.sqrt(TAU)
        assert (uLo + cL) * (uRo + cR) > 0.0 and (uLo - cL) * (uRo - cR) > 0.0
        n += 1
    assert n > 20000
