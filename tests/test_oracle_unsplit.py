"""Pins of the oracle's unsplit step with transverse Riemann solves (oracle/gco_unsplit.c, S-21).
The paper only names the algorithm; what the reading fixes is checked against what does not depend on it: the transverse split
must reassemble the Jacobian-vector product; data that vary in one direction only make every transverse term cancel, so the step
must equal the 1-D sweep bit for bit; the scheme treats x and y alike, so transposed data give the transposed result (the
dimensionally split scheme does not); lake at rest, the closed-basin mass balance and tiling invariance hold as for the split
step; and the two schemes converge to each other under refinement."""
import numpy as np

import workloads
from harness import driver

G = 9.81


def test_transverse_split_reassembles_the_jacobian_product(gco):
    rng = np.random.default_rng(71)
    for _ in range(2000):
        h = 10.0 ** rng.uniform(-1, 3.5)
        c = np.sqrt(G * h)
        w, z = rng.uniform(-2, 2) * c, rng.uniform(-2, 2) * c
        a = rng.standard_normal(3) * 10.0 ** rng.uniform(-3, 3)
        bm, bp = gco.transverse(G, 1e-3, h, h * w, h * z, a)
        B = np.array([[0.0, 1.0, 0.0], [G * h - w * w, 2.0 * w, 0.0], [-w * z, z, w]])     # d(pn, pn^2/h + g h^2/2, pn pt/h)/d(h, pn, pt)
        scale = np.abs(B).max() * np.abs(a).max()
        assert np.abs((bm + bp) - B @ a).max() <= 1e-12 * scale
        if w > 1.0001 * c:
            assert np.all(bm == 0.0)                    # supercritical: nothing travels against the flow
        if w < -1.0001 * c:
            assert np.all(bp == 0.0)
    bm, bp = gco.transverse(G, 1e-3, 5e-4, 1.0, 1.0, np.ones(3))
    assert np.all(bm == 0.0) and np.all(bp == 0.0)      # a dry cell passes nothing on
    # a pure down-going eigenvector comes back whole in bm, scaled by its eigenvalue
    h, w, z = 40.0, 1.5, -0.7
    c = np.sqrt(G * h)
    r1 = np.array([1.0, w - c, z])
    bm, bp = gco.transverse(G, 1e-3, h, h * w, h * z, r1)
    assert np.abs(bm - (w - c) * r1).max() < 1e-11 and np.abs(bp).max() < 1e-11


def _level(gco, n, bathy, eta0, dx=500.0, bc=(1, 1, 1, 1), tiles=None, hu=None, hv=None):
    wl = workloads.Workload("unsplit", dict(coord=0, dry_tol=1e-3, bc=bc), 0.0, 0.0, dx, dx, n, n, bathy, eta0, cfl=0.9)
    L = driver.setup_level(gco.Context(**wl.params), wl, patches=tiles)
    if hu is not None:
        x = (np.arange(n) + 0.5) * dx
        X, Y = np.meshgrid(x, x)
        L.set_global("hu", hu(X, Y)); L.set_global("hv", hv(X, Y))
    return wl, L


def _run(L, nsteps, unsplit, cfl=0.45, dt=None):
    L.fill_ghost(None, 1.0)
    if dt is None:
        dt = cfl / L.step(0.0)["s_over_dx_max"]
    hist = []
    for _ in range(nsteps):
        L.fill_ghost(None, 1.0)
        hist.append(L.step_unsplit(dt) if unsplit else L.step(dt))
    return dt, hist


def test_one_directional_data_reduce_to_the_1d_sweep_bitwise(gco):
    n = 40
    bx = lambda X, Y: -30.0 + 35.0 * X / (n * 500.0)                 # a beach in x: wet and dry cells
    ex = lambda X, Y: 1.5 * np.exp(-((X - 6000.0) / 1500.0) ** 2)
    for tr in (False, True):
        f = (lambda g: (lambda X, Y: g(Y, X))) if tr else (lambda g: g)
        _, Ls = _level(gco, n, f(bx), f(ex), bc=(0, 0, 0, 0)); _, Lu = _level(gco, n, f(bx), f(ex), bc=(0, 0, 0, 0))
        dt, hs = _run(Ls, 12, False)
        _, hu_ = _run(Lu, 12, True, dt=dt)
        for fld in ("h", "hu", "hv"):
            assert np.array_equal(Ls.get_global(fld), Lu.get_global(fld)), (tr, fld)
        assert [s["n_clipped"] for s in hs] == [s["n_clipped"] for s in hu_] and 0 < Ls.wet_mask().sum() < n * n


def test_unsplit_treats_x_and_y_alike_the_split_scheme_does_not(gco):
    n = 48
    bathy = lambda X, Y: -60.0 + 8.0 * np.sin(X / 3000.0) * np.cos(Y / 2500.0) + 0.002 * X
    eta = lambda X, Y: 1.2 * np.exp(-(((X - 9000.0) / 2500.0) ** 2 + ((Y - 14000.0) / 3500.0) ** 2))
    T = lambda g: (lambda X, Y: g(Y, X))
    res = {}
    for name, unsplit in (("unsplit", True), ("split", False)):
        _, La = _level(gco, n, bathy, eta); _, Lb = _level(gco, n, T(bathy), T(eta))
        dt, _ = _run(La, 15, unsplit)
        _run(Lb, 15, unsplit, dt=dt)
        d = max(np.abs(La.get_global("h") - Lb.get_global("h").T).max(), np.abs(La.get_global("hu") - Lb.get_global("hv").T).max() / 25.0)
        res[name] = d
    assert res["unsplit"] < 1e-12 * 70.0, res                        # rounding only
    assert res["split"] > 1e4 * max(res["unsplit"], 1e-15), res      # x-then-y is not transpose invariant


def test_lake_at_rest_mass_balance_and_tiling_invariance(gco):
    n = 32
    rng = np.random.default_rng(3)
    ph = rng.uniform(0, 2 * np.pi, 4)
    rough = lambda X, Y: -20.0 + 26.0 * X / (n * 500.0) + 1.5 * np.sin(X / 900.0 + ph[0]) * np.cos(Y / 700.0 + ph[1]) + 0.8 * np.cos(Y / 1300.0 + ph[2])
    _, L = _level(gco, n, rough, lambda X, Y: 0.0 * X)
    _run(L, 40, True)
    h, b = L.get_global("h"), L.get_global("b")
    wet = h > 1e-3
    assert 0 < wet.sum() < n * n and np.abs((h + b)[wet]).max() < 1e-12 * 25.0
    assert max(np.abs(L.get_global("hu")).max(), np.abs(L.get_global("hv")).max()) < 1e-11 * 25.0 * np.sqrt(G * 25.0)
    # a wave running up the beach in a closed basin: mass changes by what the clean-up clipped, exactly
    eta = lambda X, Y: 1.0 * np.exp(-(((X - 4000.0) / 1800.0) ** 2 + ((Y - 8000.0) / 2500.0) ** 2))
    ref = None
    for tiles in (None, workloads.tile(n, n, 8), np.array([[0, 0, 20, 32], [20, 0, 12, 10], [20, 10, 12, 22]], dtype=np.int32)):
        _, L = _level(gco, n, rough, eta, tiles=tiles)
        m0 = L.mass()
        dt, hist = _run(L, 30, True)
        m1 = L.mass()
        assert abs((m1 - m0) - sum(s["clipped_mass"] for s in hist)) < 1e-12 * m0
        out = [L.get_global(f) for f in ("h", "hu", "hv")] + [[s["s_over_dx_max"] for s in hist]]
        if ref is None:
            ref = out
            assert np.abs(out[1]).max() > 0.5
        else:
            assert all(np.array_equal(a, c) for a, c in zip(ref[:3], out[:3])) and ref[3] == out[3]


def test_split_and_unsplit_converge_to_each_other(gco):
    """the same smooth problem at two resolutions, to the same time: the two schemes differ by the splitting error, which shrinks
    under refinement (observed order about 2 for a smooth short run: require a factor 2.5)"""
    bathy = lambda X, Y: -50.0 + 0.0 * X
    diff = []
    for n in (32, 64):
        dx = 16000.0 / n
        eta = lambda X, Y: 0.5 * np.exp(-(((X - 8000.0) / 2200.0) ** 2 + ((Y - 8000.0) / 2200.0) ** 2))
        _, Ls = _level(gco, n, bathy, eta, dx=dx); _, Lu = _level(gco, n, bathy, eta, dx=dx)
        dt, _ = _run(Ls, n // 2, False, cfl=0.5)
        _run(Lu, n // 2, True, dt=dt)
        diff.append(np.abs(Ls.get_global("h") - Lu.get_global("h")).max())
    assert diff[0] > 1e-6 and diff[1] < diff[0] / 2.5, diff
