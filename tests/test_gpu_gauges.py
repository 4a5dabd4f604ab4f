"""GPU parity of the gauges (reading S-19) against the oracle, through the C ABI: the sampling itself on a
wet/dry state (the CUDA side tiled raggedly, so that many stencils read a sibling's cells through the ghost ring, the oracle on one
patch: tiling invariance makes them comparable), the recorded series of a two-level AMR run with regrids, the device-resident
series against the host path, and a spherical run.  Everything bit for bit."""
import numpy as np
import pytest

import workloads
from harness import driver

pytestmark = pytest.mark.gpu


def owner_patch(L, pts):
    return [driver.GaugeRecorder.patch_of(L, x, y) for x, y in pts]


def test_sampling_matches_the_oracle_on_a_wet_dry_state(gc, gco):
    n = 48
    wl = workloads.cfg2(n)
    ragged = np.array([[0, 0, 20, 48], [20, 0, 28, 10], [20, 10, 28, 38]], dtype=np.int32)
    for pats in (ragged, workloads.tile(n, n, 6)):
        Lg = driver.setup_level(gc.Context(**wl.params), wl, patches=pats)
        Lo = driver.setup_level(gco.Context(**wl.params), wl)
        driver.run_single_level(Lg, 30, wl.cfl); driver.run_single_level(Lo, 30, wl.cfl)
        Lg.fill_ghost(None, 1.0); Lo.fill_ghost(None, 1.0)
        rng = np.random.default_rng(12)
        L_ = n * wl.dx
        pts = np.vstack([rng.uniform(0.0, L_ * (1 - 1e-12), (600, 2)),
                         [[wl.dx * (i + 0.5), wl.dy * (j + 0.5)] for i in range(0, n, 5) for j in range(0, n, 7)],     # cell centres
                         [[20 * wl.dx + s, 7.3 * wl.dy] for s in (-1e-6, 0.0, 1e-6)],                                  # astride a patch edge
                         [[0.0, 0.0], [L_ * (1 - 1e-13), 3 * wl.dy]]])                                                 # the domain corner / edge
        og = Lg.gauges_sample(owner_patch(Lg, pts), pts)
        oo = Lo.gauges_sample(owner_patch(Lo, pts), pts)
        assert np.array_equal(og, oo)
        dry = oo[:, 0] <= 1e-3
        assert 20 < dry.sum() < len(pts) - 20                                   # both rules exercised
        # a gauge outside its patch is refused, and the earlier binding survives
        with pytest.raises(RuntimeError):
            Lg.gauges_bind([0], [[L_ * 2, 0.0]])
        assert np.array_equal(Lg.gauges_sample(), og)


def run_with_gauges(backend, wl, pts, nsteps, **kw):
    G = driver.GaugeRecorder(pts, **kw)
    H = driver.Hierarchy(backend.Context(**wl.params), wl, gauges=G)
    H.run(nsteps=nsteps)
    return H, G


def test_recorded_series_of_an_amr_run(gc, gco):
    base = workloads.cfg2(48)
    wl = workloads.Workload("amr2g", base.params, 0.0, 0.0, base.dx, base.dy, 48, 48, base.bathy, base.eta0, cfl=0.9,
                            ratios=(2,), flag=dict(tol_eta=0.1, buffer=2), regrid_interval=2, patch_max=24)
    Lx = 48 * base.dx
    pts = np.array([[x, y] for x in np.linspace(0.06, 0.94, 9) * Lx for y in (0.3 * Lx, 0.71 * Lx)])
    Ho, Go = run_with_gauges(gco, wl, pts, 12)
    Hg, Gg = run_with_gauges(gc, wl, pts, 12)
    Hd, Gd = run_with_gauges(gc, wl, pts, 12, device_series=True, capacity=7)   # small capacity: the series is flushed mid-run too
    assert Hg.t == Ho.t == Hd.t and Hg.regrids == Ho.regrids >= 5
    longest = 0
    for g in range(len(pts)):
        So, Sg, Sd = Go.series(g), Gg.series(g), Gd.series(g)
        assert np.array_equal(Sg, So), g                                        # times and all four quantities, bit for bit
        assert np.array_equal(Sd, So), g                                        # the device-resident series is the same series
        longest = max(longest, len(So))
    assert longest > 13                                                         # some gauge was sampled at the fine level's rate


def test_recorded_series_on_the_sphere(gc, gco):
    n = 96
    wl = workloads.cfg5(n)
    rng = np.random.default_rng(3)
    pts = np.stack([wl.xlo + rng.uniform(0.02, 0.98, 25) * n * wl.dx, wl.ylo + rng.uniform(0.02, 0.98, 25) * n * wl.dy], axis=1)
    Go = driver.GaugeRecorder(pts); Gg = driver.GaugeRecorder(pts, device_series=True)
    Ho = driver.Hierarchy(gco.Context(**wl.params), wl, gauges=Go)
    Hg = driver.Hierarchy(gc.Context(**wl.params), wl, gauges=Gg, patches1=workloads.tile(n, n, 16))
    Ho.run(nsteps=15); Hg.run(nsteps=15)
    for g in range(len(pts)):
        So, Sg = Go.series(g), Gg.series(g)
        assert len(So) == 16 and np.array_equal(Sg, So), g
    assert max(np.ptp(Go.series(g)[:, 4]) for g in range(len(pts))) > 1e-4      # the waves did pass the gauges
