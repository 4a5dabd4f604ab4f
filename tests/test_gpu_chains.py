"""GPU parity of the chained marching lines (gc_internal.h "chains"): same-level patches that continue each other
along a sweep are walked as one line, each piece read and written in its own storage, and the x-sweep leaves out the ghost rows
no y line reads.  Whatever the chains are, the bits are those of the oracle's single patch -- with chains (the default), without
(GC_OPT_CHAINS = 1), with segment boundaries on, next to and far from piece boundaries (GC_OPT_MARCH_SEG)."""
import numpy as np
import pytest

import workloads
from harness import driver
from test_gpu_parity import lockstep

pytestmark = pytest.mark.gpu


def grid(xs, ys):
    """patches of the tensor grid with column widths xs and row heights ys"""
    out = []
    j0 = 0
    for ny in ys:
        i0 = 0
        for nx in xs:
            out.append([i0, j0, nx, ny])
            i0 += nx
        j0 += ny
    return np.array(out, dtype=np.int32)


def run(gc, gco, wl, pats, nsteps, eta_scale, chains, seg, step_fill=False):
    from paper_1901_06798_b200 import binding
    cg = gc.Context(**wl.params)
    cg.set_option(binding.OPT_SWEEP_FAMILY, binding.SWEEP_MARCH)
    cg.set_option(binding.OPT_CHAINS, 0 if chains else 1)
    cg.set_option(binding.OPT_MARCH_SEG, seg)
    Lg = driver.setup_level(cg, wl, patches=pats)
    if step_fill:                                   # gc_fill_ghost_step before every step: only what the step reads is filled
        Lg.fill_ghost = Lg.fill_ghost_step
    Lo = driver.setup_level(gco.Context(**wl.params), wl)
    lockstep(Lg, Lo, nsteps, wl.cfl, eta_scale)
    return Lg


# widths: pieces of 8 and 12 (multiples of 4: chained along x), 20, then 9 (odd: may only end a chain), 3 (too short to chain);
# heights: 8, 24, 11 (any length >= 8 chains along y), 5 (too short)
XS, YS = (8, 12, 20, 9, 3), (8, 24, 11, 5)


@pytest.mark.parametrize("chains", [True, False])
@pytest.mark.parametrize("seg", [0, 4, 8, 12, 16, 28, 4096])
def test_chains_wet_dry_mixed_sizes(gc, gco, chains, seg):
    wl = workloads.cfg2(64)
    wl.nx, wl.ny = sum(XS), sum(YS)
    run(gc, gco, wl, grid(XS, YS), 25, 2.0, chains, seg)


@pytest.mark.parametrize("seg", [8, 12, 16])
def test_chains_segment_starts_on_last_cell_of_a_piece(gc, gco, seg):
    """heights 11, 9, 14: the pieces of the y chains end at positions 13, 22 -- a segment that starts at position 12 (seg = 12)
    reads its first cell from one piece and the second from the next (the chained y-sweep requests rows two ahead)"""
    ys = (11, 9, 14)
    wl = workloads.cfg2(64)
    wl.nx, wl.ny = sum(XS), sum(ys)
    run(gc, gco, wl, grid(XS, ys), 25, 2.0, True, seg)


@pytest.mark.parametrize("seg", [0, 16, 40])
def test_chains_spherical_side16(gc, gco, seg):
    """config 5 recipe (spherical: the y-sweep's per-row metric follows the chain through its pieces), side 16 and side 8"""
    n = 128
    wl = workloads.cfg5(n)
    for side in (16, 8):
        on = run(gc, gco, wl, workloads.tile(n, n, side), 6, 1.0, True, seg).fallback_counts()["warp_iters"]
        off = run(gc, gco, wl, workloads.tile(n, n, side), 6, 1.0, False, seg).fallback_counts()["warp_iters"]
        # the chains are there: fewer warp iterations (no ghost rows between the pieces of a y chain, and with segments longer
        # than a patch fewer redundant cells along the lines)
        assert on < 0.95 * off, (side, seg, on, off)


def test_chains_partial_cover_and_walls(gc, gco):
    """an L-shaped set of patches next to a long one: chains end where the neighbour's extent differs; walls on every side"""
    wl = workloads.cfg2(48)
    wl.params = dict(wl.params, bc=(1, 1, 1, 1))
    pats = np.array([[0, 0, 16, 16], [16, 0, 16, 16], [32, 0, 16, 32], [0, 16, 32, 16], [0, 32, 16, 16], [16, 32, 32, 16]], dtype=np.int32)
    run(gc, gco, wl, pats, 30, 2.0, True, 0)
    run(gc, gco, wl, pats, 30, 2.0, True, 12)


def test_chains_friction_and_first_order(gc, gco):
    wl = workloads.cfg2(48)
    wl.params = dict(wl.params, manning_n=0.025)
    run(gc, gco, wl, workloads.tile(48, 48, 16), 25, 2.0, True, 0)
    wl = workloads.cfg2(48)
    wl.params = dict(wl.params, limiter=0)
    run(gc, gco, wl, workloads.tile(48, 48, 8), 25, 2.0, True, 20)


@pytest.mark.parametrize("seg", [0, 12, 40])
def test_fill_ghost_step_same_bits(gc, gco, seg):
    """gc_fill_ghost_step leaves out the same-level copies no sweep line reads; the steps after it give the oracle's bits --
    regular tilings (every same-level copy is dead), mixed sizes (chains end in the middle of the level), the L-shaped set."""
    wl = workloads.cfg2(64)
    wl.nx, wl.ny = sum(XS), sum(YS)
    run(gc, gco, wl, grid(XS, YS), 25, 2.0, True, seg, step_fill=True)
    wl = workloads.cfg2(48)
    wl.params = dict(wl.params, bc=(1, 0, 0, 1))
    for side in (8, 16):
        run(gc, gco, wl, workloads.tile(48, 48, side), 25, 2.0, True, seg, step_fill=True)
    pats = np.array([[0, 0, 16, 16], [16, 0, 16, 16], [32, 0, 16, 32], [0, 16, 32, 16], [0, 32, 16, 16], [16, 32, 32, 16]], dtype=np.int32)
    run(gc, gco, wl, pats, 25, 2.0, True, seg, step_fill=True)
    wl = workloads.cfg5(128)
    run(gc, gco, wl, workloads.tile(128, 128, 16), 6, 1.0, True, seg, step_fill=True)


def test_fill_ghost_step_poisoned_ghosts(gc, gco):
    """the cells gc_fill_ghost_step does not fill are really not read: NaN in every ghost cell before each fill changes nothing"""
    from paper_1901_06798_b200 import binding
    n = 64
    wl = workloads.cfg2(n)
    cg = gc.Context(**wl.params)
    cg.set_option(binding.OPT_SWEEP_FAMILY, binding.SWEEP_MARCH)
    pats = workloads.tile(n, n, 16)
    Lg = driver.setup_level(cg, wl, patches=pats)
    Lo = driver.setup_level(gco.Context(**wl.params), wl)
    dt = driver.probe_dt(Lo, wl.cfl)
    for it in range(12):
        for p in range(len(pats)):
            for f in ("h", "hu", "hv"):
                a = Lg.get_field(p, f)
                keep = a[2:-2, 2:-2].copy()
                a[:] = np.nan
                a[2:-2, 2:-2] = keep
                Lg.set_field(p, f, a)
        Lg.fill_ghost_step(None, 1.0); Lo.fill_ghost(None, 1.0)
        sg = Lg.step(dt); so = Lo.step(dt)
        assert sg["nan_seen"] == 0 and sg["s_over_dx_max"] == so["s_over_dx_max"], it
        dt = wl.cfl / so["s_over_dx_max"]
    for f in ("h", "hu", "hv"):
        assert np.array_equal(Lg.get_global(f), Lo.get_global(f))


def test_sweep_cells_accounting(gc):
    """gc_level_sweep_cells: a regular tiling with chains sweeps the level's own 4 ghost rows only; without chains 4 per patch"""
    from paper_1901_06798_b200 import binding
    n, side = 128, 16
    wl = workloads.cfg5(n)
    for chains, want in ((True, (n * (n + 4 * n // side), n * (n + 4), n * n)), (False, (n * (n + 4 * n // side),) * 2 + (n * n,))):
        ctx = gc.Context(**wl.params)
        ctx.set_option(binding.OPT_SWEEP_FAMILY, binding.SWEEP_MARCH)
        ctx.set_option(binding.OPT_CHAINS, 0 if chains else 1)
        L = driver.setup_level(ctx, wl, patches=workloads.tile(n, n, side))
        assert L.sweep_cells() == want, (chains, L.sweep_cells(), want)
