"""Host control code: time-step control and the AMR recursion (section 3.1), regridding
cadence and Berger-Rigoutsos clustering.  Everything here is bookkeeping: every
arithmetic step of the method runs in the kernels behind the C ABI (include/gc.h).  The driver talks
to a *backend* (an object with level_create(...) returning Level objects with the methods of
binding.Level); the product backend is paper_1901_06798_b200.binding.Context.  Tests drive the
oracle through the same code to compare the two.
"""
import numpy as np


def setup_level(ctx, wl, level=1, dx=None, dy=None, nxl=None, nyl=None, ratio=1, patches=None):
    """Create a level of workload `wl`, set b, h, hu, hv from the analytic inputs (cell centres of
    THIS level, reading S-18) on every patch including its in-domain ghost cells."""
    dx = wl.dx if dx is None else dx
    dy = wl.dy if dy is None else dy
    nxl = wl.nx if nxl is None else nxl
    nyl = wl.ny if nyl is None else nyl
    if patches is None:
        patches = np.array([[0, 0, nxl, nyl]], dtype=np.int32)
    L = ctx.level_create(level, wl.xlo, wl.ylo, dx, dy, nxl, nyl, ratio, patches)
    set_initial(L, wl, state=True)
    return L


def set_initial(L, wl, state=True):
    """b (and optionally h, hu, hv) from the analytic workload functions, patch by patch, over the
    patch box grown by the ghost width and clipped to the domain."""
    pats = L.patches
    # group: if patches tile a modest domain, evaluate once globally
    if L.nxl * L.nyl <= (1 << 27):
        b, h, hu, hv = wl.fields(L.dx, L.dy, 0, 0, L.nxl, L.nyl)
        L.set_global("b", b)
        if state:
            L.set_global("h", h); L.set_global("hu", hu); L.set_global("hv", hv)
    else:
        for p in range(len(pats)):
            i0, j0, nx, ny = (int(v) for v in pats[p])
            a0, a1 = max(i0 - 2, 0), min(i0 + nx + 2, L.nxl)
            c0, c1 = max(j0 - 2, 0), min(j0 + ny + 2, L.nyl)
            b, h, hu, hv = wl.fields(L.dx, L.dy, a0, c0, a1 - a0, c1 - c0)
            L.set_global("b", b, a0, c0)
            if state:
                L.set_global("h", h, a0, c0); L.set_global("hu", hu, a0, c0); L.set_global("hv", hv, a0, c0)
    L.fill_ghost_b()


def probe_dt(L, cfl, coarser=None, alpha=1.0):
    """dt_0 from a probe step with dt = 0: dt = cfl / max(s / (kappa dx))."""
    L.fill_ghost(coarser, alpha)
    st = L.step(0.0)
    return cfl / st["s_over_dx_max"]


def run_single_level(L, nsteps, cfl, dt0=None, record=None):
    """nsteps level steps with dt_{n+1} = cfl / sigma_n (sigma = max s/(kappa dx) of step n).
    Returns the list of (dt, stats)."""
    dt = probe_dt(L, cfl) if dt0 is None else dt0
    hist = []
    for n in range(nsteps):
        L.fill_ghost(None, 1.0)
        st = L.step(dt)
        hist.append((dt, st))
        if record is not None:
            record(n, dt, st, L)
        dt = cfl / st["s_over_dx_max"]
    return hist
