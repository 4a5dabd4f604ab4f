"""gc_level_step_unsplit_static (include/gc.h): the unsplit step for callers that may not allocate -- its 18 scratch planes in a static
device array inside the library.  Checked against the existing path (gc_level_step_unsplit, whose scratch is allocated per level) bit
for bit -- the tolerance of every GPU test here -- on two calls in a row on DIFFERENT levels, so that the second call starts from the
first one's leftovers in the shared array; that the call allocates nothing through the library's allocator; and that a level beyond
the stated limit is refused with a clear message.  Collected last (pytest -x stops at the first failure)."""
import numpy as np
import pytest

import workloads
from harness import driver

pytestmark = pytest.mark.gpu


def _pair(gc, wl, tiles):
    ctx = gc.Context(**wl.params)
    return ctx, driver.setup_level(ctx, wl, patches=tiles), driver.setup_level(ctx, wl, patches=tiles)


def _same(La, Lb):
    for f in ("h", "hu", "hv"):
        a, b = La.get_global(f), Lb.get_global(f)
        assert np.array_equal(a, b), (f, np.abs(a - b).max())


def test_static_scratch_step_equals_the_allocating_step_on_two_calls_in_a_row(gc):
    import torch
    lim = gc.lib().gc_unsplit_static_max_cells()
    assert lim == 1 << 18
    # level 1: Cartesian wet/dry beach in ragged patches; level 2: the sphere (config 5's recipe), other sizes and offsets
    wl1 = workloads.cfg2(64)
    ragged = np.array([[0, 0, 38, 20], [38, 0, 26, 20], [0, 20, 5, 44], [5, 20, 59, 3], [5, 23, 59, 41]], dtype=np.int32)
    wl2 = workloads.cfg5(96)
    c1, A1, B1 = _pair(gc, wl1, ragged)
    c2, A2, B2 = _pair(gc, wl2, workloads.tile(96, 96, 32))
    dts = []
    for A, B in ((A1, B1), (A2, B2)):
        A.fill_ghost(None, 1.0); B.fill_ghost(None, 1.0)
        sa, sb = A.step_unsplit(0.0), B.step_unsplit_static(0.0)          # probe: nothing changes, speeds returned
        assert sa["s_over_dx_max"] == sb["s_over_dx_max"] > 0.0
        dts.append(0.45 / sa["s_over_dx_max"])
        _same(A, B)
    for rnd in range(6):                                                   # calls alternate between the two levels
        for k, (ctx, A, B) in enumerate(((c1, A1, B1), (c2, A2, B2))):
            A.fill_ghost(None, 1.0); B.fill_ghost(None, 1.0)
            sa = A.step_unsplit(dts[k])
            torch.cuda.synchronize()
            nb, mem = len(ctx._bufs), torch.cuda.memory_allocated()
            sb = B.step_unsplit_static(dts[k])
            assert len(ctx._bufs) == nb and torch.cuda.memory_allocated() == mem      # nothing allocated, nothing freed
            assert sa["s_over_dx_max"] == sb["s_over_dx_max"] and sa["n_clipped"] == sb["n_clipped"] and sb["nan_seen"] == 0
            assert abs(sa["clipped_mass"] - sb["clipped_mass"]) <= 1e-12 * abs(sa["clipped_mass"]) + 1e-300
            _same(A, B)
    assert 0 < A1.wet_mask().sum() < 64 * 64 and np.abs(A2.get_global("hu")).max() > 0.0
    # two calls in a row on ONE level without a host wait in between (out = NULL), then compared
    for _ in range(2):
        A2.fill_ghost(None, 1.0); B2.fill_ghost(None, 1.0)
        A2.step_unsplit(dts[1]); B2.step_unsplit_static(dts[1], sync=False)
    assert B2.stats()["nan_seen"] == 0
    _same(A2, B2)


def test_static_scratch_step_refuses_a_level_beyond_its_limit(gc):
    n = 520                                                                 # 524 x 524 storage cells > 2^18
    wl = workloads.cfg5(n)
    ctx = gc.Context(**wl.params)
    L = ctx.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, np.array([[0, 0, n, n]], dtype=np.int32))
    b, h, hu, hv = wl.fields(i0=0, j0=0, nx=n, ny=n)
    for f, v in zip(("b", "h", "hu", "hv"), (b, h, hu, hv)):
        L.set_global(f, v)
    L.fill_ghost_b(); L.fill_ghost(None, 1.0)
    before = L.get_global("h")
    with pytest.raises(RuntimeError, match="GC_UNS_STATIC_MAX_CELLS"):
        L.step_unsplit_static(1.0)
    assert np.array_equal(before, L.get_global("h"))                       # nothing changed
    assert L.step_unsplit(0.0)["s_over_dx_max"] > 0.0                       # the allocating path takes it
