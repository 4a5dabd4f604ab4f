"""Neutral AMR harness: time-step control and the AMR recursion (section 3.1),
regridding cadence and Berger-Rigoutsos clustering.  Everything here is bookkeeping: every
arithmetic step of the method runs behind a *backend* -- an object with level_create(...) returning Level objects
with the methods of paper_1901_06798_b200.binding.Level (the product, through the C ABI of include/gc.h) or of
oracle.gco.Level (the oracle).  This package imports neither; tests drive both through it to compare them, and
tests/test_harness_pins.py pins the recursion itself against a straight-line script and a uniformly fine run.
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
    # if the patches cover most of a modest domain, evaluate once globally; else patch by patch
    # (the bathymetry comes from the workload's tile cache either way; the initial state only when asked for)
    if L.nxl * L.nyl <= (1 << 27) and L.nxl * L.nyl <= 2 * L.ncells:
        if state:
            b, h, hu, hv = wl.fields(L.dx, L.dy, 0, 0, L.nxl, L.nyl)
            L.set_global("b", b); L.set_global("h", h); L.set_global("hu", hu); L.set_global("hv", hv)
        else:
            L.set_global("b", wl.bathy_box(L.dx, L.dy, 0, 0, L.nxl, L.nyl))
    else:
        # every patch's storage-shaped block (its box grown by the ghost width; the part inside the level is filled) packed back to
        # back and handed over in one call; cells outside the level stay 0 here and belong to the boundary fill
        names = ("b", "h", "hu", "hv") if state else ("b",)
        # a level defined by fixed boxes comes back with the same patch list at every regrid: its packed bathymetry is kept (a few
        # entries per workload, most recent first) and handed over again as it is
        key = (L.dx, L.dy, L.nxl, L.nyl, np.ascontiguousarray(pats).tobytes())
        cache = wl.__dict__.setdefault("_packed_b", [])
        if not state:
            for k, (ck, arr) in enumerate(cache):
                if ck == key:
                    cache.insert(0, cache.pop(k))
                    L.set_patches("b", arr)
                    L.fill_ghost_b()
                    return
        if not state and L.nxl * L.nyl <= CANVAS_MAX_CELLS:
            set_bathy_from_canvas(L, wl)       # no host assembly, no upload: the level's cells are gathered from a resident canvas
            L.fill_ghost_b()
            return
        if not state:
            packed_b = pack_bathy_native(L, wl)
            L.set_patches("b", packed_b)
            cache.insert(0, (key, packed_b))
            del cache[6:]
            L.fill_ghost_b()
            return
        sizes = [(int(p[2]) + 4) * (int(p[3]) + 4) for p in pats]
        packed = {f: np.zeros(int(np.sum(sizes, dtype=np.int64))) for f in names}
        o = 0
        for p in range(len(pats)):
            i0, j0, nx, ny = (int(v) for v in pats[p])
            a0, a1 = max(i0 - 2, 0), min(i0 + nx + 2, L.nxl)
            c0, c1 = max(j0 - 2, 0), min(j0 + ny + 2, L.nyl)
            vals = wl.fields(L.dx, L.dy, a0, c0, a1 - a0, c1 - c0) if state else (wl.bathy_box(L.dx, L.dy, a0, c0, a1 - a0, c1 - c0),)
            for f, v in zip(names, vals):
                blk = packed[f][o:o + sizes[p]].reshape(ny + 4, nx + 4)
                blk[c0 - (j0 - 2):c1 - (j0 - 2), a0 - (i0 - 2):a1 - (i0 - 2)] = v
            o += sizes[p]
        for f in names:
            L.set_patches(f, packed[f])
        cache.insert(0, (key, packed["b"]))
        del cache[6:]
    L.fill_ghost_b()


def deform_ramp(wl, t):
    """weight of the seafloor deformation at time t: 0 before t0, 1 from t1 on, linear in between"""
    d = wl.deform
    if d is None or t < d["t0"]:
        return 0.0
    if t >= d["t1"]:
        return 1.0
    return (t - d["t0"]) / (d["t1"] - d["t0"])


def deform_to(L, wl, t):
    """bring the bathymetry of level L to time t: b += (rho(t) - rho already applied) dz, then its ghost cells outside the domain"""
    if wl.deform is None:
        return
    rho = deform_ramp(wl, t)
    w = rho - getattr(L, "rho_applied", 0.0)
    if w != 0.0:
        d = wl.deform
        L.bathy_update(d["x0"], d["y0"], d["ddx"], d["ddy"], d["dz"], w)
        L.fill_ghost_b()
        L.rho_applied = rho


def probe_dt(L, cfl, coarser=None, alpha=1.0):
    """dt_0 from a probe step with dt = 0: dt = cfl / max(s / (kappa dx))."""
    L.fill_ghost(coarser, alpha)
    st = L.step(0.0)
    return cfl / st["s_over_dx_max"]


def run_single_level(L, nsteps, cfl, dt0=None, record=None, wl=None):
    """nsteps level steps with dt_{n+1} = cfl / sigma_n (sigma = max s/(kappa dx) of step n).
    Returns the list of (dt, stats).  wl with a deformation: the bathymetry is brought to each step's start time first."""
    dt = probe_dt(L, cfl) if dt0 is None else dt0
    hist = []
    t = 0.0
    # nothing but the step reads the ghost cells between a fill and the step here: a backend that has the narrower fill
    # (gc_fill_ghost_step: only the ghost cells the step reads; same result) is given the chance to use it
    fill = getattr(L, "fill_ghost_step", L.fill_ghost)
    for n in range(nsteps):
        if wl is not None:
            deform_to(L, wl, t)
        t += dt
        fill(None, 1.0)
        st = L.step(dt)
        hist.append((dt, st))
        if record is not None:
            record(n, dt, st, L)
        dt = cfl / st["s_over_dx_max"]
    return hist


# ---------------------------------------------------------------------------------------------------------
# Clustering ("Berger-Rigoutsos"): flagged cells of level l -> rectangles.  Deterministic (ties to the
# lower index), shared by both backends AFTER their flags have been compared bit for bit (DESIGN.md 3.11 S-13).
def _signature_cut(sig):
    """Cut position (1..n-1) for a 1-D signature: first a hole (zero entry) nearest the centre, else the strongest
    inflection of the discrete Laplacian; None if neither exists."""
    n = len(sig)
    zeros = [k for k in range(1, n - 1) if sig[k] == 0]
    if zeros:
        k = min(zeros, key=lambda z: (abs(z - n / 2.0), z))
        return k
    if n < 4:
        return None
    lap = sig[:-2] - 2 * sig[1:-1] + sig[2:]          # lap[k] belongs to cell k+1
    best, bestk = 0, None
    for k in range(len(lap) - 1):
        if lap[k] * lap[k + 1] < 0:
            mag = abs(int(lap[k]) - int(lap[k + 1]))
            if mag > best or (mag == best and bestk is not None and abs(k + 2 - n / 2.0) < abs(bestk - n / 2.0)):
                best, bestk = mag, k + 2               # cut between cells k+1 and k+2
    return bestk


def cluster(flags, valid=None, efficiency=0.7, max_side=64):
    """flags: 2-D uint8 (ny, nx) of one level.  valid (optional, same shape): cells a box may contain.
    Returns a list of (i0, j0, nx, ny) boxes (cells of that level), disjoint, covering every flagged cell,
    sorted by (j0, i0).  Signatures and box counts come from two running sums (along y per column, along x per row) and a
    summed-area table, so a box costs O(nx + ny) instead of O(nx ny)."""
    out = []
    fl = np.asarray(flags, dtype=bool)
    NY, NX = fl.shape
    cy = np.zeros((NY + 1, NX), dtype=np.int64); np.cumsum(fl, axis=0, out=cy[1:])          # cy[j, i] = flags in column i below row j
    cx = np.zeros((NY, NX + 1), dtype=np.int64); np.cumsum(fl, axis=1, out=cx[:, 1:])       # cx[j, i] = flags in row j left of column i
    bad = None
    if valid is not None:                                                                    # summed-area table of the invalid cells
        bad = np.zeros((NY + 1, NX + 1), dtype=np.int64)
        np.cumsum(np.cumsum(~np.asarray(valid, dtype=bool), axis=0), axis=1, out=bad[1:, 1:])
    stack = [(0, 0, NX, NY)]
    while stack:
        i0, j0, nx, ny = stack.pop()
        sx = cy[j0 + ny, i0:i0 + nx] - cy[j0, i0:i0 + nx]                # flags per column of the box
        xs = np.nonzero(sx)[0]
        if len(xs) == 0:
            continue
        sy = cx[j0:j0 + ny, i0 + nx] - cx[j0:j0 + ny, i0]                # flags per row of the box
        ys = np.nonzero(sy)[0]
        i0, nx = i0 + int(xs[0]), int(xs[-1] - xs[0] + 1)                # shrink to the bounding box of the flags
        j0, ny = j0 + int(ys[0]), int(ys[-1] - ys[0] + 1)
        sx = sx[int(xs[0]):int(xs[-1]) + 1]; sy = sy[int(ys[0]):int(ys[-1]) + 1]
        ok_valid = True if bad is None else (bad[j0 + ny, i0 + nx] - bad[j0, i0 + nx] - bad[j0 + ny, i0] + bad[j0, i0]) == 0
        eff = int(sx.sum()) / float(nx * ny)
        if eff >= efficiency and ok_valid and nx <= max_side and ny <= max_side:
            out.append((i0, j0, nx, ny))
            continue
        cut = None
        if nx > max_side or ny > max_side:             # chop oversize boxes first, in the middle of the long side
            cut = ("x", nx // 2) if nx >= ny else ("y", ny // 2)
        else:
            cx_ = _signature_cut(sx); cy_ = _signature_cut(sy)
            hx = cx_ is not None and sx[cx_] == 0; hy = cy_ is not None and sy[cy_] == 0
            if hx or hy:
                cut = ("x", cx_) if (hx and (not hy or nx >= ny)) else ("y", cy_)
            elif cx_ is not None or cy_ is not None:
                cut = ("x", cx_) if (cx_ is not None and (cy_ is None or nx >= ny)) else ("y", cy_)
            elif nx > 1 or ny > 1:
                cut = ("x", nx // 2) if nx >= ny else ("y", ny // 2)
        if cut is None:                                 # a single cell: accept (flagged cells are valid by construction)
            out.append((i0, j0, nx, ny))
            continue
        if cut[0] == "x":
            stack.append((i0 + cut[1], j0, nx - cut[1], ny)); stack.append((i0, j0, cut[1], ny))
        else:
            stack.append((i0, j0 + cut[1], nx, ny - cut[1])); stack.append((i0, j0, nx, cut[1]))
    out.sort(key=lambda b: (b[1], b[0]))
    return out


_native_lib = None


def native():
    """harness/libamr_host.so (amr_host.c: the same clustering, nesting mask and unpacking in C), built on first use"""
    global _native_lib
    if _native_lib is None:
        import ctypes as C
        from harness import build as hb
        lib = C.CDLL(hb.build())
        vp, i = C.c_void_p, C.c_int
        lib.amr_unpack.argtypes = [vp, vp, i, i, i, i, i, vp]; lib.amr_unpack.restype = None
        lib.amr_nesting_mask.argtypes = [vp, i, i, i, i, i, i, i, vp]; lib.amr_nesting_mask.restype = None
        lib.amr_cluster.argtypes = [vp, vp, i, i, C.c_double, i, vp, i]; lib.amr_cluster.restype = i
        _native_lib = lib
    return _native_lib


def cluster_native(flags, valid=None, efficiency=0.7, max_side=64):
    """cluster() in C: identical boxes (tests/test_harness_pins.py)"""
    fl = np.ascontiguousarray(flags, dtype=np.uint8)
    va = None if valid is None else np.ascontiguousarray(valid, dtype=np.uint8)
    cap = 1024
    while True:
        out = np.empty((cap, 4), dtype=np.int32)
        n = native().amr_cluster(fl.ctypes.data, None if va is None else va.ctypes.data, fl.shape[0], fl.shape[1],
                                 float(efficiency), int(max_side), out.ctypes.data, cap)
        if n >= 0:
            return [tuple(b) for b in out[:n].tolist()]
        cap *= 8


def unpack_cells_native(L, packed, bbox):
    bi, bj, ei, ej = bbox
    pats = np.ascontiguousarray(L.patches, dtype=np.int32)
    pk = np.ascontiguousarray(packed, dtype=np.uint8)
    out = np.empty((ej - bj, ei - bi), dtype=np.uint8)
    native().amr_unpack(pk.ctypes.data, pats.ctypes.data, len(pats), bi, bj, ei, ej, out.ctypes.data)
    return out


def nesting_mask_native(L, bbox):
    bi, bj, ei, ej = bbox
    pats = np.ascontiguousarray(L.patches, dtype=np.int32)
    ok = np.empty((ej - bj, ei - bi), dtype=np.uint8)
    native().amr_nesting_mask(pats.ctypes.data, len(pats), bi, bj, ei, ej, int(L.nxl), int(L.nyl), ok.ctypes.data)
    return ok.view(bool)


CANVAS_MAX_CELLS = 1 << 27      # 1 GiB of doubles: larger levels (their fine levels come from fixed boxes and are cached) are packed


def _tiles_needed(L, T):
    pats = np.ascontiguousarray(L.patches, dtype=np.int32)
    lo_i = np.maximum(pats[:, 0] - 2, 0) // T; hi_i = np.minimum(pats[:, 0] + pats[:, 2] + 1, L.nxl - 1) // T
    lo_j = np.maximum(pats[:, 1] - 2, 0) // T; hi_j = np.minimum(pats[:, 1] + pats[:, 3] + 1, L.nyl - 1) // T
    need = set()
    for a0, a1, c0, c1 in set(zip(lo_i.tolist(), hi_i.tolist(), lo_j.tolist(), hi_j.tolist())):
        for tj in range(c0, c1 + 1):
            for ti in range(a0, a1 + 1):
                need.add((ti, tj))
    return need


def set_bathy_from_canvas(L, wl):
    """b of every patch of L from a canvas over the whole level that lives with the backend (device memory for the CUDA path):
    the tiles the patches touch are evaluated and put on the canvas once, then one set_global gathers every storage cell inside the
    level.  Same values as wl.bathy_box patch by patch: a cell's value does not depend on who asks."""
    T = wl.TILE
    store = wl.__dict__.setdefault("_canvas", {})
    key = (id(L.ctx), L.dx, L.dy, int(L.nxl), int(L.nyl))
    if key not in store:
        store[key] = (L.ctx, L.ctx.canvas_new(L.nyl, L.nxl), set())
    _, canvas, have = store[key]
    for ti, tj in _tiles_needed(L, T) - have:
        t = wl.bathy_tile(L.dx, L.dy, ti, tj)
        h, w = min(T, int(L.nyl) - tj * T), min(T, int(L.nxl) - ti * T)
        L.ctx.canvas_put(canvas, tj * T, ti * T, t[:h, :w])
        have.add((ti, tj))
    L.set_global("b", canvas)


def pack_bathy_native(L, wl):
    """every patch's storage-shaped bathymetry block, back to back, copied from the workload's tile cache in one native call
    (amr_pack_from_tiles); the tiles a patch touches are evaluated first where the cache does not hold them yet.  Same values
    as wl.bathy_box patch by patch (tests/test_harness_pins.py): a cell's value does not depend on who asks."""
    import ctypes as C
    pats = np.ascontiguousarray(L.patches, dtype=np.int32)
    T = wl.TILE
    ntx, nty = (int(L.nxl) + T - 1) // T, (int(L.nyl) + T - 1) // T
    lo_i = np.maximum(pats[:, 0] - 2, 0) // T; hi_i = np.minimum(pats[:, 0] + pats[:, 2] + 1, L.nxl - 1) // T
    lo_j = np.maximum(pats[:, 1] - 2, 0) // T; hi_j = np.minimum(pats[:, 1] + pats[:, 3] + 1, L.nyl - 1) // T
    need = set()
    for a0, a1, c0, c1 in set(zip(lo_i.tolist(), hi_i.tolist(), lo_j.tolist(), hi_j.tolist())):
        for tj in range(c0, c1 + 1):
            for ti in range(a0, a1 + 1):
                need.add((ti, tj))
    table = np.zeros(ntx * nty, dtype=np.uint64)
    keep = []
    for ti, tj in need:
        t = wl.bathy_tile(L.dx, L.dy, ti, tj)
        keep.append(t)
        table[tj * ntx + ti] = t.ctypes.data
    n = int(((pats[:, 2].astype(np.int64) + 4) * (pats[:, 3] + 4)).sum())
    out = np.empty(n, dtype=np.float64)
    lib = native()
    lib.amr_pack_from_tiles.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
    rc = lib.amr_pack_from_tiles(table.ctypes.data, ntx, nty, T, pats.ctypes.data, len(pats), int(L.nxl), int(L.nyl), out.ctypes.data)
    assert rc == 0, "tile missing"
    del keep
    return out


def level_bbox(L):
    """bounding box (i0, j0, i1, j1) of the patches of a level, grown by one cell and clipped to the domain"""
    p = np.asarray(L.patches)
    i0 = max(int(p[:, 0].min()) - 1, 0); j0 = max(int(p[:, 1].min()) - 1, 0)
    i1 = min(int((p[:, 0] + p[:, 2]).max()) + 1, L.nxl); j1 = min(int((p[:, 1] + p[:, 3]).max()) + 1, L.nyl)
    return i0, j0, i1, j1


def unpack_cells(L, packed, fill=0, bbox=None):
    """interior-packed per-patch array (flags, masks) -> 2-D array over the level (or over bbox = (i0, j0, i1, j1))"""
    bi, bj, ei, ej = (0, 0, L.nxl, L.nyl) if bbox is None else bbox
    out = np.full((ej - bj, ei - bi), fill, dtype=packed.dtype)
    o = 0
    for i0, j0, nx, ny in L.patches:
        out[j0 - bj:j0 - bj + ny, i0 - bi:i0 - bi + nx] = packed[o:o + nx * ny].reshape(ny, nx)
        o += nx * ny
    return out


def nesting_mask(L, bbox=None):
    """Cells of level L whose 3x3 neighbourhood (clipped to the domain) lies inside the level: a finer patch on
    top of them has every ghost cell over level-L interior cells (proper nesting by one coarse cell).
    Over the whole level, or over bbox = (i0, j0, i1, j1)."""
    bi, bj, ei, ej = (0, 0, L.nxl, L.nyl) if bbox is None else bbox
    nx_, ny_ = ei - bi, ej - bj
    cov = np.zeros((ny_ + 2, nx_ + 2), dtype=bool)      # index (j - bj + 1, i - bi + 1)
    if bj == 0: cov[0, :] = True                         # outside the domain counts as fine (physical BC)
    if ej == L.nyl: cov[-1, :] = True
    if bi == 0: cov[:, 0] = True
    if ei == L.nxl: cov[:, -1] = True
    for i0, j0, nx, ny in L.patches:
        a0, a1 = max(i0 - bi + 1, 0), min(i0 - bi + 1 + nx, nx_ + 2)
        c0, c1 = max(j0 - bj + 1, 0), min(j0 - bj + 1 + ny, ny_ + 2)
        if a0 < a1 and c0 < c1:
            cov[c0:c1, a0:a1] = True
    ok = np.ones((ny_, nx_), dtype=bool)
    for dj in (0, 1, 2):
        for di in (0, 1, 2):
            ok &= cov[dj:dj + ny_, di:di + nx_]
    return ok


class GaugeRecorder:
    """Gauges (reading S-19): host bookkeeping around the backends' sampling call.  Each gauge belongs to
    the finest level whose interior holds it (re-decided after every regrid); a level's gauges are sampled right after its ghost
    fill and before its step, and once more at the end of the run.  records[g] = list of (t, h, hu, hv, eta).
    device_series=True (CUDA backend only): samples go into a device tensor per level, one small kernel per record and no
    copy; they are read back when the assignment changes and at the end."""

    def __init__(self, xy, device_series=False, capacity=4096):
        self.xy = np.ascontiguousarray(xy, dtype=np.float64).reshape(-1, 2)
        self.records = [[] for _ in range(len(self.xy))]
        self.device_series = device_series
        self.capacity = capacity
        self.assign = []            # per level: (gauge ids, patch ids)
        self._series = []           # per level (device path): [level object, tensor capacity x n x 4, list of times]

    @staticmethod
    def patch_of(L, x, y):
        ic = np.floor((x - L.xlo) / L.dx); jc = np.floor((y - L.ylo) / L.dy)
        p = np.asarray(L.patches)
        hit = np.nonzero((p[:, 0] <= ic) & (ic < p[:, 0] + p[:, 2]) & (p[:, 1] <= jc) & (jc < p[:, 1] + p[:, 3]))[0]
        return int(hit[0]) if len(hit) else -1

    def rebind(self, levels):
        self.flush()
        owner = [None] * len(self.xy)
        for k in reversed(range(len(levels))):                      # finest level first
            for g, (x, y) in enumerate(self.xy):
                if owner[g] is None:
                    pch = self.patch_of(levels[k], x, y)
                    if pch >= 0:
                        owner[g] = (k, pch)
        self.assign = []
        for k in range(len(levels)):
            ids = [g for g, o in enumerate(owner) if o is not None and o[0] == k]
            self.assign.append((ids, [owner[g][1] for g in ids]))
        self._series = []
        if self.device_series:
            for k, L in enumerate(levels):
                ids, pats = self.assign[k]
                L.gauges_bind(pats, self.xy[ids])
                buf = L.ctx.torch.empty((self.capacity, max(len(ids), 1), 4), dtype=L.ctx.torch.float64, device=L.ctx.device) if ids else None
                self._series.append([L, buf, []])

    def record(self, k, L, t):
        ids, pats = self.assign[k]
        if not ids:
            return
        if self.device_series:
            lev, buf, times = self._series[k]
            if len(times) == self.capacity:
                self.flush(only=k)
                lev, buf, times = self._series[k]
            L.gauges_sample_into(buf[len(times)])
            times.append(t)
        else:
            out = L.gauges_sample(pats, self.xy[ids])
            for n, g in enumerate(ids):
                self.records[g].append((t,) + tuple(float(v) for v in out[n]))

    def flush(self, only=None):
        """device path: read the finished part of every series back and append it to the records"""
        for k, ser in enumerate(self._series):
            if (only is not None and k != only) or ser[1] is None or not ser[2]:
                continue
            lev, buf, times = ser
            host = buf[:len(times)].cpu().numpy()
            for n, g in enumerate(self.assign[k][0]):
                for r, t in enumerate(times):
                    self.records[g].append((t,) + tuple(float(v) for v in host[r, n]))
            ser[2] = []

    def series(self, g):
        """records of gauge g sorted by time, as an array n x 5 (t, h, hu, hv, eta)"""
        self.flush()
        return np.array(sorted(self.records[g]), dtype=np.float64).reshape(-1, 5)


class Hierarchy:
    """The AMR recursion of P:140-146 (steps 1-5) with regridding every `regrid_interval` steps of a level,
    driving one backend through the C-ABI calls.  Bookkeeping only."""

    def __init__(self, ctx, wl, max_levels=None, reflux=True, patches1=None, efficiency=0.7, gauges=None, keep_unchanged=True,
                 accumulate=True):
        self.ctx, self.wl, self.reflux, self.eff = ctx, wl, reflux, efficiency
        self.gauges = gauges             # GaugeRecorder or None
        # a backend with step_accum / stats_reset (the CUDA path) is not waited for step by step: the levels' statistics accumulate
        # on the device and are read once per coarse step and before a level is replaced (same numbers: a max of maxima)
        self.accumulate = accumulate
        self.keep_unchanged = keep_unchanged   # keep a level whose regrid reproduces its patch list (bit-identical to recreating it)
        self.reuse_box_flags = keep_unchanged  # and do not re-flag a level whose flags can only come from unchanged forced boxes
        self._boxflag_cache = {}
        self._attached = {}              # level index k -> (coarse, fine) level objects whose flux registers are attached
        self.kept = 0
        nl = 1 + len(wl.ratios) if max_levels is None else min(max_levels, 1 + len(wl.ratios))
        self.ratios = list(wl.ratios)[:nl - 1]
        self.levels = [setup_level(ctx, wl, patches=patches1)]
        self.t = 0.0
        self.alpha_now = [1.0]          # time of level l inside the last step of level l-1, as a fraction
        self.steps = [0]
        self.sdx = [0.0]
        self.updates = 0
        self.flag_log = []              # (level index, t, packed flags) of every flagging pass, for parity checks
        self.regrids = 0
        self._regrid(0, initial=True)

    # ---- geometry of level index k (0-based)
    def _geom(self, k):
        R = 1
        for r in self.ratios[:k]:
            R *= r
        return self.wl.dx / R, self.wl.dy / R, self.wl.nx * R, self.wl.ny * R

    def _flag_boxes(self, k, t):
        """flag level k at its current time t, cluster -> patches of level k+1 (in cells of level k+1), or None"""
        L = self.levels[k]
        f = dict(self.wl.flag)
        # a box that refines level lv -> lv + 1 needs every coarser level underneath: it flags levels 1..lv
        boxes = [b[1:] for b in self.wl.forced_boxes if b[0] >= k + 1]
        wave = k + 1 <= self.wl.wave_levels and f.get("tol_eta", 0.0) > 0.0
        # nothing can flag this level now (no wave criterion here, no box whose window [t0, t1] holds t -- the test the
        # flag kernel applies): the pass would return no flags, so it is not launched and nothing is downloaded
        if not wave and not any(b[4] <= t <= b[5] for b in boxes):
            return None
        # flags that come from forced boxes alone are a function of the level's patch list and of the set of active boxes: a level
        # that regrids every few of its steps over the same patches inside the same boxes is not flagged again (no launch, no
        # download, no clustering; the flagging passes that are run are still logged for the parity check)
        ckey = None
        if not wave and self.reuse_box_flags:
            ckey = (k, np.ascontiguousarray(L.patches).tobytes(), tuple(b for b in boxes if b[4] <= t <= b[5]))
            hit = self._boxflag_cache.get(k)
            if hit is not None and hit[0] == ckey:
                return None if hit[1] is None else hit[1].copy()
        pats = self._flag_and_cluster(k, t, L, f, wave, boxes)
        if ckey is not None:
            self._boxflag_cache[k] = (ckey, None if pats is None else pats.copy())
        return pats

    def _flag_and_cluster(self, k, t, L, f, wave, boxes):
        packed, n = L.flag(tol_eta=f.get("tol_eta", 0.0) if wave else 0.0, tol_slope=0.0, offshore_only=f.get("offshore_only", 0),
                           buffer=f.get("buffer", 0), boxes=boxes, t=t)
        self.flag_log.append((k, t, packed.copy()))
        if n == 0:
            return None
        bbox = level_bbox(L)
        fl = unpack_cells_native(L, packed, bbox).view(bool)          # bytes 0 / 1
        # everything below happens inside the bounding box of the flags (clustering starts by shrinking to it anyway)
        rows = np.flatnonzero(fl.any(axis=1)); cols = np.flatnonzero(fl.any(axis=0))
        bbox = (bbox[0] + int(cols[0]), bbox[1] + int(rows[0]), bbox[0] + int(cols[-1]) + 1, bbox[1] + int(rows[-1]) + 1)
        fl = np.ascontiguousarray(fl[rows[0]:rows[-1] + 1, cols[0]:cols[-1] + 1])
        ok = nesting_mask_native(L, bbox)
        fl &= ok
        if not fl.any():
            return None
        r = self.ratios[k]
        boxes = cluster_native(fl, valid=ok, efficiency=self.eff, max_side=max(1, self.wl.patch_max // r))
        return np.array([[(b[0] + bbox[0]) * r, (b[1] + bbox[1]) * r, b[2] * r, b[3] * r] for b in boxes], dtype=np.int32)

    def _accum(self, L):
        return self.accumulate and hasattr(L, "step_accum")

    def _harvest(self, k, L):
        """the statistics level k's steps left on the device since the last harvest -> self.sdx[k]"""
        if not self._accum(L):
            return
        st = L.stats()
        if st["nan_seen"]:
            raise RuntimeError("NaN in the updated state of level %d" % (k + 1))
        self.sdx[k] = max(self.sdx[k], st["s_over_dx_max"])
        L.stats_reset()

    def _regrid(self, k0, initial=False, t=None):
        """rebuild levels k0+1.. from the flags of the level below each; t = the time the levels k0.. have reached
        (a level regrids at the end of one of its own steps, when it and every finer level stand at the same time)"""
        t = self.t if t is None else t
        self.regrids += 0 if initial else 1
        for k in range(k0, len(self.ratios)):
            if k >= len(self.levels):
                break
            C = self.levels[k]
            pats = self._flag_boxes(k, t)
            old = self.levels[k + 1] if k + 1 < len(self.levels) else None
            if pats is None:
                for L in self.levels[k + 1:]:
                    L.destroy()
                del self.levels[k + 1:]; del self.alpha_now[k + 1:]; del self.steps[k + 1:]; del self.sdx[k + 1:]
                break
            if self.keep_unchanged and not initial and old is not None and np.array_equal(pats, old.patches):
                # the regrid reproduced the level's patch list (always so for a level defined by forced boxes).  The regrid transfer
                # would copy every interior cell from the old level, and every ghost cell is rewritten before it is read (DESIGN.md
                # 3.6), so the level stays as it is: bit-identical to recreating it (tests/test_oracle_amr.py)
                C.fill_ghost(self.levels[k - 1] if k > 0 else None, self.alpha_now[k])
                a = self._attached.get(k)
                if self.reflux and not (a is not None and a[0] is C and a[1] is old):
                    C.flux_attach(old)             # (else both levels are unchanged and their registers just fixed up and re-zeroed)
                    self._attached[k] = (C, old)
                self.kept += 1
                continue
            dx, dy, nxl, nyl = self._geom(k + 1)
            N = self.ctx.level_create(k + 2, self.wl.xlo, self.wl.ylo, dx, dy, nxl, nyl, self.ratios[k], pats)
            set_initial(N, self.wl, state=initial)
            deform_to(N, self.wl, t)             # the new level's bathymetry at the regrid time, before it is interpolated onto
            if not initial:
                C.fill_ghost(self.levels[k - 1] if k > 0 else None, self.alpha_now[k])
                N.init_from(old, C)
            if old is not None:
                if not initial:
                    self._harvest(k + 1, old)
                old.destroy()
                self.levels[k + 1] = N
            else:
                self.levels.append(N); self.alpha_now.append(1.0); self.steps.append(0); self.sdx.append(0.0)
            if self.reflux:
                C.flux_attach(N)
                self._attached[k] = (C, N)
        if self.gauges is not None:
            self.gauges.rebind(self.levels)

    def probe(self):
        """dt of level 1 from dt = 0 probe steps of every level"""
        m, R = 0.0, 1
        for k, L in enumerate(self.levels):
            R = R * (self.ratios[k - 1] if k > 0 else 1)
            L.fill_ghost(self.levels[k - 1] if k > 0 else None, self.alpha_now[k])
            m = max(m, L.step(0.0)["s_over_dx_max"] / R)
        return self.wl.cfl / m

    def _advance(self, k, dt, alpha, t):
        """one step of level k from its time t (alpha: that time as a fraction of the coarser level's current step)"""
        L = self.levels[k]
        deform_to(L, self.wl, t)                 # B(x, y, t) at the start of the step
        L.fill_ghost(self.levels[k - 1] if k > 0 else None, alpha)
        if self.gauges is not None:
            self.gauges.record(k, L, t)
        if self._accum(L):
            L.step_accum(dt)
        else:
            st = L.step(dt)
            self.sdx[k] = max(self.sdx[k], st["s_over_dx_max"])
        self.steps[k] += 1
        self.updates += L.ncells
        # the step wrote interior cells only: bring the new buffer's ghost ring to the new state's time before the finer level's
        # substeps read it as slope neighbours on patch seams; alpha_now[k] is that time as a fraction.  The finest
        # level has no such reader: its ring is next read by its own next step, whose fill rewrites it (and a regrid that puts a
        # level on top of it fills first), so the fill is left out there -- same numbers, a fifth of that level's launches
        if k + 1 < len(self.levels):
            L.fill_ghost(self.levels[k - 1] if k > 0 else None, self.alpha_now[k])
        if k + 1 < len(self.levels):
            r = self.ratios[k]
            for s in range(r):
                self.alpha_now[k + 1] = (s + 1) / r
                self._advance(k + 1, dt / r, s / r, t + s * (dt / r))
        if k + 1 < len(self.levels):        # the finer level may have vanished in a regrid below
            F = self.levels[k + 1]
            if self.reflux:
                L.flux_fixup(F)
            L.average_down_from(F)
        if k > 0 and k < len(self.ratios) and self.steps[k] % self.wl.regrid_interval == 0:
            self._regrid(k, t=t + dt)

    def step(self, dt):
        """one step of level 1 (and everything above it); returns the next dt of level 1"""
        self.sdx = [0.0] * len(self.levels)
        self.alpha_now[0] = 1.0
        for L in self.levels:
            if self._accum(L):
                L.stats_reset()
        self._advance(0, dt, 1.0, self.t)
        self.t += dt
        if len(self.ratios) > 0 and self.steps[0] % self.wl.regrid_interval == 0:
            self._regrid(0)
        for k, L in enumerate(self.levels):
            self._harvest(k, L)
        m, R = 0.0, 1
        for k in range(len(self.sdx)):
            R = R * (self.ratios[k - 1] if k > 0 else 1)
            m = max(m, self.sdx[k] / R)
        return self.wl.cfl / m

    def run(self, nsteps=None, t_end=None, record=None):
        dt = self.probe()
        n = 0
        while (nsteps is None or n < nsteps) and (t_end is None or self.t < t_end):
            if t_end is not None and self.t + dt > t_end:
                dt = t_end - self.t
            dtn = self.step(dt)
            if record is not None:
                record(n, dt, self)
            dt = dtn
            n += 1
        self.record_gauges_now()
        return n

    def record_gauges_now(self):
        """one record of every gauge at the hierarchy's current time (all levels are at self.t between coarse steps)"""
        if self.gauges is None:
            return
        for k, L in enumerate(self.levels):
            L.fill_ghost(self.levels[k - 1] if k > 0 else None, 1.0)
            self.gauges.record(k, L, self.t)

    def composite_mass(self):
        """mass over the finest available cells: sum over levels of the mass of cells not covered by a finer level.
        Needs get_global on every level (small test problems only)."""
        tot = 0.0
        for k, L in enumerate(self.levels):
            h = L.get_global("h", fill=0.0)
            kap = self._kappa(L)
            w = np.ones_like(h, dtype=bool)
            cov = np.zeros_like(w)
            for i0, j0, nx, ny in L.patches:
                cov[j0:j0 + ny, i0:i0 + nx] = True
            w &= cov
            if k + 1 < len(self.levels):
                r = self.ratios[k]
                for i0, j0, nx, ny in self.levels[k + 1].patches:
                    w[j0 // r:(j0 + ny) // r, i0 // r:(i0 + nx) // r] = False
            tot += float((h * kap[:, None] * (L.dx * L.dy))[w].sum())
        return tot

    def _kappa(self, L):
        if self.wl.params.get("coord", 0) == 0:
            return np.ones(L.nyl)
        R = self.wl.params.get("earth_radius", 6367500.0)
        d2r = np.pi / 180.0
        lat0 = (L.ylo + np.arange(L.nyl) * L.dy) * d2r
        lat1 = (L.ylo + (np.arange(L.nyl) + 1) * L.dy) * d2r
        return d2r * R * R * (np.sin(lat1) - np.sin(lat0)) / L.dy

    def destroy(self):
        for L in self.levels:
            L.destroy()
        self.levels = []
