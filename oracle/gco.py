"""ORACLE binding (test infrastructure, NOT the product).

ctypes wrapper around oracle/libgco.so (plain C, fp64, single thread; see oracle/gco.h).  Exposes the
same Python method names as paper_1901_06798_b200.binding so the AMR driver can run on either.  Only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = ["gco_riemann.c", "gco_sweep.c", "gco_level.c", "gco_amr.c", "gco_flux.c", "gco_bathy.c", "gco_unsplit.c"]
_LIB = os.path.join(_DIR, "libgco.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-Wall", "-shared", "-fPIC", "-fopenmp"]


def _cpu_has_fma():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return " fma " in line + " "
    except OSError:
        pass
    return False


def _flags():
    """-mfma where the host has it: the C99 fma() calls DESIGN.md 3.1 specifies then compile to the hardware instruction instead
    of a libm call (same correctly rounded result either way; -ffp-contract=off still forbids every other contraction)"""
    return CFLAGS + (["-mfma"] if _cpu_has_fma() else [])


def build(force=False):
    srcs = [os.path.join(_DIR, s) for s in _SRC]
    deps = srcs + [os.path.join(_DIR, "gco.h"), os.path.join(_DIR, "gco_int.h")]
    tag = os.path.join(_DIR, "libgco.flags")
    want = " ".join(_flags())
    have = open(tag).read() if os.path.exists(tag) else ""
    if not force and have == want and os.path.exists(_LIB) and all(os.path.getmtime(_LIB) >= os.path.getmtime(d) for d in deps):
        return _LIB
    subprocess.check_call(["gcc"] + _flags() + ["-o", _LIB] + srcs + ["-lm"])
    with open(tag, "w") as f:          # a library built for another host's instruction set (it travels with the tree) is rebuilt
        f.write(want)
    return _LIB


class Params(C.Structure):
    _fields_ = [("coord", C.c_int), ("g", C.c_double), ("dry_tol", C.c_double), ("sea_level", C.c_double),
                ("earth_radius", C.c_double), ("limiter", C.c_int), ("bc", C.c_int * 4),
                ("manning_n", C.c_double), ("friction_depth", C.c_double)]


class FlagParams(C.Structure):
    _fields_ = [("tol_eta", C.c_double), ("tol_slope", C.c_double), ("offshore_only", C.c_int),
                ("buffer", C.c_int), ("nboxes", C.c_int), ("boxes", C.POINTER(C.c_double))]


class Deform(C.Structure):
    _fields_ = [("x0", C.c_double), ("y0", C.c_double), ("ddx", C.c_double), ("ddy", C.c_double),
                ("mx", C.c_int64), ("my", C.c_int64), ("dz", C.POINTER(C.c_double))]


def make_deform(x0, y0, ddx, ddy, dz):
    """-> (Deform, array kept alive): dz is (my, mx), node (m, n) at (x0 + m ddx, y0 + n ddy)"""
    a = np.ascontiguousarray(dz, dtype=np.float64)
    d = Deform(float(x0), float(y0), float(ddx), float(ddy), a.shape[1], a.shape[0], a.ctypes.data_as(C.POINTER(C.c_double)))
    return d, a


def deform_at(x0, y0, ddx, ddy, dz, x, y):
    d, keep = make_deform(x0, y0, ddx, ddy, dz)
    f = lib().gco_deform_at; f.restype = C.c_double; f.argtypes = [C.POINTER(Deform), C.c_double, C.c_double]
    return f(C.byref(d), float(x), float(y))


class StepStats(C.Structure):
    _fields_ = [("cfl_max", C.c_double), ("s_over_dx_max", C.c_double), ("clipped_mass", C.c_double),
                ("n_clipped", C.c_int64), ("nan_seen", C.c_int32)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.gco_level_mass.restype = C.c_double
        _lib.gco_level_ncells.restype = C.c_int64
        _lib.gco_riemann.argtypes = [C.c_double] * 10 + [_dp, _dp]
        _lib.gco_middle_state.argtypes = [C.c_double] * 8 + [_dp, _dp, _dp]
        _lib.gco_level_create.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                          C.c_int64, C.c_int64, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        _lib.gco_level_set_field.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int64]
        _lib.gco_level_get_field.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_int64]
        _lib.gco_level_set_global.argtypes = [C.c_void_p, C.c_int, C.c_void_p] + [C.c_int64] * 5
        _lib.gco_level_get_global.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p] + [C.c_int64] * 5
        _lib.gco_fill_ghost.argtypes = [C.c_void_p, C.c_void_p, C.c_double]
        _lib.gco_fill_ghost_b.argtypes = [C.c_void_p]
        _lib.gco_level_step.argtypes = [C.c_void_p, C.c_double, C.c_void_p]
        _lib.gco_wet_mask.argtypes = [C.c_void_p, C.c_void_p]
        _lib.gco_level_mass.argtypes = [C.c_void_p]
        _lib.gco_level_ncells.argtypes = [C.c_void_p]
        _lib.gco_flag_cells.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        _lib.gco_average_down.argtypes = [C.c_void_p, C.c_void_p]
        _lib.gco_level_init_from.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.gco_flux_attach.argtypes = [C.c_void_p, C.c_void_p]
        _lib.gco_flux_fixup.argtypes = [C.c_void_p, C.c_void_p]
        _lib.gco_level_metric.argtypes = [C.c_void_p] * 5
        _lib.gco_level_destroy.argtypes = [C.c_void_p]
        _lib.gco_ctx_destroy.argtypes = [C.c_void_p]
        _lib.gco_sweep_line.argtypes = [C.c_void_p, C.c_int] + [C.c_void_p] * 6 + [C.c_double] + [C.c_void_p] * 5 + [C.c_int, C.c_void_p]
    return _lib


def set_threads(n):
    """threads of the level step's loop over patches (default 1); returns the number in use.  n = 0: all host cores."""
    n = (os.cpu_count() or 1) if n == 0 else int(n)
    _chk(lib().gco_set_threads(n), "set_threads")
    return lib().gco_get_threads()


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError("oracle %s failed: %d" % (what, rc))


def make_params(coord=0, g=9.81, dry_tol=1e-3, sea_level=0.0, earth_radius=6367500.0, limiter=1, bc=(1, 1, 1, 1),
                manning_n=0.0, friction_depth=1.0e6):
    p = Params()
    p.coord, p.g, p.dry_tol, p.sea_level, p.earth_radius, p.limiter = coord, g, dry_tol, sea_level, earth_radius, limiter
    p.manning_n, p.friction_depth = manning_n, friction_depth
    for i in range(4):
        p.bc[i] = int(bc[i])
    return p


def cbrt(x):
    """the fixed cube-root sequence of DESIGN.md 3.9"""
    f = lib().gco_cbrt; f.restype = C.c_double; f.argtypes = [C.c_double]
    return f(float(x))


def friction(dt, h, hu, hv, **kw):
    """one cell's friction step -> (hu, hv)"""
    p = make_params(**kw)
    a, b = C.c_double(hu), C.c_double(hv)
    f = lib().gco_friction; f.restype = None
    f.argtypes = [C.POINTER(Params), C.c_double, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    f(C.byref(p), float(dt), float(h), C.byref(a), C.byref(b))
    return a.value, b.value


def transverse(g, eps, h, pn, pt, a):
    """split of the vector a (target frame) by the target direction's Jacobian at (h, pn, pt) -> (bm, bp)"""
    bm = np.zeros(3); bp = np.zeros(3); av = np.ascontiguousarray(a, dtype=np.float64)
    f = lib().gco_transverse; f.restype = None; f.argtypes = [C.c_double] * 5 + [_dp, _dp, _dp]
    f(g, eps, h, pn, pt, av.ctypes.data_as(_dp), bm.ctypes.data_as(_dp), bp.ctypes.data_as(_dp))
    return bm, bp


def riemann(g, eps, hL, pL, tL, bL, hR, pR, tR, bR):
    Z = np.zeros((3, 3)); s = np.zeros(3)
    lib().gco_riemann(g, eps, hL, pL, tL, bL, hR, pR, tR, bR, Z.ctypes.data_as(_dp), s.ctypes.data_as(_dp))
    return Z, s


def middle_state(g, eps, hL, hR, uL, uR):
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    lib().gco_middle_state(g, eps, hL, hR, uL, uR, np.sqrt(g * hL), np.sqrt(g * hR), C.byref(a), C.byref(b), C.byref(c))
    return a.value, b.value, c.value


def sweep_line(params, h, p, t, b, rdx, efac, dt, want_flux=False):
    """One 1-D sweep over a line with 2 ghost cells each side; returns updated (h, p, t) (ghosts copied) and max s*rdx."""
    n = len(h) - 4
    arr = [np.ascontiguousarray(a, dtype=np.float64) for a in (h, p, t, b, rdx, efac)]
    out = [a.copy() for a in arr[:3]]
    fm = np.zeros((n + 4) * 3); fp = np.zeros((n + 4) * 3)
    sdx = C.c_double(0.0)
    lib().gco_sweep_line(C.byref(params), n, *[a.ctypes.data for a in arr], dt, *[a.ctypes.data for a in out],
                         fm.ctypes.data, fp.ctypes.data, 1, C.byref(sdx))
    if want_flux:
        return out[0], out[1], out[2], sdx.value, fm.reshape(-1, 3), fp.reshape(-1, 3)
    return out[0], out[1], out[2], sdx.value


FIELDS = {"h": 0, "hu": 1, "hv": 2, "b": 3}


class Level:
    def __init__(self, ctx, level, xlo, ylo, dx, dy, nxl, nyl, ratio, patches):
        self.ctx = ctx
        self.level, self.xlo, self.ylo, self.dx, self.dy = level, xlo, ylo, dx, dy
        self.nxl, self.nyl, self.ratio = int(nxl), int(nyl), int(ratio)
        self.patches = np.ascontiguousarray(patches, dtype=np.int32).reshape(-1, 4)
        h = C.c_void_p()
        _chk(lib().gco_level_create(ctx.h, level, xlo, ylo, dx, dy, nxl, nyl, ratio, len(self.patches),
                                    self.patches.ctypes.data, C.byref(h)), "level_create")
        self.h = h
        self.ncells = int((self.patches[:, 2].astype(np.int64) * self.patches[:, 3]).sum())

    def destroy(self):
        if self.h:
            lib().gco_level_destroy(self.h); self.h = None

    def set_field(self, p, field, arr):
        a = np.ascontiguousarray(arr, dtype=np.float64)
        _chk(lib().gco_level_set_field(self.h, p, FIELDS[field], a.ctypes.data, a.shape[1]), "set_field")

    def get_field(self, p, field, which=0):
        nx, ny = int(self.patches[p, 2]), int(self.patches[p, 3])
        a = np.empty((ny + 4, nx + 4))
        _chk(lib().gco_level_get_field(self.h, p, FIELDS[field], which, a.ctypes.data, nx + 4), "get_field")
        return a

    def set_global(self, field, arr, gi0=0, gj0=0):
        a = np.ascontiguousarray(arr, dtype=np.float64)
        _chk(lib().gco_level_set_global(self.h, FIELDS[field], a.ctypes.data, a.shape[1], gi0, gj0, a.shape[1], a.shape[0]), "set_global")

    def set_patches(self, field, packed):
        """the CUDA binding's call shape: every patch's storage-shaped block (ghost cells included), back to back"""
        a = np.ascontiguousarray(packed, dtype=np.float64).ravel()
        o = 0
        for p, (i0, j0, nx, ny) in enumerate(self.patches):
            n = (nx + 4) * (ny + 4)
            self.set_field(p, field, a[o:o + n].reshape(ny + 4, nx + 4))
            o += n
        assert o == a.size

    def get_global(self, field, which=0, gi0=0, gj0=0, gnx=None, gny=None, fill=np.nan):
        gnx = self.nxl if gnx is None else gnx
        gny = self.nyl if gny is None else gny
        a = np.full((gny, gnx), fill)
        _chk(lib().gco_level_get_global(self.h, FIELDS[field], which, a.ctypes.data, gnx, gi0, gj0, gnx, gny), "get_global")
        return a

    def fill_ghost_b(self):
        _chk(lib().gco_fill_ghost_b(self.h), "fill_ghost_b")

    def fill_ghost(self, coarser=None, alpha=1.0):
        _chk(lib().gco_fill_ghost(self.h, coarser.h if coarser is not None else None, alpha), "fill_ghost")

    def step(self, dt):
        st = StepStats()
        _chk(lib().gco_level_step(self.h, dt, C.byref(st)), "level_step")
        return dict(cfl_max=st.cfl_max, s_over_dx_max=st.s_over_dx_max, clipped_mass=st.clipped_mass,
                    n_clipped=st.n_clipped, nan_seen=st.nan_seen)

    def step_unsplit(self, dt):
        """one unsplit level step with transverse Riemann solves"""
        st = StepStats()
        lib().gco_level_step_unsplit.argtypes = [C.c_void_p, C.c_double, C.c_void_p]
        _chk(lib().gco_level_step_unsplit(self.h, dt, C.byref(st)), "level_step_unsplit")
        return dict(cfl_max=st.cfl_max, s_over_dx_max=st.s_over_dx_max, clipped_mass=st.clipped_mass,
                    n_clipped=st.n_clipped, nan_seen=st.nan_seen)

    def gauges_sample(self, patch, xy):
        """(h, hu, hv, eta) at the points xy (n x 2), point k inside patch[k] -> n x 4"""
        patch = np.ascontiguousarray(patch, dtype=np.int32); xy = np.ascontiguousarray(xy, dtype=np.float64).reshape(-1, 2)
        out = np.empty((len(patch), 4))
        _chk(lib().gco_gauges_sample(self.h, len(patch), patch.ctypes.data_as(C.POINTER(C.c_int32)), xy.ctypes.data_as(_dp),
                                     out.ctypes.data_as(_dp)), "gauges_sample")
        return out

    def bathy_update(self, x0, y0, ddx, ddy, dz, w):
        """b <- fma(w, dz(cell centre), b); dz (my, mx) on the node grid (x0 + m ddx, y0 + n ddy)"""
        d, keep = make_deform(x0, y0, ddx, ddy, dz)
        lib().gco_bathy_update.argtypes = [C.c_void_p, C.POINTER(Deform), C.c_double]
        _chk(lib().gco_bathy_update(self.h, C.byref(d), float(w)), "bathy_update")

    def wet_mask(self):
        m = np.zeros(self.ncells, dtype=np.uint8)
        _chk(lib().gco_wet_mask(self.h, m.ctypes.data), "wet_mask")
        return m

    def mass(self):
        return lib().gco_level_mass(self.h)

    def flag(self, tol_eta=0.0, tol_slope=0.0, offshore_only=0, buffer=0, boxes=(), t=0.0):
        fp = FlagParams()
        bx = np.ascontiguousarray(np.array(boxes, dtype=np.float64).reshape(-1, 6))
        fp.tol_eta, fp.tol_slope, fp.offshore_only, fp.buffer, fp.nboxes = tol_eta, tol_slope, offshore_only, buffer, len(bx)
        fp.boxes = bx.ctypes.data_as(_dp)
        fl = np.zeros(self.ncells, dtype=np.uint8)
        n = C.c_int64(0)
        _chk(lib().gco_flag_cells(self.h, C.byref(fp), t, fl.ctypes.data, C.byref(n)), "flag_cells")
        return fl, n.value

    def average_down_from(self, fine):
        _chk(lib().gco_average_down(self.h, fine.h), "average_down")

    def init_from(self, old, coarse):
        _chk(lib().gco_level_init_from(self.h, old.h if old is not None else None, coarse.h), "init_from")

    def flux_attach(self, fine):
        _chk(lib().gco_flux_attach(self.h, fine.h), "flux_attach")

    def flux_fixup(self, fine):
        _chk(lib().gco_flux_fixup(self.h, fine.h), "flux_fixup")

    def metric(self):
        k = np.zeros(self.nyl + 4); rx = np.zeros(self.nyl + 4); ry = np.zeros(self.nyl + 4); ey = np.zeros(self.nyl + 5)
        lib().gco_level_metric(self.h, k.ctypes.data, rx.ctypes.data, ry.ctypes.data, ey.ctypes.data)
        return k, rx, ry, ey


class Context:
    """Oracle backend: Context(**params).level_create(...) -> Level."""
    name = "oracle"

    def __init__(self, **kw):
        self.params = make_params(**kw)
        self.kw = kw
        h = C.c_void_p()
        _chk(lib().gco_ctx_create(C.byref(self.params), C.byref(h)), "ctx_create")
        self.h = h

    def level_create(self, level, xlo, ylo, dx, dy, nxl, nyl, ratio, patches):
        return Level(self, level, xlo, ylo, dx, dy, nxl, nyl, ratio, patches)

    # the harness's bathymetry canvas (an array over a whole level, filled tile by tile, handed to set_global): host memory here
    def canvas_new(self, ny, nx):
        return np.zeros((int(ny), int(nx)))

    def canvas_put(self, canvas, j0, i0, block):
        canvas[j0:j0 + block.shape[0], i0:i0 + block.shape[1]] = block

    def destroy(self):
        if self.h:
            lib().gco_ctx_destroy(self.h); self.h = None
