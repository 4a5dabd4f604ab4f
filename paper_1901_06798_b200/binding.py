"""Thin Python binding of libgeoclaw_b200.so (include/gc.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory (through
the allocator callbacks), the stream and nothing else.  There is NO CPU fallback: importing works without a
GPU (so the symbols can be checked), but creating a Context without a CUDA device raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgeoclaw_b200.so")

SYMBOLS = [
    "gc_ctx_create", "gc_ctx_destroy", "gc_last_error", "gc_level_create", "gc_level_destroy", "gc_level_ncells",
    "gc_level_set_field", "gc_level_get_field", "gc_level_set_global", "gc_level_get_global", "gc_fill_ghost", "gc_fill_ghost_step",
    "gc_fill_ghost_b", "gc_level_step", "gc_level_step_auto", "gc_level_stats", "gc_wet_mask", "gc_level_mass",
    "gc_flag_cells", "gc_average_down", "gc_level_init_from", "gc_flux_attach", "gc_flux_fixup", "gc_probe_fp64_peak",
    "gc_launch_count", "gc_profile_enable", "gc_profile_read", "gc_selftest_math", "gc_gauges_bind", "gc_gauges_sample", "gc_level_set_patches",
    "gc_ctx_set_option", "gc_level_upload_state_async", "gc_level_download_state_async", "gc_bathy_update", "gc_level_fallback_counts", "gc_level_sweep_cells", "gc_level_step_unsplit",
    "gc_level_step_accum", "gc_level_stats_reset", "gc_level_step_unsplit_static", "gc_unsplit_static_max_cells",
]


class Params(C.Structure):
    _fields_ = [("coord", C.c_int), ("g", C.c_double), ("dry_tol", C.c_double), ("sea_level", C.c_double),
                ("earth_radius", C.c_double), ("limiter", C.c_int), ("bc", C.c_int * 4),
                ("manning_n", C.c_double), ("friction_depth", C.c_double)]


class Deform(C.Structure):
    _fields_ = [("x0", C.c_double), ("y0", C.c_double), ("ddx", C.c_double), ("ddy", C.c_double),
                ("mx", C.c_int64), ("my", C.c_int64), ("dz", C.c_void_p), ("dz_is_device", C.c_int)]


class FlagParams(C.Structure):
    _fields_ = [("tol_eta", C.c_double), ("tol_slope", C.c_double), ("offshore_only", C.c_int),
                ("buffer", C.c_int), ("nboxes", C.c_int), ("boxes", C.POINTER(C.c_double))]


class StepStats(C.Structure):
    _fields_ = [("cfl_max", C.c_double), ("s_over_dx_max", C.c_double), ("clipped_mass", C.c_double),
                ("n_clipped", C.c_int64), ("nan_seen", C.c_int32)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_lib = None


def lib():
    """Loads the extension; raises if it has not been built (python -m paper_1901_06798_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("CUDA extension missing: %s (run `python -m paper_1901_06798_b200.build`); "
                           "there is no CPU fallback" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i, d, i64 = C.c_void_p, C.c_int, C.c_double, C.c_int64
    L.gc_ctx_create.argtypes = [vp, vp, ALLOC_FN, FREE_FN, vp, vp]
    L.gc_ctx_destroy.argtypes = [vp]
    L.gc_ctx_set_option.argtypes = [vp, i, i64]
    L.gc_bathy_update.argtypes = [vp, vp, d]
    L.gc_level_fallback_counts.argtypes = [vp, vp]
    L.gc_level_sweep_cells.argtypes = [vp, vp]
    L.gc_level_upload_state_async.argtypes = [vp, vp, vp]
    L.gc_level_download_state_async.argtypes = [vp, vp, vp]
    L.gc_last_error.argtypes = [vp]; L.gc_last_error.restype = C.c_char_p
    L.gc_level_create.argtypes = [vp, i, d, d, d, d, i64, i64, i, i, vp, vp]
    L.gc_level_destroy.argtypes = [vp]
    L.gc_level_ncells.argtypes = [vp]; L.gc_level_ncells.restype = i64
    L.gc_level_set_field.argtypes = [vp, i, i, vp, i, i64]
    L.gc_level_get_field.argtypes = [vp, i, i, i, vp, i, i64]
    L.gc_level_set_global.argtypes = [vp, i, vp, i, i64, i64, i64, i64, i64]
    L.gc_level_get_global.argtypes = [vp, i, i, vp, i, i64, i64, i64, i64, i64]
    L.gc_fill_ghost.argtypes = [vp, vp, d]
    L.gc_fill_ghost_step.argtypes = [vp, vp, d]
    L.gc_fill_ghost_b.argtypes = [vp]
    L.gc_level_set_patches.argtypes = [vp, i, vp, i]
    L.gc_gauges_bind.argtypes = [vp, i, vp, vp]
    L.gc_gauges_sample.argtypes = [vp, vp, i]
    L.gc_level_step.argtypes = [vp, d, vp]
    L.gc_level_step_auto.argtypes = [vp, vp, d]
    L.gc_level_step_unsplit.argtypes = [vp, d, vp]
    L.gc_level_step_accum.argtypes = [vp, d]
    L.gc_level_step_unsplit_static.argtypes = [vp, d, vp]
    L.gc_unsplit_static_max_cells.argtypes = []; L.gc_unsplit_static_max_cells.restype = C.c_int64
    L.gc_level_stats_reset.argtypes = [vp]
    L.gc_level_stats.argtypes = [vp, vp]
    L.gc_wet_mask.argtypes = [vp, vp, i]
    L.gc_level_mass.argtypes = [vp]; L.gc_level_mass.restype = d
    L.gc_flag_cells.argtypes = [vp, vp, d, vp, i, vp]
    L.gc_average_down.argtypes = [vp, vp]
    L.gc_level_init_from.argtypes = [vp, vp, vp]
    L.gc_flux_attach.argtypes = [vp, vp]
    L.gc_flux_fixup.argtypes = [vp, vp]
    L.gc_probe_fp64_peak.argtypes = [vp, vp]
    L.gc_launch_count.argtypes = [vp]; L.gc_launch_count.restype = i64
    L.gc_profile_enable.argtypes = [vp, i]
    L.gc_profile_read.argtypes = [vp, vp, vp]
    L.gc_selftest_math.argtypes = [vp, vp, vp, i64, vp, vp]
    _lib = L
    return L


FIELDS = {"h": 0, "hu": 1, "hv": 2, "b": 3}


def _is_torch(x):
    return type(x).__module__.startswith("torch")


class Level:
    def __init__(self, ctx, level, xlo, ylo, dx, dy, nxl, nyl, ratio, patches):
        self.ctx = ctx
        self.level, self.xlo, self.ylo, self.dx, self.dy = level, xlo, ylo, dx, dy
        self.nxl, self.nyl, self.ratio = int(nxl), int(nyl), int(ratio)
        self.patches = np.ascontiguousarray(patches, dtype=np.int32).reshape(-1, 4)
        h = C.c_void_p()
        ctx._chk(lib().gc_level_create(ctx.h, level, xlo, ylo, dx, dy, nxl, nyl, ratio, len(self.patches),
                                       self.patches.ctypes.data, C.byref(h)), "gc_level_create")
        self.h = h
        self.ncells = int(lib().gc_level_ncells(h))

    def destroy(self):
        if self.h:
            lib().gc_level_destroy(self.h)
            self.h = None

    def _src(self, arr):
        if _is_torch(arr):
            assert arr.is_cuda and arr.dtype.is_floating_point and arr.element_size() == 8 and arr.stride(-1) == 1
            return arr, arr.data_ptr(), 1, arr.stride(0)
        a = np.ascontiguousarray(arr, dtype=np.float64)
        return a, a.ctypes.data, 0, a.shape[1]

    def set_field(self, p, field, arr):
        a, ptr, dev, ld = self._src(arr)
        self.ctx._chk(lib().gc_level_set_field(self.h, p, FIELDS[field], ptr, dev, ld), "gc_level_set_field")

    def get_field(self, p, field, which=0):
        nx, ny = int(self.patches[p, 2]), int(self.patches[p, 3])
        a = np.empty((ny + 4, nx + 4))
        self.ctx._chk(lib().gc_level_get_field(self.h, p, FIELDS[field], which, a.ctypes.data, 0, nx + 4), "gc_level_get_field")
        return a

    def set_global(self, field, arr, gi0=0, gj0=0):
        a, ptr, dev, ld = self._src(arr)
        self.ctx._chk(lib().gc_level_set_global(self.h, FIELDS[field], ptr, dev, ld, gi0, gj0, a.shape[1], a.shape[0]),
                      "gc_level_set_global")

    def set_patches(self, field, packed):
        """every patch at once: packed = for each patch in order its (ny + 4) x (nx + 4) block, ghost cells included, back to back"""
        a = np.ascontiguousarray(packed, dtype=np.float64).ravel()
        assert a.size == int(((self.patches[:, 2] + 4).astype(np.int64) * (self.patches[:, 3] + 4)).sum())
        self.ctx._chk(lib().gc_level_set_patches(self.h, FIELDS[field], a.ctypes.data, 0), "gc_level_set_patches")

    def get_global(self, field, which=0, gi0=0, gj0=0, gnx=None, gny=None, fill=np.nan, out=None):
        gnx = self.nxl if gnx is None else gnx
        gny = self.nyl if gny is None else gny
        if out is not None:  # device tensor supplied by the caller
            self.ctx._chk(lib().gc_level_get_global(self.h, FIELDS[field], which, out.data_ptr(), 1, out.stride(0),
                                                    gi0, gj0, gnx, gny), "gc_level_get_global")
            return out
        a = np.full((gny, gnx), fill)
        self.ctx._chk(lib().gc_level_get_global(self.h, FIELDS[field], which, a.ctypes.data, 0, gnx, gi0, gj0, gnx, gny),
                      "gc_level_get_global")
        return a

    def fill_ghost_b(self):
        self.ctx._chk(lib().gc_fill_ghost_b(self.h), "gc_fill_ghost_b")

    def fill_ghost(self, coarser=None, alpha=1.0):
        self.ctx._chk(lib().gc_fill_ghost(self.h, coarser.h if coarser is not None else None, alpha), "gc_fill_ghost")

    def fill_ghost_step(self, coarser=None, alpha=1.0):
        """gc_fill_ghost_step: the ghost cells the next split step reads (the rest may stay stale); same result of that step"""
        self.ctx._chk(lib().gc_fill_ghost_step(self.h, coarser.h if coarser is not None else None, alpha), "gc_fill_ghost_step")

    def step(self, dt, sync=True):
        if not sync:
            self.ctx._chk(lib().gc_level_step(self.h, dt, None), "gc_level_step")
            return None
        st = StepStats()
        self.ctx._chk(lib().gc_level_step(self.h, dt, C.byref(st)), "gc_level_step")
        return dict(cfl_max=st.cfl_max, s_over_dx_max=st.s_over_dx_max, clipped_mass=st.clipped_mass,
                    n_clipped=st.n_clipped, nan_seen=st.nan_seen)

    def step_accum(self, dt):
        """gc_level_step_accum: a step the host does not wait for; the level's statistics accumulate until stats_reset()"""
        self.ctx._chk(lib().gc_level_step_accum(self.h, dt), "gc_level_step_accum")

    def stats_reset(self):
        self.ctx._chk(lib().gc_level_stats_reset(self.h), "gc_level_stats_reset")

    def step_unsplit_static(self, dt, sync=True):
        """gc_level_step_unsplit_static: the unsplit step with its scratch in the library's static device array (allocates nothing;
        levels of at most gc_unsplit_static_max_cells() storage cells)"""
        if not sync:
            self.ctx._chk(lib().gc_level_step_unsplit_static(self.h, dt, None), "gc_level_step_unsplit_static")
            return None
        st = StepStats()
        self.ctx._chk(lib().gc_level_step_unsplit_static(self.h, dt, C.byref(st)), "gc_level_step_unsplit_static")
        return dict(cfl_max=st.cfl_max, s_over_dx_max=st.s_over_dx_max, clipped_mass=st.clipped_mass,
                    n_clipped=st.n_clipped, nan_seen=st.nan_seen)

    def step_unsplit(self, dt):
        """gc_level_step_unsplit: one unsplit level step with transverse Riemann solves"""
        st = StepStats()
        self.ctx._chk(lib().gc_level_step_unsplit(self.h, dt, C.byref(st)), "gc_level_step_unsplit")
        return dict(cfl_max=st.cfl_max, s_over_dx_max=st.s_over_dx_max, clipped_mass=st.clipped_mass,
                    n_clipped=st.n_clipped, nan_seen=st.nan_seen)

    def step_auto(self, dt_dev, cfl):
        """dt_dev: 1-element float64 CUDA tensor holding dt; updated in place to the next dt."""
        self.ctx._chk(lib().gc_level_step_auto(self.h, dt_dev.data_ptr(), cfl), "gc_level_step_auto")

    def bathy_update(self, x0, y0, ddx, ddy, dz, w):
        """gc_bathy_update: b <- fma(w, dz(cell centre), b); dz (my, mx) numpy array on the node grid (x0 + m ddx, y0 + n ddy)"""
        a = np.ascontiguousarray(dz, dtype=np.float64)
        d = Deform(float(x0), float(y0), float(ddx), float(ddy), a.shape[1], a.shape[0], a.ctypes.data, 0)
        self.ctx._chk(lib().gc_bathy_update(self.h, C.byref(d), C.c_double(float(w))), "gc_bathy_update")

    def upload_state_async(self, host3, copy_stream):
        """host3: three pinned CPU tensors (h, hu, hv) of shape (nyl, nxl), float64; copy_stream: a torch.cuda.Stream"""
        ptrs = (C.c_void_p * 3)(*[t.data_ptr() for t in host3])
        self.ctx._chk(lib().gc_level_upload_state_async(self.h, ptrs, C.c_void_p(copy_stream.cuda_stream)), "gc_level_upload_state_async")

    def download_state_async(self, host3, copy_stream):
        ptrs = (C.c_void_p * 3)(*[t.data_ptr() for t in host3])
        self.ctx._chk(lib().gc_level_download_state_async(self.h, ptrs, C.c_void_p(copy_stream.cuda_stream)), "gc_level_download_state_async")

    def sweep_cells(self):
        """gc_level_sweep_cells -> (x-sweep cells per launch over every row, without the unread ghost rows, y-sweep cells)"""
        out = (C.c_int64 * 3)()
        self.ctx._chk(lib().gc_level_sweep_cells(self.h, out), "gc_level_sweep_cells")
        return tuple(int(v) for v in out)

    def fallback_counts(self):
        """gc_level_fallback_counts -> dict(warp_iters, fb_warp_iters, fb_solves, fb_fluxes), cumulative for this level"""
        out = (C.c_int64 * 4)()
        self.ctx._chk(lib().gc_level_fallback_counts(self.h, out), "gc_level_fallback_counts")
        return dict(warp_iters=out[0], fb_warp_iters=out[1], fb_solves=out[2], fb_fluxes=out[3])

    def stats(self):
        st = StepStats()
        self.ctx._chk(lib().gc_level_stats(self.h, C.byref(st)), "gc_level_stats")
        return dict(cfl_max=st.cfl_max, s_over_dx_max=st.s_over_dx_max, clipped_mass=st.clipped_mass,
                    n_clipped=st.n_clipped, nan_seen=st.nan_seen)

    # ---- gauges
    def gauges_bind(self, patch, xy):
        """binds gauge k = point xy[k] inside the interior of patch[k]; replaces any earlier binding (empty lists unbind)"""
        patch = np.ascontiguousarray(patch, dtype=np.int32); xy = np.ascontiguousarray(xy, dtype=np.float64).reshape(-1, 2)
        self.ctx._chk(lib().gc_gauges_bind(self.h, len(patch), patch.ctypes.data, xy.ctypes.data), "gc_gauges_bind")
        self.ngauge = len(patch)

    def gauges_sample(self, patch=None, xy=None):
        """(h, hu, hv, eta) per gauge -> n x 4 on the host.  With patch, xy: binds them first (the oracle's call shape)."""
        if patch is not None:
            self.gauges_bind(patch, xy)
        out = np.empty((getattr(self, "ngauge", 0), 4))
        self.ctx._chk(lib().gc_gauges_sample(self.h, out.ctypes.data, 0), "gc_gauges_sample")
        return out

    def gauges_sample_into(self, row):
        """the same, written into a device tensor of at least 4 * ngauge float64 (a row of a device-resident series);
        enqueued on the context's stream, no synchronisation"""
        assert row.is_cuda and row.dtype == self.ctx.torch.float64 and row.is_contiguous() and row.numel() >= 4 * getattr(self, "ngauge", 0)
        self.ctx._chk(lib().gc_gauges_sample(self.h, row.data_ptr(), 1), "gc_gauges_sample")

    def wet_mask(self):
        m = np.zeros(self.ncells, dtype=np.uint8)
        self.ctx._chk(lib().gc_wet_mask(self.h, m.ctypes.data, 0), "gc_wet_mask")
        return m

    def mass(self):
        return lib().gc_level_mass(self.h)

    def flag(self, tol_eta=0.0, tol_slope=0.0, offshore_only=0, buffer=0, boxes=(), t=0.0):
        fp = FlagParams()
        bx = np.ascontiguousarray(np.array(boxes, dtype=np.float64).reshape(-1, 6))
        fp.tol_eta, fp.tol_slope, fp.offshore_only, fp.buffer, fp.nboxes = tol_eta, tol_slope, offshore_only, buffer, len(bx)
        fp.boxes = bx.ctypes.data_as(C.POINTER(C.c_double))
        fl = np.zeros(self.ncells, dtype=np.uint8)
        n = C.c_int64(0)
        self.ctx._chk(lib().gc_flag_cells(self.h, C.byref(fp), t, fl.ctypes.data, 0, C.byref(n)), "gc_flag_cells")
        return fl, n.value

    def average_down_from(self, fine):
        self.ctx._chk(lib().gc_average_down(self.h, fine.h), "gc_average_down")

    def init_from(self, old, coarse):
        self.ctx._chk(lib().gc_level_init_from(self.h, old.h if old is not None else None, coarse.h), "gc_level_init_from")

    def flux_attach(self, fine):
        self.ctx._chk(lib().gc_flux_attach(self.h, fine.h), "gc_flux_attach")

    def flux_fixup(self, fine):
        self.ctx._chk(lib().gc_flux_fixup(self.h, fine.h), "gc_flux_fixup")


OPT_SWEEP_FAMILY, OPT_MARCH_SEG, OPT_CHAINS = 0, 1, 2          # gc_ctx_set_option keys (include/gc.h)
SWEEP_AUTO, SWEEP_EDGE, SWEEP_MARCH = 0, 1, 2
DEFAULT_OPTIONS = {}                            # applied to every new Context (tests select a sweep kernel family here)


class Context:
    """The CUDA backend: Context(**params).level_create(...) -> Level.  Device memory comes from torch."""
    name = "b200"

    def __init__(self, coord=0, g=9.81, dry_tol=1e-3, sea_level=0.0, earth_radius=6367500.0, limiter=1,
                 bc=(1, 1, 1, 1), manning_n=0.0, friction_depth=1.0e6, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1901_06798_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._bufs = {}
        self._alloc_cb = ALLOC_FN(self._alloc)
        self._free_cb = FREE_FN(self._free)
        p = Params()
        p.coord, p.g, p.dry_tol, p.sea_level, p.earth_radius, p.limiter = coord, g, dry_tol, sea_level, earth_radius, limiter
        p.manning_n, p.friction_depth = manning_n, friction_depth
        for k in range(4):
            p.bc[k] = int(bc[k])
        self.params = p
        h = C.c_void_p()
        rc = lib().gc_ctx_create(C.byref(p), C.c_void_p(self.stream.cuda_stream), self._alloc_cb, self._free_cb, None, C.byref(h))
        if rc != 0:
            raise RuntimeError("gc_ctx_create failed: %d" % rc)
        self.h = h
        for key, value in DEFAULT_OPTIONS.items():
            self.set_option(key, value)

    # a device-resident array over a whole level that the harness fills tile by tile and hands to set_global (bathymetry canvas)
    def canvas_new(self, ny, nx):
        with self.torch.cuda.stream(self.stream):
            return self.torch.zeros((int(ny), int(nx)), dtype=self.torch.float64, device=self.device)

    def canvas_put(self, canvas, j0, i0, block):
        with self.torch.cuda.stream(self.stream):
            canvas[j0:j0 + block.shape[0], i0:i0 + block.shape[1]].copy_(self.torch.from_numpy(np.ascontiguousarray(block)))

    def set_option(self, key, value):
        """gc_ctx_set_option: tuning knobs that change no result bit (OPT_SWEEP_FAMILY, OPT_MARCH_SEG, OPT_CHAINS); read at level creation."""
        self._chk(lib().gc_ctx_set_option(self.h, int(key), C.c_int64(int(value))), "gc_ctx_set_option")

    def _alloc(self, nbytes, user):
        # large requests are rounded up to one of eight size classes per octave (<= 12.5 % more): the levels of an AMR run are
        # recreated at every regrid with slightly different sizes, and a request that misses torch's cache of freed blocks costs a
        # cudaMalloc (5-100 ms, and a device synchronisation)
        nbytes = int(nbytes)
        if nbytes >= (1 << 20):
            q = 1 << max(nbytes.bit_length() - 4, 21)
            nbytes = (nbytes + q - 1) // q * q
        try:
            with self.torch.cuda.stream(self.stream):
                t = self.torch.empty(nbytes, dtype=self.torch.uint8, device=self.device)
        except Exception:
            return None
        self._bufs[t.data_ptr()] = t
        return t.data_ptr()

    def _free(self, ptr, user):
        self._bufs.pop(ptr, None)

    def _chk(self, rc, what):
        if rc != 0:
            msg = lib().gc_last_error(self.h)
            raise RuntimeError("%s failed: %d (%s)" % (what, rc, msg.decode() if msg else ""))

    def level_create(self, level, xlo, ylo, dx, dy, nxl, nyl, ratio, patches):
        return Level(self, level, xlo, ylo, dx, dy, nxl, nyl, ratio, patches)

    def fp64_peak(self):
        v = C.c_double(0.0)
        self._chk(lib().gc_probe_fp64_peak(self.h, C.byref(v)), "gc_probe_fp64_peak")
        return v.value

    def selftest_math(self, a, b):
        """-> (mismatches, fallbacks) of the fast divide / reciprocal / sqrt against the IEEE operators"""
        a = np.ascontiguousarray(a, dtype=np.float64); b = np.ascontiguousarray(b, dtype=np.float64)
        nm, nf = C.c_int64(0), C.c_int64(0)
        self._chk(lib().gc_selftest_math(self.h, a.ctypes.data, b.ctypes.data, a.size, C.byref(nm), C.byref(nf)), "gc_selftest_math")
        return nm.value, nf.value

    def launch_count(self):
        return int(lib().gc_launch_count(self.h))

    def profile(self, on):
        self._chk(lib().gc_profile_enable(self.h, 1 if on else 0), "gc_profile_enable")

    def profile_read(self):
        """-> {slot name: (milliseconds, groups)} since the last read"""
        ms = (C.c_double * 10)(); cnt = (C.c_int64 * 10)()
        self._chk(lib().gc_profile_read(self.h, ms, cnt), "gc_profile_read")
        names = ["copy", "bc", "xsweep", "ysweep", "coarse", "avg", "flag", "flux", "misc", "fused"]
        return {n: (ms[k], cnt[k]) for k, n in enumerate(names)}

    def synchronize(self):
        self.stream.synchronize()

    def destroy(self):
        if self.h:
            lib().gc_ctx_destroy(self.h)
            self.h = None
