/* gc.h -- C ABI of libgeoclaw_b200.so: the per-level time step of GPU GeoClaw on one B200.
 *
 * Source of the operations: "Efficient Tsunami Modeling on Adaptive Grids with GPUs"
 * (arXiv 1901.06798; /root/reference/PAPER.md, cited as P:<line>), AMR steps 1-5 (P:140-146,
 * section 3.1), regridding (section 3.2), the wave-propagation update
 * (eqs. 4-14) and the CFL condition (eq. 15).  Everything the paper leaves
 * open is fixed in DESIGN.md section 3 ("readings").
 *
 * Conventions
 *  - plain C, extern "C"; every call returns int: 0 = GC_OK, < 0 = GC_ERR_*; nothing throws or aborts.
 *  - DEVICE vs HOST pointers are stated per argument.  All device work is enqueued on the CUDA
 *    stream given to gc_ctx_create (caller-owned) and is asynchronous unless the call returns a
 *    host scalar / fills a host struct (then the call synchronises that stream).
 *  - Ownership: the caller owns every array it passes and the stream.  The library takes device
 *    memory only through the allocator callbacks given to gc_ctx_create (so PyTorch can own it);
 *    with NULL callbacks it falls back to cudaMalloc / cudaFree.
 *  - Layout: a level is one pool; each patch stores (nx+4) x (ny+4) doubles per field, row-major,
 *    x fastest, ghost width 2 (interior cell (i,j) of the patch at storage (i+2, j+2)).  Fields are
 *    SoA planes h, hu, hv (two buffers each: "new" = current, "old" = previous step) and b.
 *  - Indices are 0-based global cell indices of the level; patches must not overlap; for level > 1
 *    patch boxes are aligned to coarse cells (i0, j0, nx, ny multiples of ratio_to_coarser).
 *  - fp64 throughout; fused multiply-adds exactly where DESIGN.md section 3 writes fma(a, b, c), no contraction anywhere
 *    else (-fmad=false), correctly rounded divide / sqrt: results are bit-identical to a plain C evaluation of
 *    DESIGN.md section 3 in the stated order.
 */
#ifndef GC_H
#define GC_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { GC_OK = 0, GC_ERR_BADARG = -1, GC_ERR_NOMEM = -2, GC_ERR_CUDA = -3, GC_ERR_NAN = -4,
       GC_ERR_NEGDEPTH = -5, GC_ERR_STATE = -6 };
enum { GC_FIELD_H = 0, GC_FIELD_HU = 1, GC_FIELD_HV = 2, GC_FIELD_B = 3 };
enum { GC_NEW = 0, GC_OLD = 1 };

typedef struct gc_ctx gc_ctx;
typedef struct gc_level gc_level;

typedef struct {
    int coord;            /* 0 Cartesian (metres), 1 spherical lon/lat (degrees), capacity form */
    double g;             /* gravity, 9.81 */
    double dry_tol;       /* dry tolerance epsilon: a cell with h <= dry_tol is dry ("handling dry states") */
    double sea_level;     /* eta_sea used by the flagging criterion */
    double earth_radius;  /* metres; used when coord == 1 */
    int limiter;          /* 0 none (first-order Godunov, eq. 4), 1 MC */
    int bc[4];            /* xlo, xhi, ylo, yhi: 0 zero-order extrapolation, 1 reflecting wall */
    double manning_n;     /* Manning coefficient n of the drag term, eq. 1b-1c, 2 (the paper uses 0.025); 0 = friction off.
                             Fractional step after the y-sweep of every level step with dt > 0 (reading S-16) */
    double friction_depth;/* friction acts in cells with dry_tol < h <= friction_depth */
} gc_params;

typedef struct { int32_t i0, j0, nx, ny; } gc_patch;   /* interior box of a patch */

typedef struct {
    double tol_eta;       /* flag wet cells with |h + b - sea_level| > tol_eta; <= 0: off */
    double tol_slope;     /* flag wet cells whose central-difference surface slope per cell > tol_slope; <= 0: off */
    int offshore_only;    /* wave criteria apply only where b < 0 */
    int buffer;           /* dilation by this many cells, Chebyshev distance */
    int nboxes;           /* forced space-time regions */
    const double *boxes;  /* HOST, 6 per box: x0, x1, y0, y1, t0, t1 */
} gc_flag_params;

typedef struct {
    double cfl_max;       /* nu = dt * s_over_dx_max (eq. 15) */
    double s_over_dx_max; /* max over both sweeps, all patches, interior lines, of |s| / (kappa dx) */
    double clipped_mass;  /* sum over interior cells of (-h) * area for cells with h < 0 set to 0 by the clean-up; accumulated with
                             floating-point atomics, so its last bits depend on the order (every other statistic and the state do not) */
    int64_t n_clipped;    /* number of such cells */
    int32_t nan_seen;     /* 1 if any updated value is NaN */
} gc_step_stats;

/* Allocator callbacks: alloc returns a DEVICE pointer (>= 256-byte aligned) or NULL. */
typedef void *(*gc_alloc_fn)(size_t bytes, void *user);
typedef void (*gc_free_fn)(void *ptr, void *user);

/* Gauges ("finding the best grid patch to sample quantities of interest from, interpolating from cell values"; DESIGN.md
 * 3.10, reading S-19).  The caller finds the best patch (finest level whose interior holds the point: host bookkeeping).
 * gc_gauges_bind: gauge k = point (xy[2k], xy[2k+1]) in the level's coordinates, inside the INTERIOR of patch patch[k] of L
 * (else GC_ERR_BADARG, nothing changes); both arrays HOST, read before return; replaces any earlier binding; n = 0 unbinds.
 * The binding dies with the level.
 * gc_gauges_sample: 4 doubles per bound gauge, in binding order -- h, hu, hv, eta = h + b -- from the level's current state with
 * its ghost cells as they are (call gc_fill_ghost first): bilinear between the four cell centres around the point when all four
 * are wet (h > dry_tol), else the values of the cell containing the point.  out DEVICE: enqueued on the context's stream,
 * returns without synchronising (a device-resident series costs one small kernel per record); out HOST: synchronous. */
int gc_gauges_bind(gc_level *L, int n, const int32_t *patch /*HOST*/, const double *xy /*HOST*/);
int gc_gauges_sample(const gc_level *L, double *out, int out_is_device);

/* Context: parameters + the CUDA stream (cudaStream_t passed as void*; NULL = legacy default stream). */
int gc_ctx_create(const gc_params *params /*HOST*/, void *cuda_stream, gc_alloc_fn alloc, gc_free_fn free_,
                  void *user, gc_ctx **out);
int gc_ctx_destroy(gc_ctx *);
const char *gc_last_error(const gc_ctx *);
/* Tuning knobs; none changes a result bit (all sweep kernel families compute the same bits).  Read when a level
 * is created.  GC_OPT_SWEEP_FAMILY: 0 = by level size (default), 1 = edge-parallel tiles, 2 = line marching.
 * GC_OPT_MARCH_SEG: cells per marching segment, 4..4096 (rounded down to a multiple of 4); 0 = by level size (default).
 * GC_OPT_CHAINS: 0 = marching lines run through same-level patches that continue each other (default), 1 = every patch on its own,
 * k >= 8 = patches of k cells or more along the sweep stay on their own.
 * Unknown key or value out of range: GC_ERR_BADARG, nothing changes. */
enum { GC_OPT_SWEEP_FAMILY = 0, GC_OPT_MARCH_SEG = 1, GC_OPT_CHAINS = 2 };
int gc_ctx_set_option(gc_ctx *, int key, int64_t value);

/* A1: one level = one device pool with all its patches, a patch-descriptor table,
 * per-row metric tables and the host-built work lists for ghost filling.  level is 1-based; level 1
 * covers the domain.  xlo, ylo: lower-left corner of the DOMAIN; dx, dy: cell size of THIS level;
 * nx_level, ny_level: domain size in cells of this level.  patches: HOST array.  State is zero. */
int gc_level_create(gc_ctx *, int level, double xlo, double ylo, double dx, double dy,
                    int64_t nx_level, int64_t ny_level, int ratio_to_coarser,
                    int npatch, const gc_patch *patches, gc_level **out);
int gc_level_destroy(gc_level *);
int64_t gc_level_ncells(const gc_level *);   /* interior cells of the level */

/* Sets a field on every patch of the level at once, ghost cells included: one transfer and one kernel, against one
 * gc_level_set_global per patch when a level is initialised patch by patch (every regrid).  src: for patch p = 0 .. np-1 in
 * order, (ny_p + 4) rows of (nx_p + 4) doubles, x fastest, back to back (HOST or DEVICE; a host array is free on return).  Cells
 * outside the level are not read; field GC_H..GC_B, written to the "new" buffer. */
int gc_level_set_patches(gc_level *L, int field, const double *src, int src_is_device);

/* Field transfer.  Per patch: arrays shaped like the storage, (ny+4) rows of (nx+4), leading dimension
 * ld (elements).  Global: the array covers global cells [gi0, gi0+gnx) x [gj0, gj0+gny) of the level with
 * leading dimension ld; set writes every storage cell (ghosts included) that falls inside, get reads
 * interior cells.  src/dst are DEVICE pointers if is_device != 0, else HOST (the call then stages through
 * a device buffer and synchronises).  which: GC_NEW (current state) or GC_OLD (before the last step). */
int gc_level_set_field(gc_level *, int patch, int field, const double *src, int is_device, int64_t ld);
int gc_level_get_field(const gc_level *, int patch, int field, int which, double *dst, int is_device, int64_t ld);
int gc_level_set_global(gc_level *, int field, const double *src, int is_device, int64_t ld,
                        int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny);
int gc_level_get_global(const gc_level *, int field, int which, double *dst, int is_device, int64_t ld,
                        int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny);

/* Asynchronous whole-level state transfer for pipelines ("overlapping memory copies with kernel execution").
 * host[0..2]: PINNED HOST arrays of h, hu, hv over the whole level, ny_level rows of nx_level doubles (a pageable array makes
 * the copies synchronous but stays correct).  copy_stream: a cudaStream_t (as void*) other than the context's stream.
 * upload: enqueues the three host->device copies on copy_stream into staging planes the library owns, then -- on the context's
 * stream, after an event -- the scatter into the pool ("new" buffer, every storage cell inside the level incl. ghost cells).
 * download: the gather of the interior cells of the "new" buffer on the context's stream (cells no patch covers read 0), then the
 * three device->host copies on copy_stream.  Both return without synchronising; consecutive calls on a level are ordered by
 * events, so a caller only has to synchronise copy_stream before it reads a downloaded array or reuses an uploaded one.
 * First use allocates 3 staging planes of nx_level * ny_level doubles per direction (released with the level). */
int gc_level_upload_state_async(gc_level *L, const double *const host[3] /*HOST, pinned*/, void *copy_stream);
int gc_level_download_state_async(gc_level *L, double *const host[3] /*HOST, pinned*/, void *copy_stream);

/* A2-A4 (P:143 step 2): fill the ghost cells of the current state.  Order: same-level
 * copy incl. corners; remaining in-domain ghosts from `coarser` interpolated in space (limited linear in
 * eta, u, v) and time (alpha = (t - t_coarse_old) / dt_coarse, linear between coarser's OLD and NEW buffers,
 * whose own ghosts must be filled); physical boundary (x faces, then y faces).  coarser == NULL: level 1.
 * gc_fill_ghost_b does same-level copy + physical boundary for the bathymetry (once per regrid). */
int gc_fill_ghost(gc_level *L, const gc_level *coarser, double alpha);
int gc_fill_ghost_b(gc_level *L);
/* The same, for a caller whose NEXT call on L is a split step (gc_level_step, gc_level_step_auto, gc_level_step_accum): it fills
 * the ghost cells that step reads and may leave the others as they are.  Where same-level patches continue each other, the
 * marching sweeps read the neighbour's interior directly (chains) and the copy into the ghost cells between them is
 * dead work -- on a regular tiling of small patches, all of it.  The step's result is bit-identical to the one after
 * gc_fill_ghost.  Anything else that reads ghost cells (gc_level_get_field, gc_flag_cells, gc_gauges_sample, a finer level's
 * gc_fill_ghost or gc_level_init_from, gc_level_step_unsplit) needs gc_fill_ghost.  Levels without chains, or with flux
 * registers attached, get the full fill. */
int gc_fill_ghost_step(gc_level *L, const gc_level *coarser, double alpha);

/* Time-dependent bathymetry B(x, y, t) (the seafloor-deformation source that starts both of the paper's tsunamis, P:273
 * "deformation information on uniform grids", "ground deformation file", reading S-20).  dz: vertical
 * seafloor displacement in metres (+ up) on a uniform node grid, node (m, n) at (x0 + m ddx, y0 + n ddy) in the level's
 * coordinates, my rows of mx values (HOST, or DEVICE if dz_is_device); bilinear between nodes, zero outside the grid.
 * gc_bathy_update: b <- fma(w, dz(cell centre), b) on every storage cell of L whose centre lies inside the domain (ghost cells
 * included; follow with gc_fill_ghost_b for the cells outside).  h, hu, hv are not touched: the water column rides on the
 * seafloor, so the surface moves with it.  The caller supplies w, the increment of its ramp over [t0, t1] since its last call on
 * this level (a new level starts from the undeformed bathymetry it was given). */
typedef struct {
    double x0, y0, ddx, ddy;
    int64_t mx, my;             /* nodes per direction, >= 2 */
    const double *dz;
    int dz_is_device;
} gc_deform;
int gc_bathy_update(gc_level *L, const gc_deform *D /*HOST struct*/, double w);

/* A5-A7 (P:142 step 1; eqs. 13-15): x-sweep then y-sweep over every patch of the level, dry clean-up,
 * exact order-independent max reduction of the wave speeds, swap NEW/OLD.  dt == 0 is a probe: state and
 * buffers unchanged, speeds returned.  out: HOST struct, or NULL = keep the statistics on the device (no
 * synchronisation; read them later with gc_level_stats). */
int gc_level_step(gc_level *L, double dt, gc_step_stats *out);
/* Same with dt held in device memory: dt_used = *dt_dev (DEVICE double, read by the kernels); after the
 * step the library writes the next dt = cfl_target / s_over_dx_max into *dt_dev.  No host sync; CUDA-graph
 * capturable. */
int gc_level_step_auto(gc_level *L, double *dt_dev, double cfl_target);
int gc_level_stats(const gc_level *, gc_step_stats *out /*HOST*/);
/* For the subcycled levels of the AMR recursion, whose steps the host has no reason to wait for one by one:
 * gc_level_step_accum is gc_level_step(L, dt, NULL) with dt > 0 WITHOUT zeroing the level's statistics first, so that over a run of
 * steps s_over_dx_max becomes their maximum (exact: a max of bit images), n_clipped and clipped_mass their sums, nan_seen their
 * OR; gc_level_stats reads them (and waits), gc_level_stats_reset zeroes them (no wait).  cfl_max is not formed (0). */
int gc_level_step_accum(gc_level *L, double dt);
int gc_level_stats_reset(gc_level *L);
/* The same level step by the UNSPLIT wave-propagation method with transverse Riemann solves -- "the original GeoClaw ... with the
 * unsplit algorithm" that the paper simplifies to dimensional splitting and validates against (DESIGN.md 3.13,
 * reading S-21): every edge's fluctuations and limited correction flux from Q^n, each edge's vectors A-dQ + F~ and A+dQ - F~ split
 * by the transverse Jacobian of the cell they enter into parts that modify the neighbouring edges' correction fluxes, one update.
 * Same arguments, statistics and dt = 0 probe as gc_level_step.  Flux registers (gc_flux_attach) are defined for the split step
 * only: GC_ERR_STATE on a level that has any.  First use allocates 18 planes of scratch (released with the level). */
int gc_level_step_unsplit(gc_level *L, double dt, gc_step_stats *out);
/* The same step for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * identical arithmetic and results, but the 18 scratch planes live in a file-scope device array inside the library instead of
 * being allocated at the level's first unsplit step.  The entry point calls no cudaMalloc / cudaFree and no allocator callback.
 * Limit: the level's storage cells (every patch's (nx + 4 rounded up to a multiple of 4) x (ny + 4), summed) must not exceed
 * GC_UNS_STATIC_MAX_CELLS, else GC_ERR_BADARG and nothing changes; gc_unsplit_static_max_cells() returns the limit.  The array
 * (18 x GC_UNS_STATIC_MAX_CELLS doubles = 37.75 MB) is held by every GPU that loads the library until the process exits.  Its
 * address is resolved once per device at gc_ctx_create (GC_ERR_CUDA here if that failed).  All calls on a device share the array,
 * which keeps the last call's contents (nothing in it has to start at zero: every value used is written by the same call first):
 * calls that overlap on the GPU -- other streams, other contexts -- race; calls on one stream do not.  out as for gc_level_step
 * (NULL: no synchronisation). */
#define GC_UNS_STATIC_MAX_CELLS (1 << 18)
int gc_level_step_unsplit_static(gc_level *L, double dt, gc_step_stats *out);
int64_t gc_unsplit_static_max_cells(void);

/* wet mask (h > dry_tol) of the current state: one byte per interior cell, patch after patch, row-major. */
int gc_wet_mask(const gc_level *, uint8_t *mask, int is_device);
/* sum of h * cell area over interior cells, fixed-order (deterministic) reduction; returns NaN on error. */
double gc_level_mass(const gc_level *);

/* A10: refinement flags of the current state, one byte per interior cell (layout as
 * gc_wet_mask); ghost cells must be filled if tol_slope > 0.  nflag (HOST, nullable) receives the count. */
int gc_flag_cells(const gc_level *L, const gc_flag_params *, double t, uint8_t *flags, int is_device, int64_t *nflag);

/* A9 (P:145 step 4): every coarse cell covered by fine cells <- average of the r*r fine cells. */
int gc_average_down(gc_level *coarse, const gc_level *fine);
/* A11: interior of the new fine level <- copy from oldfine where it overlapped (nullable), else
 * interpolation from coarse's NEW buffer (ghosts filled).  b of newfine must be set already. */
int gc_level_init_from(gc_level *newfine, const gc_level *oldfine, const gc_level *coarse);

/* A8 (P:146 step 5): flux registers on the boundary of the fine region.  attach builds and zeroes them
 * (and makes both levels record what the registers need during gc_level_step); fixup applies
 * Q_C += side * delta / area to the uncovered coarse neighbours, then the clean-up rule, and re-zeroes.
 * GC_ERR_BADARG for a refinement ratio above 128, GC_ERR_STATE if the fine level is not nested in the coarse one. */
int gc_flux_attach(gc_level *coarse, gc_level *fine);
int gc_flux_fixup(gc_level *coarse, gc_level *fine);

#ifdef __cplusplus
}
#endif
#endif
