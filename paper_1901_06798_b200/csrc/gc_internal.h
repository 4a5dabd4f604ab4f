// gc_internal.h -- internals of libgeoclaw_b200.so (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <unordered_map>
#include <vector>
#include "../../include/gc.h"
#include "../../include/gc_test.h"

#define GC_G 2  // ghost width
#define GC_MARCH_MIN_CELLS 800000    // levels at least this large use the line-marching sweep kernels

// patch descriptor as the kernels see it (A1): interior box, element offset of the patch in a field plane, row pitch
struct PatchDesc {
    int32_t i0, j0, nx, ny;
    int64_t off;     // element offset in every field plane of the pool; off % 4 == 2: storage column 2 of every row starts a 32-byte sector
    int64_t ioff;    // offset in interior-packed arrays (masks, flags)
    int32_t pitch;   // row pitch in elements: nx + 4 rounded up to a multiple of 4
    int32_t bcmask;  // bit0 touches xlo, bit1 xhi, bit2 ylo, bit3 yhi
};

// work item of a sweep kernel: a group of lines (rows for x, columns for y) times a segment along the sweep
struct SweepTile {
    int32_t patch;
    int32_t line0, nlines;  // rows [line0, line0+nlines) (x-sweep) or columns (y-sweep), storage indices
    int32_t c0, nc;         // cells [c0, c0+nc) along the sweep direction, storage indices (edges c0-1 .. c0+nc+1 are solved)
};

// work item of a marching sweep kernel: ONE thread walks cells [c0-2, c0+nc+2) of a line (row for x, column for y),
// solving edges c0-1 .. c0+nc+1 and updating cells c0 .. c0+nc-1 (storage indices along the sweep)
// With chains (below) c0 counts positions along the chain and `patch` is the piece holding position c0 - 2.
struct LineDesc {
    int32_t patch, line, c0, nc;
};

// Chains: same-level patches that continue each other along a sweep direction (x: equal j0, ny, side by side; y: equal i0, nx,
// stacked) are walked by the marching kernels as ONE line, each piece's interior read and written in that patch's own storage --
// the redundant edges and ghost cells of a patch boundary are paid once per segment instead of once per patch, which is what
// small patches cost (DESIGN.md 5 "chains").  Position s along a chain = (interior cells of the pieces before
// the patch) + storage index inside the patch; a position of piece p on line l sits at A + l * pitch + s (x) or A + s * pitch + l
// (y) in a field plane.  One link per patch and direction; a patch outside any chain is a chain of one (A = off, end = INT_MAX).
struct ChainLink {
    int64_t A;          // plane offset of position 0 of line 0, extrapolated back from this piece
    int32_t end;        // first position of the next piece (= this piece's position of storage index n + 2), INT_MAX in the last piece
    int32_t next;       // patch index of the next piece, -1 in the last one
    int32_t pitch;      // row pitch of this piece
    int32_t org;        // y chains: j0 of the chain's head (global row + 2 of position s is org + s); x chains: j0
};

// same-level ghost copy: rectangle of w x h cells
struct CopyRect {
    int64_t dst, src;       // element offsets in a field plane
    int32_t w, h, dpitch, spitch;
};

// a rectangle of fine cells (w x h) lying inside ONE coarse patch, to be interpolated from the coarser level
// (ghost fill A3 / regrid transfer A11).  Fine cell (x, y) of the rectangle sits at sub-position
// ((ii0 + x) % r, (jj0 + y) % r) of the coarse cell csrc + ((jj0 + y) / r) * cpitch + (ii0 + x) / r.
struct CoarseFillRect {
    int64_t dst;            // element offset of the rectangle's lower-left fine cell in the fine plane
    int64_t csrc;           // element offset, in the coarse plane, of the coarse cell holding that fine cell
    int32_t dpitch, cpitch;
    int32_t w, h;
    int32_t ii0, jj0;       // sub-position of the lower-left fine cell inside its coarse cell, 0..r-1
};

struct AvgRect {            // average-down A9: w x h covered coarse cells under one fine patch, inside one coarse patch
    int64_t cdst;           // coarse plane offset of the lower-left coarse cell
    int64_t fsrc;           // fine plane offset of the lower-left fine cell under it
    int32_t cpitch, fpitch;
    int32_t w, h;
    int32_t frow;           // table index (global fine row + 2) of that fine cell, for the kappa weights
    int32_t pad;
};

struct FluxReg {            // A8, one register (coarse edge on the boundary of the fine region)
    int64_t ccell;          // coarse plane offset of the uncovered coarse cell C
    int64_t fcell;          // fine plane offset of the first adjacent fine cell
    int32_t cpitch, fpitch;
    int32_t crow, frow;     // global rows (coarse cell / first fine cell) for metric tables
    int32_t dir, side;      // dir 0: x-edge, 1: y-edge; side +1: fine region on the high side of C
};

struct DevStats {
    unsigned long long sdx_bits;   // max of s/(kappa dx) as the bit image of a non-negative double
    unsigned long long nclip;
    double clipped;
    int nan_seen;
    int pad;
    // cumulative since the level was created (never reset by a step): how often the marching kernels left the guarded open-ocean
    // code (divergence at shorelines).  warp_iters: warp iterations in all; fb_warp_iters: of these, the ones in which some
    // lane ran the general code; fb_solves / fb_fluxes: lane-level Riemann solves / edge fluxes redone with the general code
    unsigned long long warp_iters, fb_warp_iters, fb_solves, fb_fluxes;
};

// profiling slots (gc_profile_read): kernels grouped by the SURVEY 8(a) row they implement
enum { GC_SLOT_COPY = 0, GC_SLOT_BC = 1, GC_SLOT_XSWEEP = 2, GC_SLOT_YSWEEP = 3, GC_SLOT_COARSE = 4, GC_SLOT_AVG = 5,
       GC_SLOT_FLAG = 6, GC_SLOT_FLUX = 7, GC_SLOT_MISC = 8, GC_SLOT_FUSED = 9, GC_NSLOT = 10 };

struct gc_ctx {
    gc_params P;
    cudaStream_t stream;
    gc_alloc_fn alloc;
    gc_free_fn free_;
    void *user;
    std::string err;
    bool prof = false;
    int opt_family = 0, opt_seg = 0, opt_chains = 0;                 // gc_ctx_set_option: sweep kernel family (0 auto, 1 edge, 2 march), marching segment length
    void *stage = nullptr; size_t stage_bytes = 0;   // grow-only device staging buffer of the host-pointer paths (gc_stage_get)
    unsigned long long launches = 0;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev[GC_NSLOT];     // brackets per slot; the events themselves are owned by ev_own
    std::vector<cudaEvent_t> ev_own; cudaEvent_t prof_last = nullptr;
};

// counts kernel launches; when profiling is on, brackets them with CUDA events on the launching stream.  The event that ends one
// launch's bracket starts the next one's (the library's launches follow each other on one stream; every recorded event puts a
// small bubble between two kernels, so there are n + 1 of them for n launches, not 2 n): a launch's time then includes the gap
// before it, a few microseconds.  gc_profile_enable and gc_profile_read start a new run of brackets.
struct ProfScope {
    gc_ctx *c; int slot; cudaEvent_t e0;
    ProfScope(gc_ctx *c_, int slot_, int nlaunch = 1) : c(c_), slot(slot_), e0(nullptr)
    {
        c->launches += nlaunch;
        if (c->prof) {
            e0 = c->prof_last;
            if (!e0) { cudaEventCreate(&e0); c->ev_own.push_back(e0); cudaEventRecord(e0, c->stream); }
        }
    }
    ~ProfScope()
    {
        if (e0) {
            cudaEvent_t e1; cudaEventCreate(&e1); c->ev_own.push_back(e1); cudaEventRecord(e1, c->stream);
            c->ev[slot].push_back({e0, e1}); c->prof_last = e1;
        }
    }
};

// one bound gauge: pool offsets of stencil cell (i, j) and of the containing cell, the patch's row pitch, the weights
struct GaugeLoc { int64_t c00, cc; int32_t pitch, pad; double a, b; };

struct gc_level {
    gc_ctx *ctx;
    int level, ratio, np, cur;
    double xlo, ylo, dx, dy, ex;
    int64_t nxl, nyl, ncells, tot;
    std::vector<gc_patch> pat;
    std::unordered_map<int64_t, std::vector<int32_t>> buckets; int bsize;   // spatial hash of patch interiors (host lookups)
    std::vector<PatchDesc> hpat;
    std::vector<double> kappa, rdx, rdy, ey;        // host copies of the metric tables
    // device pool: q[2][3], b, qs[3] are planes of `tot` doubles inside one allocation
    double *pool;
    double *q[2][3];
    double *b;
    double *qs[3];
    PatchDesc *d_pat;
    double *d_kappa, *d_rdx, *d_rdy, *d_ey;
    SweepTile *d_xt, *d_yt; int nxt, nyt;            // edge-parallel tiles (small levels)
    LineDesc *d_xl, *d_yl; int64_t nxl_lines, nyl_lines;   // marching lines (large levels)
    // chains of patches along x / y (one link per patch); x lines without the ghost rows no y line reads (their patch continues
    // above / below inside a y chain) -- used when no flux register reads Q* there; chained: 1 = some chain has two pieces
    ChainLink *d_xlink = nullptr, *d_ylink = nullptr; LineDesc *d_xl_red = nullptr; int64_t nxl_red = 0; int chained = 0;
    int64_t sweep_cells[3] = {0, 0, 0};             // cells updated per launch: x-sweep over every row, x-sweep without the unread ghost rows, y-sweep
    int use_march;
    CopyRect *d_copy; int ncopy;                     // same-level copy rectangles, grouped by destination patch
    int2 *d_copy_range; int copy_wpp;               // per patch: (first rectangle, count); warps serving one patch
    CopyRect *d_copy_red = nullptr; int2 *d_copy_range_red = nullptr; int ncopy_red = -1;   // the rectangles a split step reads (gc_fill_ghost_step); -1: all
    int32_t *d_bcp; int nbcp;                       // patches touching the physical boundary
    std::vector<int64_t> coarse_ghost;              // plane offsets + global indices of ghosts to be filled from the coarser level
    std::vector<int32_t> coarse_ghost_ij;           // (gi, gj) pairs
    // cached coarse-fill list for a given coarser level (rebuilt when the coarser level changes)
    const gc_level *cf_for; uint64_t cf_gen; CoarseFillRect *d_cf; int64_t *d_cfstart; int ncf; int64_t ncfcells;
    uint64_t gen;                                   // unique id of this level object
    DevStats *d_stats;
    double *d_partial;                              // mass partials (gc_mass_partials of them)
    std::vector<void *> allocs;
    // flux registers (this level as the coarse side) + capture slots
    const gc_level *reg_fine; gc_level *reg_coarse;   // cleared by gc_level_destroy of either side
    FluxReg *d_reg; int nreg; int r_reg;
    double *d_delta, *d_base;                       // nreg*3, nreg*4
    int32_t *d_fixstart; int nfix;                  // registers grouped by coarse cell for the fix-up: group g = d_fixreg[d_fixstart[g] .. d_fixstart[g+1])
    int32_t *d_fixreg;
    // cached average-down list for a given fine level, cached neighbour lists for flag dilation
    uint64_t avg_gen; AvgRect *d_avg; int64_t *d_avgstart; int navg; int64_t navgcells;
    int nbr_buffer; int32_t *d_nbrstart, *d_nbrlist;
    int64_t *d_goff = nullptr; int64_t gtot = 0;      // packed offsets of gc_level_set_patches (built at first use)
    double *d_uns = nullptr;                         // scratch of the unsplit step: 18 planes (gc_unsplit.cu)
    GaugeLoc *d_gauge = nullptr; int ngauge = 0;     // gauges bound to this level (gc_gauges_bind)
    // asynchronous whole-level state transfer (gc_level_upload_state_async / gc_level_download_state_async): staging planes of
    // nxl * nyl doubles per field and direction, events that order the copy stream against the context's stream
    double *xfer_up[3] = {nullptr, nullptr, nullptr}, *xfer_dn[3] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_up_copied = nullptr, ev_up_free = nullptr, ev_dn_ready = nullptr, ev_dn_free = nullptr;
};

void gc_launch_gauges(const gc_level *L, double *out);

// ---- helpers (gc_api.cu)
void *gc_dev_alloc(gc_ctx *c, size_t bytes);
void gc_dev_free(gc_ctx *c, void *p);
// device staging for a host-pointer transfer: the context's retained buffer when the request is small (no allocator
// callback per call), a transient allocation otherwise (*transient = true: release with gc_dev_free after a stream sync)
void *gc_stage_get(gc_ctx *c, size_t bytes, bool *transient);
int gc_fail(gc_ctx *c, int code, const char *msg);
int gc_cuda_check(gc_ctx *c, const char *what);
int gc_find_patch_host(const gc_level *L, int64_t gi, int64_t gj);

// ---- kernel launch wrappers
// gc_sweep.cu
void gc_launch_sweeps(gc_level *L, double dt, const double *dt_dev, int write_out);
void gc_launch_stats_reset(gc_level *L);
void gc_launch_next_dt(gc_level *L, double *dt_dev, double cfl_target);
void gc_launch_math_selftest(cudaStream_t s, const double *a, const double *b, int64_t n, unsigned long long *out);
void gc_launch_fp64_probe(cudaStream_t s, double *out, int iters, int blocks, int threads);
// gc_unsplit.cu
int gc_launch_unsplit(gc_level *L, double dt, int write_out);
void gc_unsplit_static_setup(void);   // resolves the static scratch array's device address on the current device (once per device)
// gc_ghost.cu
void gc_launch_copy_rects(gc_level *L, double *f0, double *f1, double *f2, int nf, bool for_step);
void gc_launch_bc(gc_level *L, double *f0, double *f1, double *f2, int nf, int is_state);
void gc_launch_set_patches(gc_level *L, double *plane, const int64_t *goff, const double *src);
void gc_launch_set_global(gc_level *L, double *plane, const double *src, int64_t ld, int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny);
void gc_launch_get_global(const gc_level *L, const double *plane, double *dst, int64_t ld, int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny);
void gc_launch_copy2d(cudaStream_t s, double *dst, int64_t dld, const double *src, int64_t sld, int w, int h);
void gc_launch_wet_mask(const gc_level *L, uint8_t *mask);
void gc_launch_bathy_update(gc_level *L, double x0, double y0, double ddx, double ddy, int64_t mx, int64_t my, const double *d_dz, double w);
void gc_launch_mass(const gc_level *L);
int gc_mass_partials(const gc_level *L);    // number of partial sums gc_launch_mass writes to d_partial
// gc_amr.cu
void gc_launch_coarse_fill(gc_level *L, const gc_level *C, const CoarseFillRect *rects, const int64_t *start, int n, int64_t ncells,
                           double alpha, int use_old, int slot);
void gc_launch_average_down(gc_level *C, const gc_level *F, const AvgRect *rects, const int64_t *start, int n, int64_t ncells);
void gc_launch_flags(const gc_level *L, const gc_flag_params *fp, const double *d_boxes, double t, uint8_t *raw, uint8_t *flags,
                     const int32_t *nbr_start, const int32_t *nbr_list, unsigned long long *d_count);
void gc_launch_copy_overlap(gc_level *N, const gc_level *O, const CopyRect *rects, int n);
void gc_launch_flux_coarse(gc_level *C, double dt, const double *dt_dev);
void gc_launch_flux_fine(gc_level *F, double dt, const double *dt_dev);
void gc_launch_flux_fixup(gc_level *C);
