/* gc_test.h -- measurement and self-test entry points of libgeoclaw_b200.so.  They are exported by the same library but are not
 * part of the product ABI (include/gc.h): bench.py and tests/ use them to count and time kernels, to check the correctly rounded
 * fast-math sequences of csrc/gc_math.cuh against the IEEE operators on the device, and to measure the chip's fp64 rate for the
 * "alu" roofline.  Same conventions as gc.h. */
#ifndef GC_TEST_H
#define GC_TEST_H
#include "gc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Kernel accounting.  gc_launch_count: kernels launched by this context so far.  gc_profile_enable(on): bracket
 * every kernel group with CUDA events on the context's stream; gc_profile_read synchronises, returns per slot the
 * summed milliseconds and the number of bracketed groups since the last read (arrays of GC_PROFILE_SLOTS), and clears.
 * Slots: 0 same-level copy, 1 physical BC, 2 x-sweep, 3 y-sweep, 4 coarse fill, 5 average-down / regrid transfer,
 * 6 flags, 7 flux registers, 8 misc (stats, dt), 9 fused sweep. */
#define GC_PROFILE_SLOTS 10
int64_t gc_launch_count(const gc_ctx *);
int gc_profile_enable(gc_ctx *, int on);
int gc_profile_read(gc_ctx *, double *ms /*HOST*/, int64_t *count /*HOST*/);

/* How often the line-marching sweep kernels left their guarded open-ocean code on this level, cumulative since it was created
 * (the paper's hazard: divergence at shorelines).  out[0] = warp iterations of the marching kernels (one iteration = one
 * cell per lane); out[1] = those in which at least one lane's cell or edge went through the general code; out[2], out[3] =
 * lane-level Riemann solves / edge fluxes redone with the general code.  Levels swept by the edge-parallel kernels report 0.
 * Synchronises the context's stream. */
int gc_level_fallback_counts(const gc_level *L, int64_t out[4] /*HOST*/);

/* Cells one launch of the marching sweep kernels updates on this level (the unit of bench.py's per-launch roofline figures):
 * out[0] = x-sweep over every row of every patch (4 ghost rows per patch, S-5), out[1] = x-sweep without the ghost rows no y line
 * reads (chains; what runs when no flux register is attached), out[2] = y-sweep (= interior cells).  0 for levels swept by the
 * edge-parallel kernels. */
int gc_level_sweep_cells(const gc_level *L, int64_t out[3] /*HOST*/);

/* Self-test of the branch-free correctly rounded divide / reciprocal / square root the marching kernels use
 * (csrc/gc_math.cuh) against the IEEE operators: for each i, a[i]/b[i], 1/b[i], sqrt(a[i]) (a, b: HOST arrays of n).
 * nmismatch = results that differ in any bit although the fast path accepted the operands (must be 0);
 * nfallback = operations whose operands were outside the fast window (they are redone with the operators). */
int gc_selftest_math(gc_ctx *, const double *a, const double *b, int64_t n, int64_t *nmismatch, int64_t *nfallback);

/* Measured fp64 ALU throughput of this device (DFMA micro-benchmark, flop/s); for the "alu" roofline. */
int gc_probe_fp64_peak(gc_ctx *, double *flops_out /*HOST*/);

#ifdef __cplusplus
}
#endif
#endif
