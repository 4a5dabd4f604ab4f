// gc_api_amr.cu -- level-transfer entry points (A3, A8-A11): host list building + launches.
#include "gc_internal.h"

int gc_fill_coarse_ghosts(gc_level *L, const gc_level *C, double alpha)
{
    (void)C; (void)alpha;
    return gc_fail(L->ctx, GC_ERR_STATE, "coarse fill: not built yet");
}
int gc_flux_after_step(gc_level *L, double dt, const double *dt_dev) { (void)L; (void)dt; (void)dt_dev; return GC_OK; }

extern "C" int gc_flag_cells(const gc_level *L, const gc_flag_params *fp, double t, uint8_t *flags, int is_device, int64_t *nflag)
{ (void)fp; (void)t; (void)flags; (void)is_device; (void)nflag; return gc_fail(L->ctx, GC_ERR_STATE, "not built yet"); }
extern "C" int gc_average_down(gc_level *C, const gc_level *F) { (void)F; return gc_fail(C->ctx, GC_ERR_STATE, "not built yet"); }
extern "C" int gc_level_init_from(gc_level *N, const gc_level *O, const gc_level *C) { (void)O; (void)C; return gc_fail(N->ctx, GC_ERR_STATE, "not built yet"); }
extern "C" int gc_flux_attach(gc_level *C, gc_level *F) { (void)F; return gc_fail(C->ctx, GC_ERR_STATE, "not built yet"); }
extern "C" int gc_flux_fixup(gc_level *C, gc_level *F) { (void)F; return gc_fail(C->ctx, GC_ERR_STATE, "not built yet"); }
