/* gco_int.h -- ORACLE internals (test infrastructure). */
#ifndef GCO_INT_H
#define GCO_INT_H
#include "gco.h"

struct gco_ctx { gco_params P; };

/* one flux-register edge: a coarse edge on the boundary of the fine region */
typedef struct {
    int32_t cp;        /* coarse patch holding the uncovered coarse cell C */
    int32_t ci, cj;    /* storage indices of C in that patch */
    int32_t dir;       /* 0: x-edge (fine region to the left/right), 1: y-edge */
    int32_t side;      /* +1: fine region on the high side of C, -1: on the low side */
    int32_t fpat;      /* fine patch across the edge */
    int32_t fi, fj;    /* storage indices of the first adjacent fine cell (r of them along the edge) */
    double base[4];    /* state of C the coarse sweep saw: h, normal, transverse momentum, b */
    double delta[3];   /* accumulated register (h, normal, transverse) */
} gco_freg;

struct gco_level {
    gco_ctx *ctx;
    int level, ratio, np, cur;
    double xlo, ylo, dx, dy, ex;
    int64_t nxl, nyl, ncells;
    gco_patch *pat;
    int64_t *off;          /* element offset of each patch in the level arrays */
    double *q[2][3];       /* [buffer][h,hu,hv]; q[cur] = current ("new"), q[1-cur] = previous ("old") */
    double *b;
    int32_t *gsrc;         /* per storage cell: source patch of a ghost, -1 coarse, -2 outside */
    double *kappa, *rdx, *rdy, *ey; /* metric tables over global rows -2..ny+1 (edges -2..ny+2) */
    gco_step_stats last;
    /* flux registers (this level as the COARSE side of a pair) and flux saving */
    int save_flux;         /* keep fm/fp of the last step for every edge */
    double *fmx, *fpx, *fmy, *fpy; /* 3 doubles per storage cell: edge at the low side of the cell */
    double *qs[3];         /* Q* (after the x-sweep) of the last step, storage shaped */
    int nreg; gco_freg *reg;       /* registers owned by this (coarse) level */
    struct gco_level *reg_fine;    /* the fine level they belong to */
    struct gco_level *reg_coarse;  /* on the fine level: the coarse level holding its registers */
};

double *gco_field(const gco_level *L, int field, int which);
int gco_find_patch(const gco_level *L, int64_t gi, int64_t gj);
double gco_cell_area(const gco_level *L, int64_t grow);
int gco_fill_coarse(gco_level *L, const gco_level *coarser, double alpha, int all_cells);
void gco_flux_free(gco_level *L);
void gco_flux_accumulate_own(gco_level *L, double dt);
#endif
